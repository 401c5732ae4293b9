// Primitive s/p electron-repulsion integrals in registers (McMurchie-Davidson form, cf. P:130 refs 88-91).
//
// (ab|cd) = 2 pi^(5/2) / (p q sqrt(p+q)) K_ab K_cd * [ O_a O_b O_c O_d R ](0),  where R_{tuv} are the Hermite
// Coulomb integrals R^0_{tuv}(alpha, P-Q) and every p function is the operator (X_PA + (1/2p) d/dP_x) acting
// on the s-type result (for ket functions d/dQ = -d/dP, hence the minus sign).  Everything is unrolled at
// compile time; Hermite tables live in registers.
#pragma once
#include "common.cuh"

namespace rttda {

#ifndef RTTDA_SCALED_STAGES
#define RTTDA_SCALED_STAGES 1
#endif
#ifndef RTTDA_FUSED_L1
#define RTTDA_FUSED_L1 1
#endif

__host__ __device__ constexpr int nherm(int L) { return (L + 1) * (L + 2) * (L + 3) / 6; }
// index of Hermite component (t,u,v): ordered by total order N, then s = N - t, then v
__host__ __device__ constexpr int hidx(int t, int u, int v)
{
    return nherm(t + u + v - 1) + (u + v) * (u + v + 1) / 2 + v;
}
__host__ __device__ constexpr int hidx_plus(int t, int u, int v, int axis)
{
    return axis == 0 ? hidx(t + 1, u, v) : (axis == 1 ? hidx(t, u + 1, v) : hidx(t, u, v + 1));
}

// ---- Boys function F_0..F_L(T), near field ------------------------------------------------------------
// T < BOYS_TMAX = 36 (plus rounding slack of the caller's test): nearest grid point T0 = j/8; one 80-byte table row
//   {h_0..h_7, e^-T0, pad}, h_k = F_{L+k}(T0)/k!, so that F_L(T) = sum_k h_k (T0-T)^k (dF_n/dT = -F_{n+1}) is a
//   7-FMA Horner chain; then downward recursion F_{n-1} = (2T F_n + e^-T)/(2n-1) with e^-T = e^-T0 e^(T0-T)
//   (degree-8 Taylor, |T0-T| <= 1/16).
//   The row is a shared-memory gather; in the workloads of DESIGN.md only ~1 primitive quartet in 8 takes this
//   branch (few active lanes), so its cost is its instruction count, not its shared-memory traffic.
// The far field (T >= 36) never forms F_n: see hermite_R.
template <int L>
__device__ __forceinline__ void boys_near(double T, const double2* __restrict__ tab, double (&F)[L + 1])
{
    constexpr double MAGIC = 6755399441055744.0;          // 1.5 * 2^52: rounds to nearest integer
    const double t = fma(T, 8.0, MAGIC);
    const int j = __double2loint(t);
    const double dx = fma(t - MAGIC, 0.125, -T);          // T0 - T, |dx| <= 1/16
    const double2* row = tab + j * (BOYS_ROW / 2);
    const double2 h01 = row[0], h23 = row[1], h45 = row[2], h67 = row[3];
    double f = h67.y;
    f = fma(f, dx, h67.x);
    f = fma(f, dx, h45.y);
    f = fma(f, dx, h45.x);
    f = fma(f, dx, h23.y);
    f = fma(f, dx, h23.x);
    f = fma(f, dx, h01.y);
    f = fma(f, dx, h01.x);
    F[L] = f;
    if (L > 0) {
        const double e0 = row[4].x;
        double e = 1.0 / 40320.0;
        e = fma(e, dx, 1.0 / 5040.0);
        e = fma(e, dx, 1.0 / 720.0);
        e = fma(e, dx, 1.0 / 120.0);
        e = fma(e, dx, 1.0 / 24.0);
        e = fma(e, dx, 1.0 / 6.0);
        e = fma(e, dx, 0.5);
        e = fma(e, dx, 1.0);
        e = fma(e, dx, 1.0);
        e *= e0;
        const double t2 = 2.0 * T;
#pragma unroll
        for (int n = L; n >= 1; --n) F[n - 1] = fma(t2, F[n], e) * (1.0 / (2 * n - 1));
    }
}

// ---- Hermite Coulomb integrals R^0_{tuv}, |tuv| <= L, times the prefactor 2 pi^(5/2) / (pq sqrt(p+q)) K_ab K_cd ------
// r[n][0] = pref (-2 alpha)^n F_n(T), alpha = pq/(p+q), T = alpha R^2.  The kernels carry every primitive pair as
//   c' = c pi^(1/4) / sqrt(2p)   (c = row entry [4], so that c_b c_k / sqrt(p+q) = c'_b c'_k (2/sqrt(pi)) sqrt(alpha))
//   w  = 36 / p                  (so that alpha = 36 / (w_b + w_k) and T < 36  <=>  R^2 < w_b + w_k)
// (PrimPair::c and PrimPair::p hold c' and w; see to_scaled).
// Far field (T >= 36; erfc(6) = 2.2e-17 and every dropped term e^-T/2T of the upward recursion is below 4e-18 of the
// (ss|ss)-like magnitude, since (2 alpha)^n / ((2p)^k (2q)^m) <= 1 for n = k + m): F_0 = sqrt(pi/T)/2 and
// F_{n+1} = (2n+1) F_n / 2T give r[0][0] = c'_b c'_k / R and r[n+1][0] = -(2n+1) r[n][0] / R^2: alpha and (p+q)^-1/2
// cancel, so the majority branch costs ONE rsqrt, no reciprocal, and the branch test is an add and a compare.
// Near field: alpha = 36 / w needs one more rsqrt; pref = c'_b c'_k (12/sqrt(pi)) / sqrt(w).
__device__ __forceinline__ double rsqrt_fast(double x)
{
    // MUFU.RSQ64H seed (2^-20) and one third-order step: error 1.6e-16 for normal positive x (measured); the library
    // rsqrt() adds a slow-path call for subnormals / infinities that splits the scheduling region
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y * y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
}

// The seeds of the recursion alone: s[n] = pref (-2 alpha)^n F_n(T), n <= L (see hermite_R for the two branches).
template <int L>
__device__ __forceinline__ void hermite_seeds(double cc, double wb, double wk, double R2, const double2* __restrict__ tab,
                                              double (&s)[L + 1])
{
    const double w = wb + wk;
    const bool near = R2 < w;
    const double rs = rsqrt_fast(near ? w : R2);             // one rsqrt serves both branches of a mixed warp
    if (near) {
        const double alpha = 36.0 * (rs * rs);
        double F[L + 1];
        boys_near<L>(alpha * R2, tab, F);
        double sc = cc * 6.77027500257307544338 * rs;        // 12 / sqrt(pi)
#pragma unroll
        for (int n = 0; n <= L; ++n) {
            s[n] = sc * F[n];
            sc *= -2.0 * alpha;
        }
    } else {
        s[0] = cc * rs;
        const double wn = -(rs * rs);                        // -1/R^2
#pragma unroll
        for (int n = 0; n < L; ++n) s[n + 1] = ((2 * n + 1) * wn) * s[n];
    }
}

// SCALED: the table is returned as gs^(t+u+v) R_{tuv} (the operator stages of eri_prim_accum then need no multiply by
// their 1/2p: see apply_p); the powers of gs ride along the recursion, r~^n_{t+1,u,v} = (gs X) r~^{n+1}_{tuv} +
// (t gs^2) r~^{n+1}_{t-1,u,v}, at the price of five multiplies per primitive quartet.
template <int L, bool SCALED = false>
__device__ __forceinline__ void hermite_R(double cc, double wb, double wk, double X, double Y, double Z,
                                          const double2* __restrict__ tab, double (&R0)[nherm(L)], double gs = 1.0)
{
    double r[L + 1][nherm(L)];
    const double R2 = fma(X, X, fma(Y, Y, Z * Z));
    double seeds[L + 1];
    hermite_seeds<L>(cc, wb, wk, R2, tab, seeds);
#pragma unroll
    for (int n = 0; n <= L; ++n) r[n][0] = seeds[n];
    if (SCALED) { X *= gs; Y *= gs; Z *= gs; }
    const double g2 = SCALED ? gs * gs : 1.0;                // multiplies the (t-1) factors below
#pragma unroll
    for (int N = 1; N <= L; ++N)
#pragma unroll
        for (int n = 0; n <= L - N; ++n)
#pragma unroll
            for (int t = N; t >= 0; --t)
#pragma unroll
                for (int u = N - t; u >= 0; --u) {
                    const int v = N - t - u;
                    double val;
                    if (t > 0) {
                        val = X * r[n + 1][hidx(t - 1, u, v)];
                        if (t > 1) val = fma((double)(t - 1) * g2, r[n + 1][hidx(t - 2, u, v)], val);
                    } else if (u > 0) {
                        val = Y * r[n + 1][hidx(t, u - 1, v)];
                        if (u > 1) val = fma((double)(u - 1) * g2, r[n + 1][hidx(t, u - 2, v)], val);
                    } else {
                        val = Z * r[n + 1][hidx(t, u, v - 1)];
                        if (v > 1) val = fma((double)(v - 1) * g2, r[n + 1][hidx(t, u, v - 2)], val);
                    }
                    r[n][hidx(t, u, v)] = val;
                }
#pragma unroll
    for (int i = 0; i < nherm(L); ++i) R0[i] = r[0][i];
}

// One operator application: out[c][h] = X[c] * in[h] + g * in[h + e_c] for |h| <= LOUT (g = +1/2p for bra
// functions, -1/2q for ket functions).  NC = 1 means "s function": plain copy of the first nherm(LOUT).
// SCALED: the tables carry g^(order) (hermite_R<L, true>, rescale_orders), so that g * in[h + e_c] is in[h + e_c] itself
// and a stage is one FMA per output.
template <int NC, int LOUT, int NBLK, bool SCALED = false>
__device__ __forceinline__ void apply_p(const double (&in)[NBLK][nherm(LOUT + (NC == 3 ? 1 : 0))],
                                        const double* X, double g, double (&out)[NBLK * NC][nherm(LOUT)])
{
#pragma unroll
    for (int b = 0; b < NBLK; ++b) {
        if (NC == 1) {
#pragma unroll
            for (int h = 0; h < nherm(LOUT); ++h) out[b][h] = in[b][h];
        } else {
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int t = LOUT; t >= 0; --t)
#pragma unroll
                    for (int u = LOUT - t; u >= 0; --u)
#pragma unroll
                        for (int v = LOUT - t - u; v >= 0; --v)
                            out[b * 3 + c][hidx(t, u, v)] =
                                fma(X[c], in[b][hidx(t, u, v)], SCALED ? in[b][hidx_plus(t, u, v, c)] : g * in[b][hidx_plus(t, u, v, c)]);
        }
    }
}

// Primitive pair view (registers or pointers already resolved by the caller).  p and c hold the SCALED quantities
// w = 36/p and c' = c pi^(1/4)/sqrt(2p) (see hermite_R) once to_scaled() has been applied to a table row.
struct PrimPair {
    double p, Px, Py, Pz, c, inv2p;
    double two_p;   // 2p = 1 / inv2p (set by to_scaled; used for kets only)
    double XA[3];   // P - (first centre)
    double XB[3];   // P - (second centre)
};

__device__ __forceinline__ void to_scaled(PrimPair& r)
{
    r.two_p = 2.0 * r.p;
    r.c *= 1.33133536380038971280 * rsqrt(2.0 * r.p);        // pi^(1/4)
    r.p = 36.0 / r.p;
}

// Accumulate the primitive block into I[ia][ib][ic][id] (flattened, d fastest).
// Order of operator application: d, c (ket; g = -1/2q), then b, a (bra; g = +1/2p).  The flattened block
// index after the four stages is ((d*NC + c)*NB + b)*NA + a, so the caller reads I through eri_index().
template <int LA, int LB, int LC, int LD>
__device__ __forceinline__ void eri_prim_accum(const PrimPair& br, const PrimPair& kt,
                                               const double2* __restrict__ tab,
                                               double (&I)[(2 * LA + 1) * (2 * LB + 1) * (2 * LC + 1) * (2 * LD + 1)])
{
    constexpr int L = LA + LB + LC + LD;
    constexpr int NA = 2 * LA + 1, NB = 2 * LB + 1, NC = 2 * LC + 1, ND = 2 * LD + 1;
    // Scaled stages (RTTDA_SCALED_STAGES): the Hermite tables carry g^(order), g = -1/2q while the ket operators are
    // applied and +1/2p for the bra operators, so that a stage costs one FMA per output instead of a multiply and an
    // FMA; between the two phases the (few) remaining entries are rescaled by (g_bra / g_ket)^(order).
    if constexpr (RTTDA_FUSED_L1 && LA == 1 && LB + LC + LD == 0) {
        // (ps|ss): (a_c b|cd) = X_PA,c R_000 + (1/2p) R_{e_c}, R_{e_c} = (P-Q)_c r^1_000: two FMAs per component straight
        // into the accumulators, no table
        const double X = br.Px - kt.Px, Y = br.Py - kt.Py, Z = br.Pz - kt.Pz;
        double sd[2];
        hermite_seeds<1>(br.c * kt.c, br.p, kt.p, fma(X, X, fma(Y, Y, Z * Z)), tab, sd);
        const double q = br.inv2p * sd[1];
        I[0] = fma(X, q, fma(br.XA[0], sd[0], I[0]));
        I[1] = fma(Y, q, fma(br.XA[1], sd[0], I[1]));
        I[2] = fma(Z, q, fma(br.XA[2], sd[0], I[2]));
        return;
    }
    constexpr bool SC = RTTDA_SCALED_STAGES && L >= 2;
    constexpr bool KET_PHASE = LC + LD > 0, BRA_PHASE = LA + LB > 0;
    const double gk = -kt.inv2p, gb = br.inv2p;
    double V0[1][nherm(L)];
    hermite_R<L, SC>(br.c * kt.c, br.p, kt.p, br.Px - kt.Px, br.Py - kt.Py, br.Pz - kt.Pz, tab, V0[0], KET_PHASE ? gk : gb);
    double VD[ND][nherm(L - LD)];
    apply_p<ND, L - LD, 1, SC>(V0, kt.XB, gk, VD);
    double VC[ND * NC][nherm(L - LD - LC)];
    apply_p<NC, L - LD - LC, ND, SC>(VD, kt.XA, gk, VC);
    // The operators above treat X_QC, X_QD as constants; two p functions on one pair with the SAME Cartesian
    // component pick up the extra term of E_0^{11} = X_PA X_PB + 1/2p (x_P Lambda_1 = Lambda_2/2p + Lambda_0).
    if constexpr (LC == 1 && LD == 1) {
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int hh = 0; hh < nherm(L - LD - LC); ++hh)
                VC[c * NC + c][hh] = fma(kt.inv2p, V0[0][hh], VC[c * NC + c][hh]);
    }
    if constexpr (SC && KET_PHASE && BRA_PHASE) {              // g_ket^(order) -> g_bra^(order)
        const double rho = -(br.inv2p * kt.two_p), rho2 = rho * rho;
#pragma unroll
        for (int dc = 0; dc < ND * NC; ++dc)
#pragma unroll
            for (int hh = 1; hh < nherm(LA + LB); ++hh) VC[dc][hh] *= (hh < nherm(1) ? rho : rho2);
    }
    double VB[ND * NC * NB][nherm(LA)];
    apply_p<NB, LA, ND * NC, SC>(VC, br.XB, gb, VB);
    double VA[ND * NC * NB * NA][1];
    apply_p<NA, 0, ND * NC * NB, SC>(VB, br.XA, gb, VA);
    if constexpr (LA == 1 && LB == 1) {
#pragma unroll
        for (int dc = 0; dc < ND * NC; ++dc)
#pragma unroll
            for (int a = 0; a < 3; ++a)
                VA[(dc * NB + a) * NA + a][0] = fma(br.inv2p, VC[dc][0], VA[(dc * NB + a) * NA + a][0]);
    }
#pragma unroll
    for (int i = 0; i < NA * NB * NC * ND; ++i) I[i] += VA[i][0];
}

// flattened index of component (a, b, c, d) in the block produced by eri_prim_accum
template <int LA, int LB, int LC, int LD>
__host__ __device__ constexpr int eri_index(int a, int b, int c, int d)
{
    return ((d * (2 * LC + 1) + c) * (2 * LB + 1) + b) * (2 * LA + 1) + a;
}

__device__ __forceinline__ PrimPair load_prim_aos(const double* __restrict__ row)
{
    PrimPair r;
    r.p = __ldg(row + 0); r.Px = __ldg(row + 1); r.Py = __ldg(row + 2); r.Pz = __ldg(row + 3);
    r.c = __ldg(row + 4); r.inv2p = __ldg(row + 5);
    r.XA[0] = __ldg(row + 6); r.XA[1] = __ldg(row + 7); r.XA[2] = __ldg(row + 8);
    r.XB[0] = __ldg(row + 9); r.XB[1] = __ldg(row + 10); r.XB[2] = __ldg(row + 11);
    return r;
}

// SoA: element f of primitive k of ket q sits at prim[(k*PRIM_STRIDE + f)*n + q]
__device__ __forceinline__ PrimPair load_prim_soa(const double* __restrict__ prim, int n, int k, int q)
{
    const double* b = prim + (size_t)k * PRIM_STRIDE * n + q;
    PrimPair r;
    r.p = __ldg(b); r.Px = __ldg(b + n); r.Py = __ldg(b + 2 * (size_t)n); r.Pz = __ldg(b + 3 * (size_t)n);
    r.c = __ldg(b + 4 * (size_t)n); r.inv2p = __ldg(b + 5 * (size_t)n);
    r.XA[0] = __ldg(b + 6 * (size_t)n); r.XA[1] = __ldg(b + 7 * (size_t)n); r.XA[2] = __ldg(b + 8 * (size_t)n);
    r.XB[0] = __ldg(b + 9 * (size_t)n); r.XB[1] = __ldg(b + 10 * (size_t)n); r.XB[2] = __ldg(b + 11 * (size_t)n);
    return r;
}

}  // namespace rttda
