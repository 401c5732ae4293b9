// General-angular-momentum path (Cartesian d shells, the paper's 6-31G* basis): every shell
// quartet class with at least one d shell, up to (dd|dd), is evaluated and digested here.  The s/p classes keep their
// unrolled register kernels (jk_eval.cu, jk_digest.cu); this file trades speed for generality - Hermite tables live in
// per-thread local memory, loops are run-time bounded, the digestion applies the eight index images of every stored
// integral with atomics - and shares the staging-buffer layout, the screening rules and the weights with the fast path:
//   value(bra pair p, ket q, component i) at ((batch_base[p] + (q >> 5) - (same ? p >> 5 : 0)) * NI + i) * 32 + (q & 31),
//   i = ((d * NC + c) * NB + b) * NA + a, a = component of the bra pair's first (higher-l) shell,
//   stored with the weights 1/2 (ket pair diagonal) and 1/2 (bra pair == ket pair) folded in, zeros where no quartet is.
// McMurchie-Davidson scheme (P:130 refs 88-91), primitive quartet by primitive quartet:
//   (ab|cd) = c_b c_k / sqrt(p+q) sum_{tuv} E^{ab}_{tuv} sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'} R_{t+t',u+u',v+v'}
// with E_0^{00} = 1 (the Gaussian-product factors sit in the row entry c), R^n_{000} = (-2 alpha)^n F_n(alpha |PQ|^2).
// d components: xx, xy, xz, yy, yz, zz, each normalised (reading R11: xy, xz, yz carry sqrt(3)).
#include <cstdlib>
#include "common.cuh"

namespace rttda {

namespace {

constexpr int GEN_LMAX = 2;
constexpr int GEN_NHERM = 165;      // Hermite components up to total order 8
constexpr int GEN_NHB = 35;         // ... up to order 4 (one pair)

__host__ __device__ inline int gen_ncart(int l) { return (l + 1) * (l + 2) / 2; }
__host__ __device__ inline int gen_nherm(int L) { return (L + 1) * (L + 2) * (L + 3) / 6; }
// compact index of Hermite component (t,u,v): by total order N, then N - t, then v
__device__ __forceinline__ int gen_hidx(int t, int u, int v)
{
    const int N = t + u + v;
    return N * (N + 1) * (N + 2) / 6 + (u + v) * (u + v + 1) / 2 + v;
}

__device__ __forceinline__ void gen_pow(int l, int c, int (&pw)[3])
{
    pw[0] = pw[1] = pw[2] = 0;
    if (l == 1) pw[c] = 1;
    if (l == 2) {
        // xx xy xz yy yz zz
        const int first = c < 3 ? 0 : (c < 5 ? 1 : 2);
        const int second = c < 3 ? c : (c < 5 ? c - 2 : 2);
        pw[first] += 1; pw[second] += 1;
    }
}
__device__ __forceinline__ double gen_norm(int l, int c)
{
    return (l == 2 && (c == 1 || c == 2 || c == 4)) ? 1.7320508075688772935 : 1.0;
}

// Boys function F_0..F_L(T).  T < 36: F_L from the table row of the nearest grid point T0 = j/8 ({F_{L+k}(T0)/k!, k < 8;
// e^-T0}, built in long double by setup.cu: F_L(T) = sum_k h_k (T0 - T)^k since dF_n/dT = -F_{n+1}), then the stable
// downward recursion F_{n-1} = (2T F_n + e^-T)/(2n - 1) with e^-T = e^-T0 e^(T0 - T) by its Taylor series;
// T >= 36: F_0 = sqrt(pi/T)/2 (erfc(6) = 2e-17) and the upward recursion, stable there, with its e^-T term.
__device__ void gen_boys(int L, double T, const double2* __restrict__ tab, double* F)
{
    if (T < BOYS_TMAX) {
        constexpr double MAGIC = 6755399441055744.0;      // 1.5 * 2^52: rounds to nearest integer
        const double t = fma(T, 8.0, MAGIC);
        const int j = __double2loint(t);
        const double dx = fma(t - MAGIC, 0.125, -T);      // T0 - T, |dx| <= 1/16
        const double2* row = tab + j * (BOYS_ROW / 2);
        const double2 h01 = row[0], h23 = row[1], h45 = row[2], h67 = row[3];
        double f = h67.y;
        f = fma(f, dx, h67.x); f = fma(f, dx, h45.y); f = fma(f, dx, h45.x); f = fma(f, dx, h23.y);
        f = fma(f, dx, h23.x); f = fma(f, dx, h01.y); f = fma(f, dx, h01.x);
        F[L] = f;
        double e = 1.0 / 40320.0;
        e = fma(e, dx, 1.0 / 5040.0); e = fma(e, dx, 1.0 / 720.0); e = fma(e, dx, 1.0 / 120.0); e = fma(e, dx, 1.0 / 24.0);
        e = fma(e, dx, 1.0 / 6.0); e = fma(e, dx, 0.5); e = fma(e, dx, 1.0); e = fma(e, dx, 1.0);
        e *= row[4].x;
        for (int n = L; n >= 1; --n) { f = fma(2.0 * T, f, e) / (2 * n - 1); F[n - 1] = f; }
    } else {
        const double emt = exp(-T), r = 0.5 / T;
        double f = 0.5 * sqrt(3.14159265358979323846 / T);
        F[0] = f;
        for (int n = 0; n < L; ++n) { f = ((2 * n + 1) * f - emt) * r; F[n + 1] = f; }
    }
}

// E[x][i][j][t], i <= li, j <= lj, with the Gaussian-product factor taken out (E_0^{00} = 1):
//   E_t^{i+1,j} = h E_{t-1}^{ij} + XA E_t^{ij} + (t+1) E_{t+1}^{ij},  E_t^{i,j+1} likewise with XB;  h = 1/(2p)
typedef double ETable[3][GEN_LMAX + 1][GEN_LMAX + 1][2 * GEN_LMAX + 1];
__device__ void gen_build_E(int li, int lj, double h, const double* XA, const double* XB, ETable& E)
{
    for (int x = 0; x < 3; ++x) {
        for (int i = 0; i <= li; ++i)
            for (int j = 0; j <= lj; ++j)
                for (int t = 0; t <= li + lj; ++t) E[x][i][j][t] = 0.0;
        E[x][0][0][0] = 1.0;
        for (int i = 0; i < li; ++i)
            for (int t = 0; t <= i + 1; ++t) {
                const double em = t > 0 ? E[x][i][0][t - 1] : 0.0;
                const double e0 = t <= i ? E[x][i][0][t] : 0.0;
                const double ep = t + 1 <= i ? E[x][i][0][t + 1] : 0.0;
                E[x][i + 1][0][t] = h * em + XA[x] * e0 + (t + 1) * ep;
            }
        for (int i = 0; i <= li; ++i)
            for (int j = 0; j < lj; ++j)
                for (int t = 0; t <= i + j + 1; ++t) {
                    const double em = t > 0 ? E[x][i][j][t - 1] : 0.0;
                    const double e0 = t <= i + j ? E[x][i][j][t] : 0.0;
                    const double ep = t + 1 <= i + j ? E[x][i][j][t + 1] : 0.0;
                    E[x][i][j + 1][t] = h * em + XB[x] * e0 + (t + 1) * ep;
                }
    }
}

// R^0_{tuv}, t+u+v <= L, times `pref`; two ping-pong tables, level n built from level n+1:
//   R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + X R^{n+1}_{t,u,v}   (u with Y, v with Z alike)
// Returns the table that holds level 0.
__device__ double* gen_build_R(int L, double pref, double alpha, double X, double Y, double Z, const double2* __restrict__ tab,
                               double* Ra, double* Rb)
{
    double F[4 * GEN_LMAX + 1];
    gen_boys(L, alpha * (X * X + Y * Y + Z * Z), tab, F);
    double sc = pref;
    for (int n = 0; n <= L; ++n) { F[n] *= sc; sc *= -2.0 * alpha; }
    for (int n = L; n >= 0; --n) {
        double* cur = (n & 1) ? Ra : Rb;
        const double* prev = (n & 1) ? Rb : Ra;
        cur[0] = F[n];
        for (int N = 1; N <= L - n; ++N)
            for (int t = N; t >= 0; --t)
                for (int u = N - t; u >= 0; --u) {
                    const int v = N - t - u;
                    double val;
                    if (t > 0) val = (t > 1 ? (t - 1) * prev[gen_hidx(t - 2, u, v)] : 0.0) + X * prev[gen_hidx(t - 1, u, v)];
                    else if (u > 0) val = (u > 1 ? (u - 1) * prev[gen_hidx(t, u - 2, v)] : 0.0) + Y * prev[gen_hidx(t, u - 1, v)];
                    else val = (v > 1 ? (v - 1) * prev[gen_hidx(t, u, v - 2)] : 0.0) + Z * prev[gen_hidx(t, u, v - 1)];
                    cur[gen_hidx(t, u, v)] = val;
                }
    }
    return Rb;
}

struct GenPrim {
    double p, P[3], c, h, XA[3], XB[3];
};
__device__ __forceinline__ GenPrim gen_load_aos(const double* __restrict__ r)
{
    GenPrim g;
    g.p = r[0]; g.P[0] = r[1]; g.P[1] = r[2]; g.P[2] = r[3]; g.c = r[4]; g.h = r[5];
    g.XA[0] = r[6]; g.XA[1] = r[7]; g.XA[2] = r[8]; g.XB[0] = r[9]; g.XB[1] = r[10]; g.XB[2] = r[11];
    return g;
}
__device__ __forceinline__ GenPrim gen_load_soa(const double* __restrict__ prim, int n, int k, int q)
{
    const double* b = prim + (size_t)k * PRIM_STRIDE * n + q;
    const size_t N = (size_t)n;
    GenPrim g;
    g.p = b[0]; g.P[0] = b[N]; g.P[1] = b[2 * N]; g.P[2] = b[3 * N]; g.c = b[4 * N]; g.h = b[5 * N];
    g.XA[0] = b[6 * N]; g.XA[1] = b[7 * N]; g.XA[2] = b[8 * N]; g.XB[0] = b[9 * N]; g.XB[1] = b[10 * N]; g.XB[2] = b[11 * N];
    return g;
}

// The Hermite table of one primitive quartet: R (level 0) for total order L with the prefactor c_b c_k / sqrt(p+q)
// (times theta for the operator erf(omega r12)/r12, whose integrals are those of 1/r12 at alpha theta^2,
// theta^2 = omega^2 / (alpha + omega^2)).
__device__ double* gen_quartet_R(int L, const GenPrim& b, const GenPrim& k, double omega2, const double2* __restrict__ tab,
                                 double* Ra, double* Rb)
{
    const double pq = b.p + k.p;
    double alpha = b.p * k.p / pq;
    double pref = b.c * k.c / sqrt(pq);
    if (omega2 > 0.0) {
        const double th2 = omega2 / (alpha + omega2);
        pref *= sqrt(th2);
        alpha *= th2;
    }
    return gen_build_R(L, pref, alpha, b.P[0] - k.P[0], b.P[1] - k.P[1], b.P[2] - k.P[2], tab, Ra, Rb);
}

// G[tuv] = sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'} R_{t+t',u+u',v+v'} for all bra Hermite components of order <= LB
__device__ void gen_contract_ket(int LB, const ETable& Ek, const int (&pc)[3], const int (&pd)[3], const double* R, double* G)
{
    const int kx = pc[0] + pd[0], ky = pc[1] + pd[1], kz = pc[2] + pd[2];
    const double* ex = Ek[0][pc[0]][pd[0]];
    const double* ey = Ek[1][pc[1]][pd[1]];
    const double* ez = Ek[2][pc[2]][pd[2]];
    for (int N = 0; N <= LB; ++N)
        for (int t = N; t >= 0; --t)
            for (int u = N - t; u >= 0; --u) {
                const int v = N - t - u;
                double s = 0.0;
                for (int t2 = 0; t2 <= kx; ++t2)
                    for (int u2 = 0; u2 <= ky; ++u2) {
                        const double exy = ex[t2] * ey[u2];
                        for (int v2 = 0; v2 <= kz; ++v2) {
                            const double e = exy * ez[v2];
                            const double r = R[gen_hidx(t + t2, u + u2, v + v2)];
                            s += ((t2 + u2 + v2) & 1) ? -e * r : e * r;
                        }
                    }
                G[gen_hidx(t, u, v)] = s;
            }
}

__device__ double gen_contract_bra(const ETable& Eb, const int (&pa)[3], const int (&pb)[3], const double* G)
{
    const double* ex = Eb[0][pa[0]][pb[0]];
    const double* ey = Eb[1][pa[1]][pb[1]];
    const double* ez = Eb[2][pa[2]][pb[2]];
    double s = 0.0;
    for (int t = 0; t <= pa[0] + pb[0]; ++t)
        for (int u = 0; u <= pa[1] + pb[1]; ++u)
            for (int v = 0; v <= pa[2] + pb[2]; ++v) s += ex[t] * ey[u] * ez[v] * G[gen_hidx(t, u, v)];
    return s;
}

struct GenEvalArgs {
    const EvalItem* items;
    KetClass bra, ket;
    const long long* batch_base;
    const double2* boys;                 // table of the segment's total angular momentum
    double* buf;
    double tau, omega2;
    unsigned long long* primcount;
    unsigned long long flops_per_prim;   // flop model of one primitive quartet of this class (setup.cu)
    int same, la, lb, lc, ld;
};

// block = 32 consecutive kets (lane = ket pair) x GEN_WORKERS warps x a run of bra pairs (the EvalItem of the fast path
// with a 32-ket stride).  The warps of a block work on the SAME quartets and split their components: warp w owns the ket
// component pairs (c, d) with (d NC + c) % GEN_WORKERS == w, or - when the ket has fewer than GEN_WORKERS of them - the
// bra component pairs (a, b) likewise; every warp builds the (cheap) Hermite tables of the primitive quartet for itself.
constexpr int GEN_WORKERS = 4;
__global__ void __launch_bounds__(32 * GEN_WORKERS) eval_generic_kernel(GenEvalArgs g)
{
    const EvalItem it = g.items[blockIdx.x];
    const int la = g.la, lb = g.lb, lc = g.lc, ld = g.ld;
    const int NA = gen_ncart(la), NB = gen_ncart(lb), NC = gen_ncart(lc), ND = gen_ncart(ld);
    const int NI = NA * NB * NC * ND, L = la + lb + lc + ld, LB = la + lb;
    const int lane = threadIdx.x & 31, worker = threadIdx.x >> 5, nworker = blockDim.x >> 5;
    const bool split_ket = NC * ND >= nworker;
    const int q = it.k0 + lane;
    const bool active = q < g.ket.n;
    const int qq = active ? q : g.ket.n - 1;
    const double Qq = active ? g.ket.Q[qq] : 0.0;
    const double wcd = g.ket.same[qq] ? 0.5 : 1.0;
    const int npb = g.bra.np, npk = g.ket.np;
    double Ra[GEN_NHERM], Rb[GEN_NHERM], G[GEN_NHB];
    ETable Ek;
    // the bra pair is block-uniform: its primitives and their Hermite E tables are built once per pair in shared memory
    __shared__ ETable s_Eb[9];
    __shared__ GenPrim s_bp[9];
    unsigned long long nprim_done = 0;

    for (int p = it.p_begin; p < it.p_end; ++p) {
        const double Qp = g.bra.Q[p];
        const bool ok = active && (Qp * Qq >= g.tau) && (!g.same || p <= q);
        if (!__any_sync(0xffffffffu, ok)) break;           // both conditions only get worse along the bra list; the warps
                                                           // of a block hold the same kets, so the exit is block-uniform
        __syncthreads();                                   // everyone is done with the previous pair's tables
        if (threadIdx.x < npb) {
            const GenPrim bp = gen_load_aos(g.bra.prim_aos + ((size_t)p * npb + threadIdx.x) * PRIM_STRIDE);
            s_bp[threadIdx.x] = bp;
            gen_build_E(la, lb, bp.h, bp.XA, bp.XB, s_Eb[threadIdx.x]);
        }
        __syncthreads();
        const long long batch = g.batch_base[p] + (q >> 5) - (g.same ? (p >> 5) : 0);
        double* dst = g.buf + (size_t)batch * ((size_t)NI * 32) + lane;
        if (!ok) {                                         // the batch exists: lanes without a quartet store zeros
            for (int i = worker; i < NI; i += nworker) dst[(size_t)i * 32] = 0.0;
            continue;
        }
        const double w = (g.same && p == q) ? 0.5 * wcd : wcd;
        bool first = true;
        for (int kk = 0; kk < npk; ++kk) {
            const GenPrim kp = gen_load_soa(g.ket.prim, g.ket.n, kk, qq);
            gen_build_E(lc, ld, kp.h, kp.XA, kp.XB, Ek);
            for (int kb = 0; kb < npb; ++kb) {
                const double* R = gen_quartet_R(L, s_bp[kb], kp, g.omega2, g.boys, Ra, Rb);
                const ETable& Eb = s_Eb[kb];
                if (worker == 0) ++nprim_done;
                for (int cd = 0; cd < NC * ND; ++cd) {
                    if (split_ket && cd % nworker != worker) continue;
                    const int c = cd % NC, d = cd / NC;
                    int pc[3], pd[3];
                    gen_pow(lc, c, pc); gen_pow(ld, d, pd);
                    gen_contract_ket(LB, Ek, pc, pd, R, G);
                    const double ncd = w * gen_norm(lc, c) * gen_norm(ld, d);
                    for (int ab = 0; ab < NA * NB; ++ab) {
                        if (!split_ket && ab % nworker != worker) continue;
                        const int a = ab % NA, b = ab / NA;
                        int pa[3], pb[3];
                        gen_pow(la, a, pa); gen_pow(lb, b, pb);
                        const double val = ncd * gen_norm(la, a) * gen_norm(lb, b) * gen_contract_bra(Eb, pa, pb, G);
                        double* o = dst + (size_t)(cd * (NA * NB) + ab) * 32;
                        *o = first ? val : *o + val;
                    }
                }
                first = false;
            }
        }
    }
    for (int o = 16; o > 0; o >>= 1) nprim_done += __shfl_xor_sync(0xffffffffu, nprim_done, o);
    if (lane == 0 && nprim_done) {                                           // slots 5, 6: all general-path classes
        atomicAdd(g.primcount + 5, nprim_done);
        atomicAdd(g.primcount + 6, nprim_done * g.flops_per_prim);
    }
}

// Schwarz bounds of pairs with a d shell: Q = sqrt(max_{components} (ab|ab)), thread = pair.
__global__ void schwarz_generic_kernel(int la, int lb, int npairs, const int* __restrict__ np, const int* __restrict__ off,
                                       const double* __restrict__ prim, const double2* __restrict__ boys, double* __restrict__ Q)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npairs) return;
    const int NA = gen_ncart(la), NB = gen_ncart(lb), LB = la + lb;
    double Ra[GEN_NHERM], Rb[GEN_NHERM], G[GEN_NHB], diag[36];
    ETable Eb, Ek;
    for (int k = 0; k < NA * NB; ++k) diag[k] = 0.0;
    const int n = np[i], o = off[i];
    for (int k1 = 0; k1 < n; ++k1) {
        const GenPrim bp = gen_load_aos(prim + (size_t)(o + k1) * PRIM_STRIDE);
        gen_build_E(la, lb, bp.h, bp.XA, bp.XB, Eb);
        for (int k2 = 0; k2 < n; ++k2) {
            const GenPrim kp = gen_load_aos(prim + (size_t)(o + k2) * PRIM_STRIDE);
            gen_build_E(la, lb, kp.h, kp.XA, kp.XB, Ek);
            const double* R = gen_quartet_R(2 * LB, bp, kp, 0.0, boys, Ra, Rb);
            for (int b = 0; b < NB; ++b)
                for (int a = 0; a < NA; ++a) {
                    int pa[3], pb[3];
                    gen_pow(la, a, pa); gen_pow(lb, b, pb);
                    gen_contract_ket(LB, Ek, pa, pb, R, G);
                    const double nn = gen_norm(la, a) * gen_norm(lb, b);
                    diag[b * NA + a] += nn * nn * gen_contract_bra(Eb, pa, pb, G);
                }
        }
    }
    double m = 0.0;
    for (int k = 0; k < NA * NB; ++k) m = fmax(m, diag[k]);
    Q[i] = sqrt(m);
}

struct GenDigestArgs {
    KetClass bra, ket;
    const long long* batch_base;
    const double* buf;
    const double* Tq;
    double* Fq;
    double cx;
    long long nbatch;
    int same, nvt, nvec, nao, la, lb, lc, ld, do_j, do_k;
};

// block = one stored batch (bra pair (m n) x 32 kets (l s)), lane = ket, GEN_DV densities per sweep.  Every stored value I
// stands for its eight index images (mn|ls) (nm|ls) (mn|sl) (nm|sl) (ls|mn) (sl|mn) (ls|nm) (sl|nm), with 1/2 per
// coincidence (a == b here; c == d and ab == cd are folded into the stored value):
//   Coulomb   F[mn], F[nm] += 2 sum_{ls} I (T_ls + T_sl)        F[ls], F[sl] += 2 sum_{mn} I (T_mn + T_nm)
//   exchange  F[ml] -= cx sum_{ns} I T_ns   F[lm] -= cx sum I T_sn     F[nl] -= cx sum_{ms} I T_ms   F[ln] -= cx sum I T_sm
//             F[ms] -= cx sum_{nl} I T_nl   F[sm] -= cx sum I T_ln     F[ns] -= cx sum_{ml} I T_ml   F[sn] -= cx sum I T_lm
// Each line is one sweep over the batch: the warps split the OUTPUT index pair, a lane sums over the other two indices
// in registers and issues one atomic per output element and density (the F[mn] sums go through a warp reduction first).
constexpr int GEN_DV = 4;
template <bool OUT_A, bool OUT_C>
__device__ __forceinline__ void gen_exchange_sweep(const GenDigestArgs& g, const double* __restrict__ src, int NA, int NB, int NC,
                                                   int ND, int aoA, int aoB, int aoC, int aoD, double scale, int v0, int nv,
                                                   int warp, int nwarp, bool live)
{
    // output pair (o1, o2): o1 from the bra (a if OUT_A else b), o2 from the ket (c if OUT_C else d); summed pair (r1, r2)
    const int NO1 = OUT_A ? NA : NB, NO2 = OUT_C ? NC : ND, NR1 = OUT_A ? NB : NA, NR2 = OUT_C ? ND : NC;
    const int aoO1 = OUT_A ? aoA : aoB, aoO2 = OUT_C ? aoC : aoD, aoR1 = OUT_A ? aoB : aoA, aoR2 = OUT_C ? aoD : aoC;
    const size_t nvt = g.nvt, rs = (size_t)g.nao * nvt;
    for (int o = warp; o < NO1 * NO2; o += nwarp) {
        const int o1 = o % NO1, o2 = o / NO1;
        double acc1[GEN_DV], acc2[GEN_DV];
        for (int v = 0; v < GEN_DV; ++v) acc1[v] = acc2[v] = 0.0;
        for (int r2 = 0; r2 < NR2; ++r2)
            for (int r1 = 0; r1 < NR1; ++r1) {
                const int a = OUT_A ? o1 : r1, b = OUT_A ? r1 : o1, c = OUT_C ? o2 : r2, d = OUT_C ? r2 : o2;
                const double x = src[(size_t)(((d * NC + c) * NB + b) * NA + a) * 32];
                const double* T12 = g.Tq + (size_t)(aoR1 + r1) * rs + (size_t)(aoR2 + r2) * nvt + v0;
                const double* T21 = g.Tq + (size_t)(aoR2 + r2) * rs + (size_t)(aoR1 + r1) * nvt + v0;
                for (int v = 0; v < GEN_DV; ++v)
                    if (v < nv) { acc1[v] = fma(x, T12[v], acc1[v]); acc2[v] = fma(x, T21[v], acc2[v]); }
            }
        if (live) {
            double* F12 = g.Fq + (size_t)(aoO1 + o1) * rs + (size_t)(aoO2 + o2) * nvt + v0;
            double* F21 = g.Fq + (size_t)(aoO2 + o2) * rs + (size_t)(aoO1 + o1) * nvt + v0;
            for (int v = 0; v < GEN_DV; ++v)
                if (v < nv) {
                    if (acc1[v] != 0.0) atomicAdd(F12 + v, scale * acc1[v]);
                    if (acc2[v] != 0.0) atomicAdd(F21 + v, scale * acc2[v]);
                }
        }
    }
}

__global__ void __launch_bounds__(128) digest_generic_kernel(GenDigestArgs g)
{
    const long long batch = blockIdx.x;
    const int nb = g.bra.n;
    int lo = 0, hi = nb;                                   // last pair whose first batch is <= batch
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (g.batch_base[mid] <= batch) lo = mid + 1; else hi = mid;
    }
    const int p = lo - 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const long long kbi = batch - g.batch_base[p] + (g.same ? (p >> 5) : 0);
    const long long q = kbi * 32 + lane;
    const bool live = q < g.ket.n;                         // lanes beyond the ket list hold zeros; they only help to reduce
    const long long qq = live ? q : g.ket.n - 1;
    const int NA = gen_ncart(g.la), NB = gen_ncart(g.lb), NC = gen_ncart(g.lc), ND = gen_ncart(g.ld);
    const int NAB = NA * NB, NCD = NC * ND, NI = NAB * NCD;
    const int aoA = g.bra.ao_c[p], aoB = g.bra.ao_d[p], aoC = g.ket.ao_c[qq], aoD = g.ket.ao_d[qq];
    const double wab = g.bra.same[p] ? 0.5 : 1.0;
    const size_t nvt = g.nvt, rs = (size_t)g.nao * nvt;
    const double* src = g.buf + (size_t)batch * ((size_t)NI * 32) + lane;
    for (int v0 = 0; v0 < g.nvec; v0 += GEN_DV) {
        const int nv = min(GEN_DV, g.nvec - v0);
        if (g.do_j) {
            // F[mn], F[nm] += 2 w sum_{ls} I (T_ls + T_sl), summed over the kets of the batch by a warp reduction
            for (int ab = warp; ab < NAB; ab += nwarp) {
                double acc[GEN_DV];
                for (int v = 0; v < GEN_DV; ++v) acc[v] = 0.0;
                for (int cd = 0; cd < NCD; ++cd) {
                    const int c = cd % NC, d = cd / NC;
                    const double x = src[(size_t)(cd * NAB + ab) * 32];
                    const double* Tls = g.Tq + (size_t)(aoC + c) * rs + (size_t)(aoD + d) * nvt + v0;
                    const double* Tsl = g.Tq + (size_t)(aoD + d) * rs + (size_t)(aoC + c) * nvt + v0;
                    for (int v = 0; v < GEN_DV; ++v)
                        if (v < nv) acc[v] = fma(x, Tls[v] + Tsl[v], acc[v]);
                }
                for (int v = 0; v < GEN_DV; ++v)
                    for (int o = 16; o > 0; o >>= 1) acc[v] += __shfl_xor_sync(0xffffffffu, acc[v], o);
                if (lane == 0) {
                    const int a = ab % NA, b = ab / NA;
                    double* Fmn = g.Fq + (size_t)(aoA + a) * rs + (size_t)(aoB + b) * nvt + v0;
                    double* Fnm = g.Fq + (size_t)(aoB + b) * rs + (size_t)(aoA + a) * nvt + v0;
                    for (int v = 0; v < nv; ++v) {
                        atomicAdd(Fmn + v, 2.0 * wab * acc[v]);
                        atomicAdd(Fnm + v, 2.0 * wab * acc[v]);
                    }
                }
            }
            // F[ls], F[sl] += 2 w sum_{mn} I (T_mn + T_nm)
            for (int cd = warp; cd < NCD; cd += nwarp) {
                const int c = cd % NC, d = cd / NC;
                double acc[GEN_DV];
                for (int v = 0; v < GEN_DV; ++v) acc[v] = 0.0;
                for (int ab = 0; ab < NAB; ++ab) {
                    const int a = ab % NA, b = ab / NA;
                    const double x = src[(size_t)(cd * NAB + ab) * 32];
                    const double* Tmn = g.Tq + (size_t)(aoA + a) * rs + (size_t)(aoB + b) * nvt + v0;
                    const double* Tnm = g.Tq + (size_t)(aoB + b) * rs + (size_t)(aoA + a) * nvt + v0;
                    for (int v = 0; v < GEN_DV; ++v)
                        if (v < nv) acc[v] = fma(x, Tmn[v] + Tnm[v], acc[v]);
                }
                if (live) {
                    double* Fls = g.Fq + (size_t)(aoC + c) * rs + (size_t)(aoD + d) * nvt + v0;
                    double* Fsl = g.Fq + (size_t)(aoD + d) * rs + (size_t)(aoC + c) * nvt + v0;
                    for (int v = 0; v < nv; ++v)
                        if (acc[v] != 0.0) {
                            atomicAdd(Fls + v, 2.0 * wab * acc[v]);
                            atomicAdd(Fsl + v, 2.0 * wab * acc[v]);
                        }
                }
            }
        }
        if (g.do_k) {
            const double sc = -g.cx * wab;
            gen_exchange_sweep<true, true>(g, src, NA, NB, NC, ND, aoA, aoB, aoC, aoD, sc, v0, nv, warp, nwarp, live);
            gen_exchange_sweep<false, true>(g, src, NA, NB, NC, ND, aoA, aoB, aoC, aoD, sc, v0, nv, warp, nwarp, live);
            gen_exchange_sweep<true, false>(g, src, NA, NB, NC, ND, aoA, aoB, aoC, aoD, sc, v0, nv, warp, nwarp, live);
            gen_exchange_sweep<false, false>(g, src, NA, NB, NC, ND, aoA, aoB, aoC, aoD, sc, v0, nv, warp, nwarp, live);
        }
    }
}

}  // namespace

bool segment_is_general(const Segment& sg) { return sg.la > 1 || sg.lb > 1 || sg.lc > 1 || sg.ld > 1; }

int eval_segment_general(Handle* h, const Segment& sg, double* buf, cudaStream_t st)
{
    if (!getenv("RTTDA_GENERIC_ONLY")) {               // classes up to L = 5 have unrolled kernels (jk_eval_d.cu)
        bool handled = false;
        RT_TRY(eval_segment_d(h, sg, buf, st, &handled));
        if (handled) return RTTDA_OK;
    }
    GenEvalArgs g;
    g.items = sg.items;
    g.bra = h->tabs.kets[sg.kc_bra];
    g.ket = h->tabs.kets[sg.kc_ket];
    g.batch_base = sg.batch_base;
    g.boys = h->tabs.boys[sg.la + sg.lb + sg.lc + sg.ld];
    g.buf = buf;
    g.tau = h->tabs.tau;
    g.omega2 = h->pass_w_extra > 0.0 ? 36.0 / h->pass_w_extra : 0.0;     // pass_w_extra = 36 / omega^2 (jk_build)
    g.primcount = h->d_primcount;
    g.flops_per_prim = (unsigned long long)flops_prim(sg.la, sg.lb, sg.lc, sg.ld);
    g.same = (sg.kc_bra == sg.kc_ket);
    g.la = sg.la; g.lb = sg.lb; g.lc = sg.lc; g.ld = sg.ld;
    // few components per quartet: the Hermite tables every worker builds for itself would dominate - fewer workers
    const int workers = sg.ni >= 100 ? GEN_WORKERS : (sg.ni >= 36 ? 2 : 1);
    eval_generic_kernel<<<dim3(sg.nitems), dim3(32 * workers), 0, st>>>(g);
    h->kernel_launches++;
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

int digest_segment_general(Handle* h, const Segment& sg, const double* buf, int nvt, int nvec, const double* Tq, double* Fq,
                           cudaStream_t st)
{
    if (sg.nbatch == 0) return RTTDA_OK;
    GenDigestArgs g;
    g.bra = h->tabs.kets[sg.kc_bra];
    g.ket = h->tabs.kets[sg.kc_ket];
    g.batch_base = sg.batch_base;
    g.buf = buf; g.Tq = Tq; g.Fq = Fq;
    g.cx = h->pass_cx;
    g.nbatch = sg.nbatch;
    g.same = (sg.kc_bra == sg.kc_ket);
    g.nvt = nvt; g.nvec = nvec; g.nao = h->nao;
    g.la = sg.la; g.lb = sg.lb; g.lc = sg.lc; g.ld = sg.ld;
    g.do_j = h->pass_do_j ? 1 : 0;
    g.do_k = (h->pass_do_k && h->pass_cx != 0.0) ? 1 : 0;
    RT_CHECK(sg.nbatch < 2147483647LL, "digest: too many batches in one general-path segment");
    digest_generic_kernel<<<dim3((unsigned)sg.nbatch), dim3(128), 0, st>>>(g);
    h->kernel_launches++;
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

int schwarz_general(int la, int lb, int npairs, const int* d_np, const int* d_off, const double* d_prim,
                    const double2* d_boys, double* d_Q, cudaStream_t st)
{
    if (npairs == 0) return RTTDA_OK;
    schwarz_generic_kernel<<<dim3((npairs + 63) / 64), dim3(64), 0, st>>>(la, lb, npairs, d_np, d_off, d_prim, d_boys, d_Q);
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

}  // namespace rttda
