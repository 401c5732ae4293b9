// Unrolled evaluation kernels for the shell-quartet classes with a d shell up to (dd|dp), L <= 7.
// Same block shape, staging layout, screening rules and weights as eval_generic_kernel (eri_generic.cu), which keeps
// (dd|dd); what differs is that every
// angular-momentum quantity is a template parameter, so all loops unroll, every Hermite index is a constant and the
// tables are registers (or local memory at fixed offsets) instead of run-time indexed arrays.
//
// McMurchie-Davidson with explicit Hermite coefficients (the operator form of eri_eval.cuh has no closed rule for two
// powers on one centre):
//   R_{tuv}                      hermite_R<L> of eri_eval.cuh (scaled primitive data, near/far Boys split)
//   E^{ab}, E^{cd} per axis      1-D recursion, Gaussian-product factor taken out (it sits in c')
//   G^{cd}_{tuv} = sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'} R_{t+t',u+u',v+v'}           |tuv| <= la + lb
//   (ab|cd) += n_a n_b n_c n_d sum_{tuv} E^{ab}_{tuv} G^{cd}_{tuv}
// block = 32 consecutive kets (lane = ket pair) x W warps x a run of bra pairs; the warps of a block work on the same
// quartets and split the ket component pairs (c, d): warp w owns those with (d NC + c) % W == w, accumulated in registers
// over the primitive quartets and stored once.
#include "eri_eval.cuh"

namespace rttda {

namespace {

__host__ __device__ constexpr int ncart_c(int l) { return (l + 1) * (l + 2) / 2; }
__host__ __device__ constexpr int cpow(int l, int c, int x)
{
    if (l == 0) return 0;
    if (l == 1) return c == x ? 1 : 0;
    // d: xx xy xz yy yz zz
    const int first = c < 3 ? 0 : (c < 5 ? 1 : 2);
    const int second = c < 3 ? c : (c < 5 ? c - 2 : 2);
    return (first == x ? 1 : 0) + (second == x ? 1 : 0);
}
__host__ __device__ constexpr double cnorm(int l, int c)
{
    return (l == 2 && (c == 1 || c == 2 || c == 4)) ? 1.7320508075688772935 : 1.0;
}

// E[i][j][t], i <= LI, j <= LJ, t <= i + j, with E_0^{00} = 1:
//   E_t^{i+1,j} = h E_{t-1}^{ij} + xa E_t^{ij} + (t+1) E_{t+1}^{ij},  E_t^{i,j+1} likewise with xb;  h = 1/(2p)
template <int LI, int LJ>
__device__ __forceinline__ void build_E(double h, double xa, double xb, double (&E)[LI + 1][LJ + 1][LI + LJ + 1])
{
#pragma unroll
    for (int i = 0; i <= LI; ++i)
#pragma unroll
        for (int j = 0; j <= LJ; ++j)
#pragma unroll
            for (int t = 0; t <= LI + LJ; ++t) E[i][j][t] = 0.0;
    E[0][0][0] = 1.0;
#pragma unroll
    for (int i = 0; i < LI; ++i)
#pragma unroll
        for (int t = 0; t <= i + 1; ++t) {
            double v = 0.0;
            if (t > 0) v = h * E[i][0][t - 1];
            if (t <= i) v = fma(xa, E[i][0][t], v);
            if (t + 1 <= i) v = fma((double)(t + 1), E[i][0][t + 1], v);
            E[i + 1][0][t] = v;
        }
#pragma unroll
    for (int i = 0; i <= LI; ++i)
#pragma unroll
        for (int j = 0; j < LJ; ++j)
#pragma unroll
            for (int t = 0; t <= i + j + 1; ++t) {
                double v = 0.0;
                if (t > 0) v = h * E[i][j][t - 1];
                if (t <= i + j) v = fma(xb, E[i][j][t], v);
                if (t + 1 <= i + j) v = fma((double)(t + 1), E[i][j][t + 1], v);
                E[i][j + 1][t] = v;
            }
}

template <int LA, int LB, int LC, int LD, int W>
struct DClass {
    static constexpr int NA = ncart_c(LA), NB = ncart_c(LB), NC = ncart_c(LC), ND = ncart_c(LD);
    static constexpr int NAB = NA * NB, NCD = NC * ND, NI = NAB * NCD;
    static constexpr int L = LA + LB + LC + LD, LAB = LA + LB, LCD = LC + LD;
    static constexpr int NOWN = (NCD + W - 1) / W;        // ket component pairs per warp
    static constexpr int NACC = NOWN * NAB;
};

// one primitive quartet: acc[(cd / W) * NAB + ab] += (ab|cd) for the ket component pairs of this warp
template <int LA, int LB, int LC, int LD, int W>
__device__ __forceinline__ void prim_accum_d(const PrimPair& br, const PrimPair& kt, const double2* __restrict__ tab, int worker,
                                             double (&acc)[DClass<LA, LB, LC, LD, W>::NACC])
{
    using D = DClass<LA, LB, LC, LD, W>;
    double R0[nherm(D::L)];
    hermite_R<D::L>(br.c * kt.c, br.p, kt.p, br.Px - kt.Px, br.Py - kt.Py, br.Pz - kt.Pz, tab, R0);
    double Eb[3][LA + 1][LB + 1][LA + LB + 1], Ek[3][LC + 1][LD + 1][LC + LD + 1];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        build_E<LA, LB>(br.inv2p, br.XA[x], br.XB[x], Eb[x]);
        build_E<LC, LD>(kt.inv2p, kt.XA[x], kt.XB[x], Ek[x]);
    }
#pragma unroll
    for (int cd = 0; cd < D::NCD; ++cd) {
        if (W > 1 && (cd % W) != worker) continue;        // warp-uniform
        const int c = cd % D::NC, d = cd / D::NC;
        const int kx = cpow(LC, c, 0) + cpow(LD, d, 0), ky = cpow(LC, c, 1) + cpow(LD, d, 1), kz = cpow(LC, c, 2) + cpow(LD, d, 2);
        double G[nherm(D::LAB)];
#pragma unroll
        for (int i = 0; i < nherm(D::LAB); ++i) G[i] = 0.0;
#pragma unroll
        for (int t2 = 0; t2 <= kx; ++t2)
#pragma unroll
            for (int u2 = 0; u2 <= ky; ++u2)
#pragma unroll
                for (int v2 = 0; v2 <= kz; ++v2) {
                    double e = Ek[0][cpow(LC, c, 0)][cpow(LD, d, 0)][t2] * Ek[1][cpow(LC, c, 1)][cpow(LD, d, 1)][u2] *
                               Ek[2][cpow(LC, c, 2)][cpow(LD, d, 2)][v2];
                    if ((t2 + u2 + v2) & 1) e = -e;
#pragma unroll
                    for (int t = D::LAB; t >= 0; --t)
#pragma unroll
                        for (int u = D::LAB - t; u >= 0; --u)
#pragma unroll
                            for (int v = D::LAB - t - u; v >= 0; --v)
                                G[hidx(t, u, v)] = fma(e, R0[hidx(t + t2, u + u2, v + v2)], G[hidx(t, u, v)]);
                }
        const double ncd = cnorm(LC, c) * cnorm(LD, d);
#pragma unroll
        for (int ab = 0; ab < D::NAB; ++ab) {
            const int a = ab % D::NA, b = ab / D::NA;
            const int bx = cpow(LA, a, 0) + cpow(LB, b, 0), by = cpow(LA, a, 1) + cpow(LB, b, 1), bz = cpow(LA, a, 2) + cpow(LB, b, 2);
            double s = 0.0;
#pragma unroll
            for (int t = 0; t <= bx; ++t)
#pragma unroll
                for (int u = 0; u <= by; ++u) {
                    const double exy = Eb[0][cpow(LA, a, 0)][cpow(LB, b, 0)][t] * Eb[1][cpow(LA, a, 1)][cpow(LB, b, 1)][u];
#pragma unroll
                    for (int v = 0; v <= bz; ++v)
                        s = fma(exy * Eb[2][cpow(LA, a, 2)][cpow(LB, b, 2)][v], G[hidx(t, u, v)], s);
                }
            acc[(cd / W) * D::NAB + ab] = fma(ncd * cnorm(LA, a) * cnorm(LB, b), s, acc[(cd / W) * D::NAB + ab]);
        }
    }
}

struct DEvalArgs {
    const EvalItem* items;
    KetClass bra, ket;
    const long long* batch_base;
    const double2* boys;
    double* buf;
    double tau, tau_p, w_extra;
    unsigned long long* primcount;
    unsigned long long flops_per_prim;
    int same;
};

template <int LA, int LB, int LC, int LD, int W>
__global__ void __launch_bounds__(32 * W) eval_d_kernel(DEvalArgs g)
{
    using D = DClass<LA, LB, LC, LD, W>;
    __shared__ __align__(16) double s_rows[9 * PRIM_STRIDE];
    __shared__ float s_qp[9];
    const EvalItem it = g.items[blockIdx.x];
    const int lane = threadIdx.x & 31, worker = threadIdx.x >> 5;
    const int q = it.k0 + lane;
    const bool active = q < g.ket.n;
    const int qq = active ? q : g.ket.n - 1;
    const double Qq = active ? __ldg(g.ket.Q + qq) : 0.0;
    const double wcd = __ldg(g.ket.same + qq) ? 0.5 : 1.0;
    const int npb = g.bra.np, npk = g.ket.np;
    unsigned long long nprim_done = 0;

    for (int p = it.p_begin; p < it.p_end; ++p) {
        const double Qp = __ldg(g.bra.Q + p);
        const bool ok = active && (Qp * Qq >= g.tau) && (!g.same || p <= q);
        if (!__any_sync(0xffffffffu, ok)) break;           // block-uniform: all warps hold the same kets
        __syncthreads();                                   // everyone is done with the previous pair's rows
        if (threadIdx.x < npb) {                           // bra rows carry c' and w = 36/p (eri_eval.cuh)
            const double* src = g.bra.prim_aos + ((size_t)p * npb + threadIdx.x) * PRIM_STRIDE;
            double* dst = s_rows + threadIdx.x * PRIM_STRIDE;
#pragma unroll
            for (int f = 0; f < PRIM_STRIDE; ++f) dst[f] = __ldg(src + f);
            const double pp = dst[0];
            dst[4] *= 1.33133536380038971280 * rsqrt(2.0 * pp);
            dst[0] = 36.0 / pp;
            s_qp[threadIdx.x] = __ldg(g.bra.qp_aos + (size_t)p * npb + threadIdx.x);
        }
        __syncthreads();
        const long long batch = g.batch_base[p] + (q >> 5) - (g.same ? (p >> 5) : 0);
        double* dst = g.buf + (size_t)batch * ((size_t)D::NI * 32) + lane;
        double acc[D::NACC];
#pragma unroll
        for (int i = 0; i < D::NACC; ++i) acc[i] = 0.0;
        // primitive-quartet screening as in eval_kernel (jk_eval.cu): prefixes of the bound-sorted primitive lists
        int nkb_l = 0, nkk_l = 0;
        if (ok) {
            for (int kb = 0; kb < npb; ++kb) nkb_l += ((double)s_qp[kb] * Qq >= g.tau_p) ? 1 : 0;
            for (int kk = 0; kk < npk; ++kk) nkk_l += ((double)__ldg(g.ket.qp + (size_t)kk * g.ket.n + qq) * Qp >= g.tau_p) ? 1 : 0;
            nkb_l = max(nkb_l, 1); nkk_l = max(nkk_l, 1);
        }
        const int nkb = __reduce_max_sync(0xffffffffu, nkb_l), nkk = __reduce_max_sync(0xffffffffu, nkk_l);
        if (ok) {
            if (worker == 0) nprim_done += (unsigned)(nkb * nkk);
#pragma unroll 1
            for (int kk = 0; kk < nkk; ++kk) {
                PrimPair k1 = load_prim_soa(g.ket.prim, g.ket.n, kk, qq);
                to_scaled(k1);
                k1.p += g.w_extra;
#pragma unroll 1
                for (int kb = 0; kb < nkb; ++kb) {
                    const double* r = s_rows + kb * PRIM_STRIDE;
                    PrimPair bp;
                    bp.p = r[0]; bp.Px = r[1]; bp.Py = r[2]; bp.Pz = r[3]; bp.c = r[4]; bp.inv2p = r[5];
                    bp.XA[0] = r[6]; bp.XA[1] = r[7]; bp.XA[2] = r[8]; bp.XB[0] = r[9]; bp.XB[1] = r[10]; bp.XB[2] = r[11];
                    prim_accum_d<LA, LB, LC, LD, W>(bp, k1, g.boys, worker, acc);
                }
            }
        }
        const double w = (g.same && p == q) ? 0.5 * wcd : wcd;
#pragma unroll
        for (int cd = 0; cd < D::NCD; ++cd) {
            if (W > 1 && (cd % W) != worker) continue;
#pragma unroll
            for (int ab = 0; ab < D::NAB; ++ab)
                __stcs(dst + (size_t)(cd * D::NAB + ab) * 32, ok ? w * acc[(cd / W) * D::NAB + ab] : 0.0);
        }
    }
    for (int o = 16; o > 0; o >>= 1) nprim_done += __shfl_xor_sync(0xffffffffu, nprim_done, o);
    if (lane == 0 && nprim_done) {                         // slots 5, 6: all classes with a d shell
        atomicAdd(g.primcount + 5, nprim_done);
        atomicAdd(g.primcount + 6, nprim_done * g.flops_per_prim);
    }
}

template <int LA, int LB, int LC, int LD, int W>
int launch_eval_d(Handle* h, const Segment& sg, double* buf, cudaStream_t st)
{
    DEvalArgs g;
    g.items = sg.items;
    g.bra = h->tabs.kets[sg.kc_bra];
    g.ket = h->tabs.kets[sg.kc_ket];
    g.batch_base = sg.batch_base;
    g.boys = h->tabs.boys[LA + LB + LC + LD];
    g.buf = buf;
    g.tau = h->tabs.tau;
    g.tau_p = prim_threshold(h->tabs.tau);
    g.w_extra = h->pass_w_extra;
    g.primcount = h->d_primcount;
    g.flops_per_prim = (unsigned long long)flops_prim(LA, LB, LC, LD);
    g.same = (sg.kc_bra == sg.kc_ket);
    eval_d_kernel<LA, LB, LC, LD, W><<<dim3(sg.nitems), dim3(32 * W), 0, st>>>(g);
    h->kernel_launches++;
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

}  // namespace

// W (last template argument) = warps per block sharing the ket component pairs of a quartet; the values are the
// fastest of {1, 2, 3, 6} measured per class at 1884 basis functions (more workers: fewer accumulators per thread, but
// every worker rebuilds the Hermite tables of the primitive quartet).
// Classes with an unrolled kernel; *handled = false leaves the segment to eval_generic_kernel.
int eval_segment_d(Handle* h, const Segment& sg, double* buf, cudaStream_t st, bool* handled)
{
    *handled = true;
    const int key = ((sg.la * 3 + sg.lb) * 3 + sg.lc) * 3 + sg.ld;
    switch (key) {
        case ((2 * 3 + 0) * 3 + 0) * 3 + 0: return launch_eval_d<2, 0, 0, 0, 1>(h, sg, buf, st);
        case ((2 * 3 + 0) * 3 + 1) * 3 + 0: return launch_eval_d<2, 0, 1, 0, 1>(h, sg, buf, st);
        case ((2 * 3 + 1) * 3 + 0) * 3 + 0: return launch_eval_d<2, 1, 0, 0, 1>(h, sg, buf, st);
        case ((2 * 3 + 0) * 3 + 1) * 3 + 1: return launch_eval_d<2, 0, 1, 1, 1>(h, sg, buf, st);
        case ((2 * 3 + 0) * 3 + 2) * 3 + 0: return launch_eval_d<2, 0, 2, 0, 1>(h, sg, buf, st);
        case ((2 * 3 + 1) * 3 + 1) * 3 + 0: return launch_eval_d<2, 1, 1, 0, 1>(h, sg, buf, st);
        case ((2 * 3 + 2) * 3 + 0) * 3 + 0: return launch_eval_d<2, 2, 0, 0, 1>(h, sg, buf, st);
        case ((2 * 3 + 1) * 3 + 1) * 3 + 1: return launch_eval_d<2, 1, 1, 1, 1>(h, sg, buf, st);
        case ((2 * 3 + 1) * 3 + 2) * 3 + 0: return launch_eval_d<2, 1, 2, 0, 2>(h, sg, buf, st);
        case ((2 * 3 + 2) * 3 + 1) * 3 + 0: return launch_eval_d<2, 2, 1, 0, 3>(h, sg, buf, st);
        case ((2 * 3 + 1) * 3 + 2) * 3 + 1: return launch_eval_d<2, 1, 2, 1, 3>(h, sg, buf, st);
        case ((2 * 3 + 2) * 3 + 1) * 3 + 1: return launch_eval_d<2, 2, 1, 1, 2>(h, sg, buf, st);
        case ((2 * 3 + 2) * 3 + 2) * 3 + 0: return launch_eval_d<2, 2, 2, 0, 2>(h, sg, buf, st);
        case ((2 * 3 + 2) * 3 + 2) * 3 + 1: return launch_eval_d<2, 2, 2, 1, 2>(h, sg, buf, st);
        default: *handled = false; return RTTDA_OK;
    }
}

}  // namespace rttda
