// ERI evaluation (DESIGN.md step a3; eq. 4, "directly on the GPU" P:130): every unique, Schwarz-screened
// contracted shell quartet of a segment is evaluated exactly ONCE per ERI pass and its 1..81 Cartesian
// components are written to the HBM staging buffer, from which the digestion kernels (jk_digest.cu) serve all
// densities of the batch.  Nothing persists across passes: the buffer is rewritten by every pass.
//
// Work decomposition:
//   block  = JK_BLOCK consecutive kets of the (Schwarz-sorted) ket list x a run of bra pairs of the bra list
//   thread = one ket pair; its primitive data stay in registers (SoA loads, coalesced) while the block walks
//            the bra pairs, whose primitive rows are staged in shared memory and read as broadcasts
//   Boys   = Taylor coefficients from a shared-memory table row for the near-field primitive quartets, a closed form
//            for the far-field majority (eri_eval.cuh)
// The inner loops are pure FP64 ALU work: no accumulators of the J/K digestion live here.
#include "eri_eval.cuh"

namespace rttda {

struct EvalArgs {
    const EvalItem* items;
    KetClass bra, ket;
    const long long* batch_base;
    const double2* boys;
    double* buf;
    double tau;
    double tau_p;          // primitive-quartet threshold (prim_threshold(tau)): (kb, kk) is evaluated iff q_kb Q_ket >= tau_p and q_kk Q_bra >= tau_p
    unsigned long long* primcount;   // primitive quartets evaluated (lane level), one counter per total angular momentum
    double w_extra;        // 0 for 1/r12; 36 / omega^2 for erf(omega r12)/r12 (alpha -> alpha omega^2 / (alpha + omega^2))
    int same;
};

template <int LC, int LD>
__device__ __forceinline__ PrimPair load_ket_prim(const double* __restrict__ prim, int n, int k, int q)
{
    const double* b = prim + (size_t)k * PRIM_STRIDE * n + q;
    const size_t N = (size_t)n;
    PrimPair r;
    r.p = __ldg(b); r.Px = __ldg(b + N); r.Py = __ldg(b + 2 * N); r.Pz = __ldg(b + 3 * N);
    r.c = __ldg(b + 4 * N);
    if (LC + LD > 0) {
        r.inv2p = __ldg(b + 5 * N);
        r.XA[0] = __ldg(b + 6 * N); r.XA[1] = __ldg(b + 7 * N); r.XA[2] = __ldg(b + 8 * N);
    } else {
        r.inv2p = 0.0; r.XA[0] = r.XA[1] = r.XA[2] = 0.0;
    }
    if (LD > 0) {
        r.XB[0] = __ldg(b + 9 * N); r.XB[1] = __ldg(b + 10 * N); r.XB[2] = __ldg(b + 11 * N);
    } else {
        r.XB[0] = r.XB[1] = r.XB[2] = 0.0;
    }
    to_scaled(r);
    return r;
}

__device__ __forceinline__ PrimPair load_bra_prim_smem(const double* row)
{
    PrimPair r;
    const double2* r2 = reinterpret_cast<const double2*>(row);
    const double2 a = r2[0], b = r2[1], c = r2[2], d = r2[3], e = r2[4], f = r2[5];
    r.p = a.x; r.Px = a.y; r.Py = b.x; r.Pz = b.y; r.c = c.x; r.inv2p = c.y; r.two_p = 0.0;   // two_p: kets only
    r.XA[0] = d.x; r.XA[1] = d.y; r.XA[2] = e.x; r.XB[0] = e.y; r.XB[1] = f.x; r.XB[2] = f.y;
    return r;
}

template <int LA, int LB, int LC, int LD, int KP>
__global__ void __launch_bounds__(JK_BLOCK) eval_kernel(EvalArgs g)
{
    constexpr int NI = (2 * LA + 1) * (2 * LB + 1) * (2 * LC + 1) * (2 * LD + 1);
    constexpr int L = LA + LB + LC + LD;
    // ket primitives live in registers when they are few doubles; otherwise they are re-read (L1 hits)
    constexpr bool KET_IN_REGS = (KP == 1) || (L <= 3 && (KP <= 3 || (LC + LD == 0 && L <= 1)));
    __shared__ __align__(16) double2 s_boys[BOYS_NROW * (BOYS_ROW / 2)];
    __shared__ __align__(16) double s_rows[EVAL_MAX_ROWS * PRIM_STRIDE];
    __shared__ double s_Q[JK_BLOCK];
    __shared__ long long s_base[JK_BLOCK];
    __shared__ float s_qp[EVAL_MAX_ROWS];

    const EvalItem it = g.items[blockIdx.x];
    const int npb = g.bra.np, npairs = it.p_end - it.p_begin;
    for (int i = threadIdx.x; i < BOYS_NROW * (BOYS_ROW / 2); i += JK_BLOCK) s_boys[i] = g.boys[i];
    {
        const double2* src = reinterpret_cast<const double2*>(g.bra.prim_aos + (size_t)it.p_begin * npb * PRIM_STRIDE);
        double2* dst = reinterpret_cast<double2*>(s_rows);
        const int n2 = npairs * npb * (PRIM_STRIDE / 2);
        for (int i = threadIdx.x; i < n2; i += JK_BLOCK) dst[i] = src[i];
        for (int i = threadIdx.x; i < npairs * npb; i += JK_BLOCK) s_qp[i] = g.bra.qp_aos[(size_t)it.p_begin * npb + i];
        __syncthreads();
        for (int r = threadIdx.x; r < npairs * npb; r += JK_BLOCK) {     // rows carry c' and w = 36/p (eri_eval.cuh)
            const double p = s_rows[r * PRIM_STRIDE];
            s_rows[r * PRIM_STRIDE + 4] *= 1.33133536380038971280 * rsqrt(2.0 * p);
            s_rows[r * PRIM_STRIDE] = 36.0 / p;
        }
        if (threadIdx.x < npairs) {
            s_Q[threadIdx.x] = g.bra.Q[it.p_begin + threadIdx.x];
            s_base[threadIdx.x] = g.batch_base[it.p_begin + threadIdx.x];
        }
    }
    __syncthreads();

    const int q = it.k0 + threadIdx.x;
    const bool active = q < g.ket.n;
    const int qq = active ? q : g.ket.n - 1;
    const double Qq = active ? __ldg(g.ket.Q + qq) : 0.0;
    const double wcd = __ldg(g.ket.same + qq) ? 0.5 : 1.0;
    const int lane = threadIdx.x & 31;

    float kq[KP];                                           // bounds of this ket's primitive pairs, descending
#pragma unroll
    for (int k = 0; k < KP; ++k) kq[k] = __ldg(g.ket.qp + (size_t)k * g.ket.n + qq);
    unsigned long long nprim_done = 0;
    PrimPair kp[KET_IN_REGS ? KP : 1];
    if (KET_IN_REGS) {
#pragma unroll
        for (int k = 0; k < KP; ++k) { kp[k] = load_ket_prim<LC, LD>(g.ket.prim, g.ket.n, k, qq); kp[k].p += g.w_extra; }
    }

    for (int ip = 0; ip < npairs; ++ip) {
        const int p = it.p_begin + ip;
        const bool ok = active && (s_Q[ip] * Qq >= g.tau) && (!g.same || p <= q);
        if (!__any_sync(0xffffffffu, ok)) break;          // both conditions only get worse along the bra list
        // A batch (bra pair, 32 kets = this warp) that exists in the staging map is written in full: lanes whose
        // quartet is screened out, lies below the diagonal of a same-class segment or beyond the ket list store
        // zeros, and the degeneracy weights of the 8-fold symmetry that depend on the quartet alone (1/2 if bra
        // pair == ket pair, 1/2 if the ket pair is diagonal) are folded into the stored values, so the digestion
        // kernels need no per-lane tests.
        double I[NI];
#pragma unroll
        for (int i = 0; i < NI; ++i) I[i] = 0.0;
        const double* rows = s_rows + (size_t)ip * npb * PRIM_STRIDE;
        // Primitive-quartet screening (both lists are sorted by descending bound, so the primitives a quartet needs are
        // prefixes): bra primitive kb matters to this lane iff q_kb Q_ket >= tau_p, ket primitive kk iff q_kk Q_bra >=
        // tau_p.  The warp runs the longest prefix any of its lanes needs; kets of a warp are neighbours in the
        // Schwarz-sorted list, so the prefixes are nearly uniform.
        const float* qb = s_qp + ip * npb;
        int nkb_l = 0, nkk_l = 0;
        if (ok) {
            for (int kb = 0; kb < npb; ++kb) nkb_l += ((double)qb[kb] * Qq >= g.tau_p) ? 1 : 0;
#pragma unroll
            for (int kk = 0; kk < KP; ++kk) nkk_l += ((double)kq[kk] * s_Q[ip] >= g.tau_p) ? 1 : 0;
            nkb_l = max(nkb_l, 1); nkk_l = max(nkk_l, 1);
        }
        const int nkb = __reduce_max_sync(0xffffffffu, nkb_l), nkk = __reduce_max_sync(0xffffffffu, nkk_l);
        if (ok) nprim_done += (unsigned)(nkb * nkk);
        if (!ok) {
        } else if (KET_IN_REGS) {
#pragma unroll 1
            for (int kb = 0; kb < nkb; ++kb) {
                const PrimPair bp = load_bra_prim_smem(rows + kb * PRIM_STRIDE);
#pragma unroll
                for (int kk = 0; kk < KP; ++kk)
                    if (kk < nkk) eri_prim_accum<LA, LB, LC, LD>(bp, kp[kk], s_boys, I);
            }
        } else {
            // ket primitive outermost: it is loaded once (coalesced, L1) and meets every bra primitive (shared memory)
#pragma unroll 1
            for (int kk = 0; kk < nkk; ++kk) {
                PrimPair k1 = load_ket_prim<LC, LD>(g.ket.prim, g.ket.n, kk, qq);
                k1.p += g.w_extra;
#pragma unroll 1
                for (int kb = 0; kb < nkb; ++kb) {
                    const PrimPair bp = load_bra_prim_smem(rows + kb * PRIM_STRIDE);
                    eri_prim_accum<LA, LB, LC, LD>(bp, k1, s_boys, I);
                }
            }
        }
        const long long batch = s_base[ip] + (q >> 5) - (g.same ? (p >> 5) : 0);
        double* dst = g.buf + (size_t)batch * (NI * 32) + lane;
        const double w = (g.same && p == q) ? 0.5 * wcd : wcd;
#pragma unroll
        for (int i = 0; i < NI; ++i) __stcs(dst + i * 32, w * I[i]);
    }
    // primitive quartets evaluated by this block (feeds the flop model of the roofline figure)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nprim_done += __shfl_xor_sync(0xffffffffu, nprim_done, o);
    if (lane == 0 && nprim_done) atomicAdd(g.primcount + L, nprim_done);
}

template <int LA, int LB, int LC, int LD>
static int launch_eval(Handle* h, const Segment& sg, double* buf, cudaStream_t st)
{
    EvalArgs g;
    g.items = sg.items;
    g.bra = h->tabs.kets[sg.kc_bra];
    g.ket = h->tabs.kets[sg.kc_ket];
    g.batch_base = sg.batch_base;
    g.boys = h->tabs.boys[LA + LB + LC + LD];
    g.buf = buf;
    g.tau = h->tabs.tau;
    g.tau_p = prim_threshold(h->tabs.tau);
    g.primcount = h->d_primcount;
    g.w_extra = h->pass_w_extra;
    g.same = (sg.kc_bra == sg.kc_ket);
    dim3 grid(sg.nitems), block(JK_BLOCK);
    switch (g.ket.np) {
        case 1: eval_kernel<LA, LB, LC, LD, 1><<<grid, block, 0, st>>>(g); break;
        case 3: eval_kernel<LA, LB, LC, LD, 3><<<grid, block, 0, st>>>(g); break;
        case 6: eval_kernel<LA, LB, LC, LD, 6><<<grid, block, 0, st>>>(g); break;
        default: eval_kernel<LA, LB, LC, LD, 9><<<grid, block, 0, st>>>(g); break;
    }
    h->kernel_launches++;
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

int eval_segment(Handle* h, const Segment& sg, double* buf, cudaStream_t st)
{
    if (sg.nitems == 0) return RTTDA_OK;
    if (segment_is_general(sg)) return eval_segment_general(h, sg, buf, st);
    const int key = sg.la * 8 + sg.lb * 4 + sg.lc * 2 + sg.ld;
    switch (key) {
        case 0:  return launch_eval<0, 0, 0, 0>(h, sg, buf, st);
        case 8:  return launch_eval<1, 0, 0, 0>(h, sg, buf, st);
        case 10: return launch_eval<1, 0, 1, 0>(h, sg, buf, st);
        case 12: return launch_eval<1, 1, 0, 0>(h, sg, buf, st);
        case 14: return launch_eval<1, 1, 1, 0>(h, sg, buf, st);
        case 15: return launch_eval<1, 1, 1, 1>(h, sg, buf, st);
        default: set_error("eval_segment: unsupported class"); return RTTDA_EINVAL;
    }
}

// ---------------------------------------------------------------------------------------------------
// Schwarz bounds Q_ab = sqrt(max_comp (ab|ab)) for all candidate pairs of one pair type (R14).
template <int LA, int LB>
__global__ void schwarz_kernel(int npairs, const int* __restrict__ np, const int* __restrict__ off,
                               const double* __restrict__ prim, const double2* __restrict__ boys_tab,
                               double* __restrict__ Q)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npairs) return;
    constexpr int NA = 2 * LA + 1, NB = 2 * LB + 1;
    double I[NA * NB * NA * NB];
#pragma unroll
    for (int k = 0; k < NA * NB * NA * NB; ++k) I[k] = 0.0;
    const int n = np[i], o = off[i];
    for (int k1 = 0; k1 < n; ++k1) {
        PrimPair b = load_prim_aos(prim + (size_t)(o + k1) * PRIM_STRIDE);
        to_scaled(b);
        for (int k2 = 0; k2 < n; ++k2) {
            PrimPair k = load_prim_aos(prim + (size_t)(o + k2) * PRIM_STRIDE);
            to_scaled(k);
            eri_prim_accum<LA, LB, LA, LB>(b, k, boys_tab, I);
        }
    }
    double m = 0.0;
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b) m = fmax(m, I[eri_index<LA, LB, LA, LB>(a, b, a, b)]);
    Q[i] = sqrt(m);
}

int schwarz_device(int pairclass, int npairs, const int* d_np, const int* d_off, const double* d_prim,
                   const double2* d_boys, double* d_Q, cudaStream_t st)
{
    if (npairs == 0) return RTTDA_OK;
    dim3 block(128), grid((npairs + 127) / 128);
    if (pairclass == 0) schwarz_kernel<0, 0><<<grid, block, 0, st>>>(npairs, d_np, d_off, d_prim, d_boys, d_Q);
    else if (pairclass == 1) schwarz_kernel<1, 0><<<grid, block, 0, st>>>(npairs, d_np, d_off, d_prim, d_boys, d_Q);
    else schwarz_kernel<1, 1><<<grid, block, 0, st>>>(npairs, d_np, d_off, d_prim, d_boys, d_Q);
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

}  // namespace rttda
