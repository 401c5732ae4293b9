// AO-direct J/K build (DESIGN.md steps a3-a4; "Coulomb and Exchange terms ... directly on the GPU").
//
// Work decomposition ("shell a fixed per block, ket pair owned by a thread"):
//   block  = one a-list (all ordered bra pairs (a,b) for one shell a, one l_b, one contraction sub-class,
//            sorted by Schwarz bound) x JK_BLOCK consecutive kets of one ket class
//   thread = one unordered ket pair {c,d}; it walks the a-list while Q_ab Q_cd >= tau, evaluates the
//            contracted block (ab|cd) and digests it at once for NV densities:
//              K_ac += I T_bd, K_ad += I T_bc, K_ca += I T_db, K_da += I T_cb      (registers, whole b loop)
//              J_cd += I (T_ab + T_ba)                                             (registers, canonical bras)
//              J_ab += I (T_cd + T_dc)                                             (warp shuffle reduce)
//   Unique-quartet bookkeeping: bra pair >= ket pair in the (class, position) order; both orientations
//   (a,b), (b,a) of a bra pair are separate records, which is what lets all exchange updates stay in
//   registers (each quartet is evaluated twice; see DESIGN.md for the trade against global atomics).
// Densities and results use the interleaved layout Tq[mu][nu][v] (v fastest), F likewise.
#include "eri_eval.cuh"

namespace rttda {

template <int NV>
__device__ __forceinline__ void red_add(double* p, const double (&v)[NV], double s)
{
#pragma unroll
    for (int i = 0; i < NV; ++i) atomicAdd(p + i, s * v[i]);
}

__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

template <int LA, int LB, int LC, int LD, int KP, int NV>
__global__ void __launch_bounds__(JK_BLOCK)
jk_kernel(JKTables tb, const WorkItem* __restrict__ work, int ketclass, int nvt, int v0,
          const double* __restrict__ Tq, double* __restrict__ Fq, double cx)
{
    constexpr int NA = 2 * LA + 1, NB = 2 * LB + 1, NC = 2 * LC + 1, ND = 2 * LD + 1;
    constexpr int NI = NA * NB * NC * ND;
    const WorkItem wi = work[blockIdx.x];
    const AList al = tb.alists[wi.alist];
    const KetClass kc = tb.kets[ketclass];
    const int q = wi.ket0 + threadIdx.x;
    const bool active = q < kc.n;
    const int qq = active ? q : kc.n - 1;
    const double Qq = active ? __ldg(kc.Q + qq) : 0.0;
    const int aoC = __ldg(kc.ao_c + qq), aoD = __ldg(kc.ao_d + qq);
    const bool cd_same = __ldg(kc.same + qq) != 0;
    const bool same_class = (al.ketclass == ketclass);
    const int aoA = al.ao_a;
    const size_t nao = tb.nao;
    const double* Tv = Tq + v0;
    const size_t rs = nao * nvt;          // row stride of Tq / Fq
#define TQ(mu, nu) (Tv + (size_t)(mu) * rs + (size_t)(nu) * nvt)

    PrimPair kp1;
    if (KP == 1) kp1 = load_prim_soa(kc.prim, kc.n, 0, qq);

    // S_cd = T_cd + T_dc for the J_ab update
    double Scd[NC][ND][NV];
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
        for (int d = 0; d < ND; ++d)
#pragma unroll
            for (int v = 0; v < NV; ++v)
                Scd[c][d][v] = __ldg(TQ(aoC + c, aoD + d) + v) + __ldg(TQ(aoD + d, aoC + c) + v);

    double Kac[NA][NC][NV], Kad[NA][ND][NV], Kca[NC][NA][NV], Kda[ND][NA][NV], Jcd[NC][ND][NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
#pragma unroll
        for (int a = 0; a < NA; ++a) {
#pragma unroll
            for (int c = 0; c < NC; ++c) Kac[a][c][v] = Kca[c][a][v] = 0.0;
#pragma unroll
            for (int d = 0; d < ND; ++d) Kad[a][d][v] = Kda[d][a][v] = 0.0;
        }
#pragma unroll
        for (int c = 0; c < NC; ++c)
#pragma unroll
            for (int d = 0; d < ND; ++d) Jcd[c][d][v] = 0.0;
    }

    const int lane = threadIdx.x & 31;
    for (int r = al.rec_begin; r < al.rec_end; ++r) {
        const BraRec br = tb.recs[r];
        const bool ok = active && (br.Q * Qq >= tb.tau) && (!same_class || br.pos <= q);
        if (!__any_sync(0xffffffffu, ok)) break;
        const bool canonical = (br.flags & 1) != 0;
        const int aoB = br.ao_b;
        double I[NI];
#pragma unroll
        for (int i = 0; i < NI; ++i) I[i] = 0.0;
        if (ok) {
            for (int kb = 0; kb < al.np; ++kb) {
                const PrimPair bp = load_prim_aos(tb.bra_prim + (size_t)(br.prim_off + kb) * PRIM_STRIDE);
                if (KP == 1) {
                    eri_prim_accum<LA, LB, LC, LD>(bp, kp1, tb.boys, I);
                } else {
#pragma unroll 1
                    for (int kk = 0; kk < KP; ++kk) {
                        const PrimPair kp = load_prim_soa(kc.prim, kc.n, kk, qq);
                        eri_prim_accum<LA, LB, LC, LD>(bp, kp, tb.boys, I);
                    }
                }
            }
            // degeneracy weights: 1/2 if the ket is a diagonal pair, 1/2 if bra pair == ket pair
            const double wsame = (same_class && br.pos == q) ? 0.5 : 1.0;
            const double wk = wsame * (cd_same ? 0.5 : 1.0);
#pragma unroll
            for (int i = 0; i < NI; ++i) I[i] *= wk;
            // ---- exchange: four register-resident updates
#pragma unroll
            for (int b = 0; b < NB; ++b) {
#pragma unroll
                for (int d = 0; d < ND; ++d) {
                    double tbd[NV], tdb[NV];
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        tbd[v] = __ldg(TQ(aoB + b, aoD + d) + v);
                        tdb[v] = __ldg(TQ(aoD + d, aoB + b) + v);
                    }
#pragma unroll
                    for (int a = 0; a < NA; ++a)
#pragma unroll
                        for (int c = 0; c < NC; ++c) {
                            const double x = I[eri_index<LA, LB, LC, LD>(a, b, c, d)];
#pragma unroll
                            for (int v = 0; v < NV; ++v) {
                                Kac[a][c][v] = fma(x, tbd[v], Kac[a][c][v]);
                                Kca[c][a][v] = fma(x, tdb[v], Kca[c][a][v]);
                            }
                        }
                }
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    double tbc[NV], tcb[NV];
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        tbc[v] = __ldg(TQ(aoB + b, aoC + c) + v);
                        tcb[v] = __ldg(TQ(aoC + c, aoB + b) + v);
                    }
#pragma unroll
                    for (int a = 0; a < NA; ++a)
#pragma unroll
                        for (int d = 0; d < ND; ++d) {
                            const double x = I[eri_index<LA, LB, LC, LD>(a, b, c, d)];
#pragma unroll
                            for (int v = 0; v < NV; ++v) {
                                Kad[a][d][v] = fma(x, tbc[v], Kad[a][d][v]);
                                Kda[d][a][v] = fma(x, tcb[v], Kda[d][a][v]);
                            }
                        }
                }
            }
        }
        // ---- Coulomb (only the canonical orientation of the bra pair does it; uniform branch)
        if (canonical) {
            const bool ab_same = (br.flags & 2) != 0;
            // I currently carries wk = wsame * w_cd; J_cd needs wsame * w_ab instead
            const double fix = (cd_same ? 2.0 : 1.0) * (ab_same ? 0.5 : 1.0);
#pragma unroll
            for (int a = 0; a < NA; ++a)
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    double sab[NV], jab[NV];
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        sab[v] = fix * (__ldg(TQ(aoA + a, aoB + b) + v) + __ldg(TQ(aoB + b, aoA + a) + v));
                        jab[v] = 0.0;
                    }
#pragma unroll
                    for (int c = 0; c < NC; ++c)
#pragma unroll
                        for (int d = 0; d < ND; ++d) {
                            const double x = I[eri_index<LA, LB, LC, LD>(a, b, c, d)];
#pragma unroll
                            for (int v = 0; v < NV; ++v) {
                                Jcd[c][d][v] = fma(x, sab[v], Jcd[c][d][v]);
                                jab[v] = fma(x, Scd[c][d][v], jab[v]);
                            }
                        }
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        const double tot = warp_sum(jab[v]);
                        if (lane == 0 && tot != 0.0) {
                            atomicAdd(Fq + v0 + (size_t)(aoA + a) * rs + (size_t)(aoB + b) * nvt + v, 2.0 * tot);
                            if (!ab_same)
                                atomicAdd(Fq + v0 + (size_t)(aoB + b) * rs + (size_t)(aoA + a) * nvt + v, 2.0 * tot);
                        }
                    }
                }
        }
    }
#undef TQ
    if (!active) return;
    // ---- flush the register accumulators: F += 2 J - cx K
    double* Fv = Fq + v0;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            red_add<NV>(Fv + (size_t)(aoA + a) * rs + (size_t)(aoC + c) * nvt, Kac[a][c], -cx);
            red_add<NV>(Fv + (size_t)(aoC + c) * rs + (size_t)(aoA + a) * nvt, Kca[c][a], -cx);
        }
#pragma unroll
        for (int d = 0; d < ND; ++d) {
            red_add<NV>(Fv + (size_t)(aoA + a) * rs + (size_t)(aoD + d) * nvt, Kad[a][d], -cx);
            red_add<NV>(Fv + (size_t)(aoD + d) * rs + (size_t)(aoA + a) * nvt, Kda[d][a], -cx);
        }
    }
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
        for (int d = 0; d < ND; ++d) {
            red_add<NV>(Fv + (size_t)(aoC + c) * rs + (size_t)(aoD + d) * nvt, Jcd[c][d], 2.0);
            if (!cd_same) red_add<NV>(Fv + (size_t)(aoD + d) * rs + (size_t)(aoC + c) * nvt, Jcd[c][d], 2.0);
        }
}

// ---------------------------------------------------------------------------------------------------
constexpr int NV_CHUNK = 2;
int jk_nvec_chunk() { return NV_CHUNK; }

template <int LA, int LB, int LC, int LD, int NV>
static int launch_kp(Handle* h, const JKLaunch& L, int nvt, int v0, const double* Tq, double* Fq,
                     cudaStream_t st)
{
    const int np = h->tabs.kets[L.ketclass].np;
    dim3 grid(L.nwork), block(JK_BLOCK);
    if (np == 1)
        jk_kernel<LA, LB, LC, LD, 1, NV><<<grid, block, 0, st>>>(h->tabs, L.work, L.ketclass, nvt, v0, Tq, Fq, h->cx);
    else if (np == 3)
        jk_kernel<LA, LB, LC, LD, 3, NV><<<grid, block, 0, st>>>(h->tabs, L.work, L.ketclass, nvt, v0, Tq, Fq, h->cx);
    else
        jk_kernel<LA, LB, LC, LD, 9, NV><<<grid, block, 0, st>>>(h->tabs, L.work, L.ketclass, nvt, v0, Tq, Fq, h->cx);
    h->kernel_launches++;
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

template <int NV>
static int launch_all(Handle* h, int nvt, int v0, const double* Tq, double* Fq, cudaStream_t st)
{
    for (const JKLaunch& L : h->launches) {
        if (L.nwork == 0) continue;
        const int key = L.la * 8 + L.lb * 4 + L.lc * 2 + L.ld;
        switch (key) {
            case 0:  RT_TRY((launch_kp<0, 0, 0, 0, NV>(h, L, nvt, v0, Tq, Fq, st))); break;
            case 8:  RT_TRY((launch_kp<1, 0, 0, 0, NV>(h, L, nvt, v0, Tq, Fq, st))); break;
            case 4:  RT_TRY((launch_kp<0, 1, 0, 0, NV>(h, L, nvt, v0, Tq, Fq, st))); break;
            case 10: RT_TRY((launch_kp<1, 0, 1, 0, NV>(h, L, nvt, v0, Tq, Fq, st))); break;
            case 6:  RT_TRY((launch_kp<0, 1, 1, 0, NV>(h, L, nvt, v0, Tq, Fq, st))); break;
            case 12: RT_TRY((launch_kp<1, 1, 0, 0, NV>(h, L, nvt, v0, Tq, Fq, st))); break;
            case 14: RT_TRY((launch_kp<1, 1, 1, 0, NV>(h, L, nvt, v0, Tq, Fq, st))); break;
            case 15: RT_TRY((launch_kp<1, 1, 1, 1, NV>(h, L, nvt, v0, Tq, Fq, st))); break;
            default: set_error("jk: unsupported class"); return RTTDA_EINVAL;
        }
    }
    return RTTDA_OK;
}

// Fq must be zeroed by the caller.  Processes densities [v0, v0+nv) of the interleaved arrays.
int jk_build(Handle* h, int nvec_total, int v0, int nv, const double* Tq, double* Fq, cudaStream_t st)
{
    if (nv == 2) return launch_all<2>(h, nvec_total, v0, Tq, Fq, st);
    if (nv == 1) return launch_all<1>(h, nvec_total, v0, Tq, Fq, st);
    set_error("jk_build: bad chunk");
    return RTTDA_EINVAL;
}

// ---------------------------------------------------------------------------------------------------
// Schwarz bounds Q_ab = sqrt(max_comp (ab|ab)) for all candidate pairs of one pair class (R14).
template <int LA, int LB>
__global__ void schwarz_kernel(int npairs, const int* __restrict__ np, const int* __restrict__ off,
                               const double* __restrict__ prim, const double* __restrict__ boys_tab,
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
        const PrimPair b = load_prim_aos(prim + (size_t)(o + k1) * PRIM_STRIDE);
        for (int k2 = 0; k2 < n; ++k2) {
            const PrimPair k = load_prim_aos(prim + (size_t)(o + k2) * PRIM_STRIDE);
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
                   const double* d_boys, double* d_Q, cudaStream_t st)
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
