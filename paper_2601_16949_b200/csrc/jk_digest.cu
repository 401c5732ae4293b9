// J/K digestion (DESIGN.md step a4; "Coulomb and Exchange terms" P:130): F += 2 J[T] - cx K[T] from the
// contracted integrals the evaluation kernels staged in HBM (jk_eval.cu), for NV densities per launch.
//
// Work decomposition ("shell a fixed per block, ket pair owned by a thread or lane group"):
//   block  = one a-list (all ordered bra pairs (a,b) for one shell a, one l_b, one contraction sub-class, sorted by
//            Schwarz bound) x consecutive kets of one ket class; it walks the a-list while Q_ab Q_cd >= tau and
//            streams the stored blocks (ab|cd) through TMA bulk-copy rings in shared memory:
//              K_ac += I T_bd, K_ad += I T_bc, K_ca += I T_db, K_da += I T_cb      (registers, whole b loop)
//              J_cd += I (T_ab + T_ba)                                             (registers, canonical bras)
//              J_ab += I (T_cd + T_dc)                                             (warp butterfly reduce)
//   Both orientations (a,b), (b,a) of a bra pair are separate records reading the SAME stored block, which
//   keeps every exchange update in registers: no per-quartet global atomics, and no second evaluation.
// Densities and results use the interleaved layout Tq[mu][nu][v] (v fastest), F likewise.
// Two kernels: digest_j_kernel (thread = ket, NV densities in registers, 128 kets per block) does the Coulomb part
// over the canonical records without any per-lane density gather; digest_b_kernel (block = one 32-ket batch, a
// group of lanes per ket, lane = density) does the exchange part, gathering {T + T^T, T - T^T} pairs
// (symsplit_kernel) so that one 16-byte load yields both T_mn and T_nm.  DESIGN.md section 5 has the rooflines,
// profiles/ the ncu evidence.
#include "common.cuh"
#include "tma.cuh"

namespace rttda {

template <int NV>
__device__ __forceinline__ void red_add(double* p, const double (&v)[NV], double s)
{
#pragma unroll
    for (int i = 0; i < NV; ++i) atomicAdd(p + i, s * v[i]);
}

// Sum N (power of two <= 32) per-lane values over the warp with a transposing butterfly: at each of the first
// log2(N) steps a lane keeps one half of its values and hands the other half to its partner, so N values cost
// N - 1 + (5 - log2 N) shuffles instead of 5 N.  On return v[0] of lane l is the warp total of value index
// warp_reduce_owner_index<N>(l); lanes that differ only in their low (5 - log2 N) bits hold the same total.
template <int N, int W, int OFF>
__device__ __forceinline__ void warp_reduce_step(double (&v)[N], int lane)
{
    if constexpr (OFF >= 1) {
        if constexpr (W > 1) {
            constexpr int half = W / 2;
            const bool upper = (lane & OFF) != 0;
#pragma unroll
            for (int j = 0; j < half; ++j) {
                const double send = upper ? v[j] : v[j + half];
                const double keep = upper ? v[j + half] : v[j];
                v[j] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
            }
            warp_reduce_step<N, half, OFF / 2>(v, lane);
        } else {
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], OFF);
            warp_reduce_step<N, 1, OFF / 2>(v, lane);
        }
    }
}
template <int N>
__device__ __forceinline__ double warp_reduce_multi(double (&v)[N], int lane)
{
    static_assert(N == 1 || N == 2 || N == 4 || N == 8 || N == 16 || N == 32, "N must be a power of two");
    warp_reduce_step<N, N, 16>(v, lane);
    return v[0];
}
template <int N>
__device__ __forceinline__ int warp_reduce_owner_index(int lane)
{
    int idx = 0;
    if (N >= 2 && (lane & 16)) idx += N / 2;
    if (N >= 4 && (lane & 8)) idx += N / 4;
    if (N >= 8 && (lane & 4)) idx += N / 8;
    if (N >= 16 && (lane & 2)) idx += N / 16;
    if (N >= 32 && (lane & 1)) idx += N / 32;
    return idx;
}

constexpr int REC_TILE = 256;
#ifndef RTTDA_K_MAXNI
#define RTTDA_K_MAXNI 3
#endif
#ifndef RTTDA_K_PP_MAXNI
#define RTTDA_K_PP_MAXNI 27
#endif
// classes whose two-stage integral ring (4 warps x 2 x NI x 256 bytes) leaves room for several blocks per SM
constexpr bool digest_uses_tma(int ni) { return ni <= 27; }
constexpr size_t digest_ring_bytes(int ni) { return digest_uses_tma(ni) ? (size_t)(JK_BLOCK / 32) * 2 * ni * 256 : 0; }      // a-list records staged in shared memory at a time

// ring stages of digest_b_kernel: two (the copy of record r+1 flies while record r is digested) while they fit in shared
// memory, one for the largest classes (648 integrals per quartet = 166 KB per stage)
constexpr int digest_b_stages(int ni) { return (size_t)2 * ni * 256 <= 200 * 1024 ? 2 : 1; }
constexpr int next_pow2(int n) { return n <= 1 ? 1 : (n <= 2 ? 2 : (n <= 4 ? 4 : (n <= 8 ? 8 : (n <= 16 ? 16 : 32)))); }

struct DigestArgs {
    JKTables tb;
    const WorkItem* work;
    const long long* batch_base;
    const double* buf;
    const double* Tq;
    const double* PPq;      // symmetric / antisymmetric density pairs {T + T^T, T - T^T}, [mu][nu][v][2] (K-only kernel)
    double* Fq;
    double cx;
    int ketclass, same, nvt, v0;
    int nvleft;             // densities of this chunk (lanes v >= nvleft idle along)
};

template <int NV>
struct VecLoad {
    __device__ static __forceinline__ void ld(const double* __restrict__ p, double (&out)[NV])
    {
        if (NV % 2 == 0) {
            const double2* p2 = reinterpret_cast<const double2*>(p);
#pragma unroll
            for (int i = 0; i < NV / 2; ++i) {
                const double2 x = __ldg(p2 + i);
                out[2 * i] = x.x; out[2 * i + 1] = x.y;
            }
        } else {
#pragma unroll
            for (int i = 0; i < NV; ++i) out[i] = __ldg(p + i);
        }
    }
};

// Stored component order (jk_eval.cu): canonical pair orientation (first shell = higher l), eri_index of
// eri_eval.cuh: ((d * NC + c) * N2 + c2) * N1 + c1 with (c1, c2) the components of the canonical first/second
// shell.
// Coulomb part: J_cd += I (T_ab + T_ba) in registers over the canonical records of the a-list, J_ab += I (T_cd + T_dc)
// by one transposing warp butterfly per record; no per-lane density gathers at all.
template <int LA, int LB, int LC, int LD, int NV>
__global__ void __launch_bounds__(JK_BLOCK)
digest_j_kernel(DigestArgs g)
{
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    constexpr int NI = NA * NB * NC * ND;
    constexpr bool USE_TMA = digest_uses_tma(NI);
    const JKTables& tb = g.tb;
    const WorkItem wi = g.work[blockIdx.x];
    const AList al = tb.alists[wi.alist];
    const KetClass& kc = tb.kets[g.ketclass];
    const int q = wi.ket0 + threadIdx.x;
    const bool active = q < kc.n;
    const int qq = active ? q : kc.n - 1;
    const double Qq = active ? __ldg(kc.Q + qq) : 0.0;
    const int aoC = __ldg(kc.ao_c + qq), aoD = __ldg(kc.ao_d + qq);
    const bool cd_same = __ldg(kc.same + qq) != 0;
    const bool same_class = g.same != 0;
    const int aoA = al.ao_a;
    const size_t nao = tb.nao;
    const int nvt = g.nvt;
    const double* Tv = g.Tq + g.v0;
    double* Fv = g.Fq + g.v0;
    const size_t rs = nao * nvt;          // row stride of Tq / Fq
    const int lane = threadIdx.x & 31;
#define TQ(mu, nu) (Tv + (size_t)(mu) * rs + (size_t)(nu) * nvt)

    // S_cd = T_cd + T_dc for the J_ab update
    double Scd[NC][ND][NV];
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
        for (int d = 0; d < ND; ++d) {
            double x[NV], y[NV];
            VecLoad<NV>::ld(TQ(aoC + c, aoD + d), x);
            VecLoad<NV>::ld(TQ(aoD + d, aoC + c), y);
#pragma unroll
            for (int v = 0; v < NV; ++v) Scd[c][d][v] = x[v] + y[v];
        }

    double Jcd[NC][ND][NV];
#pragma unroll
    for (int v = 0; v < NV; ++v)
#pragma unroll
        for (int c = 0; c < NC; ++c)
#pragma unroll
            for (int d = 0; d < ND; ++d) Jcd[c][d][v] = 0.0;

    // The a-list's records and their staging-buffer offsets go through shared memory, REC_TILE at a time.  Each
    // warp streams its 32-ket batch of every record (NI x 256 contiguous bytes) from HBM into a two-stage shared
    // memory ring with TMA bulk copies: the copy of record r+1 is in flight while record r is digested.
    __shared__ BraRec s_rec[REC_TILE];
    __shared__ long long s_bb[REC_TILE];
    __shared__ __align__(8) uint64_t s_bar[JK_BLOCK / 32][2];
    extern __shared__ __align__(16) double s_dyn[];
    const int warp = threadIdx.x >> 5;
    double* ring = s_dyn + (size_t)warp * 2 * (NI * 32);
    if (USE_TMA) {
        if (lane == 0) { mbar_init(&s_bar[warp][0], 1); mbar_init(&s_bar[warp][1], 1); mbar_fence_init(); }
        __syncwarp();
    }
    uint32_t phase0 = 0, phase1 = 0;
    int stage = 0;
    const long long qb = q >> 5;                            // warp-uniform
    auto issue = [&](int ir, int s) {
        if (USE_TMA && lane == 0) {
            const double* gsrc = g.buf + (size_t)(s_bb[ir] + qb) * (NI * 32);
            mbar_expect_tx(&s_bar[warp][s], NI * 256);
            tma_load_1d(ring + (size_t)s * (NI * 32), gsrc, NI * 256, &s_bar[warp][s]);
        }
    };
    auto pred = [&](int ir) {
        const BraRec& b1 = s_rec[ir];
        return active && (b1.Q * Qq >= tb.tau) && (!same_class || b1.pos <= q);
    };
    bool done = false;                                      // warp-uniform
    const BraRec* recs = tb.jrecs;                          // the canonical records of the a-list
    const int rec_begin = al.jrec_begin, rec_end = al.jrec_end;
    for (int r0 = rec_begin; r0 < rec_end; r0 += REC_TILE) {
      const int nrec = min(REC_TILE, rec_end - r0);
      __syncthreads();
      for (int i = threadIdx.x; i < nrec; i += JK_BLOCK) {
          const BraRec b0 = recs[r0 + i];
          s_rec[i] = b0;
          s_bb[i] = __ldg(g.batch_base + b0.pos) - (same_class ? (b0.pos >> 5) : 0);
      }
      __syncthreads();
      bool ok_next = false;
      if (!done) {
          ok_next = pred(0);
          if (__any_sync(0xffffffffu, ok_next)) issue(0, stage); else done = true;
      }
      if (!done)
      for (int ir = 0; ir < nrec; ++ir) {
        const BraRec br = s_rec[ir];
        const bool ok = ok_next;
        bool more = false;
        if (ir + 1 < nrec) {
            ok_next = pred(ir + 1);
            more = __any_sync(0xffffffffu, ok_next);
            if (more) issue(ir + 1, stage ^ 1);
        }
        const bool ab_same = (br.flags & 2) != 0;
        const int aoB = br.ao_b;
        const double* src;
        if (USE_TMA) {
            src = ring + (size_t)stage * (NI * 32) + lane;
            if (stage == 0) { mbar_wait(&s_bar[warp][0], phase0); phase0 ^= 1; }
            else { mbar_wait(&s_bar[warp][1], phase1); phase1 ^= 1; }
        } else {
            src = g.buf + (size_t)(s_bb[ir] + qb) * (NI * 32) + lane;
        }
        // degeneracy weights: 1/2 if the ket is a diagonal pair, 1/2 if bra pair == ket pair
        // the stored values carry wsame * w_cd (jk_eval.cu) and are zero for lanes without a quartet;
        // J_cd needs wsame * w_ab instead
        const double fix = (cd_same ? 2.0 : 1.0) * (ab_same ? 0.5 : 1.0);
        // canonical records: a is the pair's first shell, the stored block is (a b|c d), a fastest
#pragma unroll
        for (int b = 0; b < NB; ++b) {
#pragma unroll
            for (int a = 0; a < NA; ++a) {
                double sab[NV], jab[next_pow2(NV)];
                {
                    double x[NV], y[NV];
                    VecLoad<NV>::ld(TQ(aoA + a, aoB + b), x);
                    VecLoad<NV>::ld(TQ(aoB + b, aoA + a), y);
#pragma unroll
                    for (int v = 0; v < NV; ++v) sab[v] = fix * (x[v] + y[v]);
                }
#pragma unroll
                for (int v = 0; v < next_pow2(NV); ++v) jab[v] = 0.0;
                // stored index of (a, b, c, d): first-shell component runs fastest
                const int i_ab = b * NA + a;
#pragma unroll
                for (int d = 0; d < ND; ++d)
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        const int i = (d * NC + c) * (NA * NB) + i_ab;
                        const double x = USE_TMA ? src[i * 32] : __ldcs(src + i * 32);
#pragma unroll
                        for (int v = 0; v < NV; ++v) {
                            Jcd[c][d][v] = fma(x, sab[v], Jcd[c][d][v]);
                            jab[v] = fma(x, Scd[c][d][v], jab[v]);
                        }
                    }
                // ---- J_ab: warp total of the kets' contributions
                {
                    constexpr int NP = next_pow2(NV);
                    const double tot = warp_reduce_multi<NP>(jab, lane);
                    const int v = warp_reduce_owner_index<NP>(lane);
                    if (v < NV && tot != 0.0 && (lane & (32 / NP - 1)) == 0) {
                        atomicAdd(Fv + (size_t)(aoA + a) * rs + (size_t)(aoB + b) * nvt + v, 2.0 * tot);
                        if (!ab_same)
                            atomicAdd(Fv + (size_t)(aoB + b) * rs + (size_t)(aoA + a) * nvt + v, 2.0 * tot);
                    }
                }
            }
        }
        if (USE_TMA) { __syncwarp(); stage ^= 1; }          // every lane is done with this stage before it is refilled
        if (!more) { if (ir + 1 < nrec) done = true; break; }
      }
      if (__syncthreads_and(done)) break;
    }
#undef TQ
    if (!active) return;
    // ---- flush the register accumulators: F += 2 J_cd
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
        for (int d = 0; d < ND; ++d) {
            red_add<NV>(Fv + (size_t)(aoC + c) * rs + (size_t)(aoD + d) * nvt, Jcd[c][d], 2.0);
            if (!cd_same) red_add<NV>(Fv + (size_t)(aoD + d) * rs + (size_t)(aoC + c) * nvt, Jcd[c][d], 2.0);
        }
}

// ---------------------------------------------------------------------------------------------------
// Block-per-batch, density-per-lane kernel: the block owns ONE 32-ket batch and walks an a-list; warp w holds
// KW = 32 / G kets of the batch, a group of G lanes per ket, lane v of the group serves density v.  The batch's
// integrals of each record (NI x 256 contiguous bytes) are fetched ONCE by a TMA bulk copy into a two-stage shared
// memory ring shared by all warps (the copy of record r+1 flies while record r is digested); every density access
// is a contiguous 16*G-byte run of an aligned slot of {Ps, Pa} pairs; a lane carries one density's accumulators
// only, so all densities of a chunk are served by one read of the staged integrals.  Exchange part only: with
//   U_ac = sum I Ps_bd, V_ac = sum I Pa_bd (Ps = T + T^T, Pa = T - T^T):  K_ac = (U + V)/2,  K_ca = (U - V)/2.
template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(256)
digest_b_kernel(DigestArgs g, int G, int KW)
{
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    constexpr int NI = NA * NB * NC * ND;
    const JKTables& tb = g.tb;
    const WorkItem wi = g.work[blockIdx.x >> 2];
    const AList al = tb.alists[wi.alist];
    const KetClass& kc = tb.kets[g.ketclass];
    const int q0 = wi.ket0 + 32 * (blockIdx.x & 3);      // first ket of this block's batch
    if (q0 >= kc.n) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kg = lane / G, v = lane - kg * G;
    const int kb = warp * KW + kg;                       // ket index inside the batch
    const int q = q0 + kb;
    const bool active = kg < KW && kb < 32 && q < kc.n && v < g.nvleft;
    const bool same_class = g.same != 0;
    const int aoA = al.ao_a;
    const size_t nao = tb.nao;
    const int nvt = g.nvt;
    const size_t rs = nao * nvt;
    const double* Tv = g.Tq + g.v0 + v;
    double* Fv = g.Fq + g.v0 + v;
    const double cx = g.cx;
#define TQ(mu, nu) (Tv + (size_t)(mu) * rs + (size_t)(nu) * nvt)
#define FQ(mu, nu) (Fv + (size_t)(mu) * rs + (size_t)(nu) * nvt)
    // {Ps, Pa}(mu, nu)[v]: one 16-byte load gives T_mn + T_nm and T_mn - T_nm, i.e. both T_mn and T_nm
    const double2* PPv = reinterpret_cast<const double2*>(g.PPq) + g.v0 + v;
#define PQ(mu, nu) (PPv + (size_t)(mu) * rs + (size_t)(nu) * nvt)
    __shared__ BraRec s_rec[REC_TILE];
    __shared__ long long s_bb[REC_TILE];
    __shared__ __align__(8) uint64_t s_bar[2];
    extern __shared__ __align__(16) double s_dyn[];      // ring: 2 stages x NI x 32 doubles
    if (threadIdx.x == 0) { mbar_init(&s_bar[0], 1); mbar_init(&s_bar[1], 1); mbar_fence_init(); }

    const double Qbatch = __ldg(kc.Q + q0);               // kets are sorted: the batch's largest bound
    const int qlast = min(q0 + 31, kc.n - 1);
    const long long qb = q0 >> 5;
    const int qq = active ? q : kc.n - 1;
    const double Qq = active ? __ldg(kc.Q + qq) : 0.0;
    const int aoC = __ldg(kc.ao_c + qq), aoD = __ldg(kc.ao_d + qq);
    const bool cd_same = __ldg(kc.same + qq) != 0;

    // Kac/Kad accumulate against Ps (symmetric part), Kca/Kda against Pa (antisymmetric part) of the density
    double Kac[NA][NC], Kca[NC][NA], Kad[NA][ND], Kda[ND][NA];
#pragma unroll
    for (int a = 0; a < NA; ++a) {
#pragma unroll
        for (int c = 0; c < NC; ++c) Kac[a][c] = Kca[c][a] = 0.0;
#pragma unroll
        for (int d2 = 0; d2 < ND; ++d2) Kad[a][d2] = Kda[d2][a] = 0.0;
    }

    // block-uniform test: does record ir reach any ket of this batch?
    auto reaches = [&](int ir) {
        const BraRec& b1 = s_rec[ir];
        return (b1.Q * Qbatch >= tb.tau) && (!same_class || b1.pos <= qlast);
    };
    auto issue = [&](int ir, int s) {
        if (threadIdx.x == 0) {
            const double* gsrc = g.buf + (size_t)(s_bb[ir] + qb) * (NI * 32);
            mbar_expect_tx(&s_bar[s], NI * 256);
            tma_load_1d(s_dyn + (size_t)s * (NI * 32), gsrc, NI * 256, &s_bar[s]);
        }
    };
    auto lane_ok = [&](int ir) {
        const BraRec& b1 = s_rec[ir];
        return active && (b1.Q * Qq >= tb.tau) && (!same_class || b1.pos <= q);
    };
    auto gather = [&](int ir, bool okx, double2 (&bd)[NB][ND], double2 (&bc)[NB][NC]) {
        const int aoBx = s_rec[ir].ao_b;
#pragma unroll
        for (int b = 0; b < NB; ++b) {
#pragma unroll
            for (int d2 = 0; d2 < ND; ++d2) bd[b][d2] = okx ? __ldg(PQ(aoBx + b, aoD + d2)) : make_double2(0.0, 0.0);
#pragma unroll
            for (int c = 0; c < NC; ++c) bc[b][c] = okx ? __ldg(PQ(aoBx + b, aoC + c)) : make_double2(0.0, 0.0);
        }
    };
    uint32_t phase0 = 0, phase1 = 0;
    int stage = 0;
    bool done = false;                                    // block-uniform
    for (int r0 = al.rec_begin; r0 < al.rec_end && !done; r0 += REC_TILE) {
        const int nrec = min(REC_TILE, al.rec_end - r0);
        __syncthreads();
        for (int i = threadIdx.x; i < nrec; i += blockDim.x) {
            const BraRec b0 = tb.recs[r0 + i];
            s_rec[i] = b0;
            s_bb[i] = __ldg(g.batch_base + b0.pos) - (same_class ? (b0.pos >> 5) : 0);
        }
        __syncthreads();
        if (!reaches(0)) { done = true; break; }
        issue(0, stage);
        // the density pairs of a record are gathered right after the previous record's arithmetic, i.e. before the
        // block barrier and the TMA wait of their own record: the L2 latency of the gathers overlaps both
        bool ok_cur = lane_ok(0);
        double2 cur_bd[NB][ND], cur_bc[NB][NC];
        gather(0, ok_cur, cur_bd, cur_bc);
        for (int ir = 0; ir < nrec; ++ir) {
            const BraRec br = s_rec[ir];
            const bool more = (ir + 1 < nrec) && reaches(ir + 1);
            __syncthreads();                              // every warp is done with the stage refilled next
            if constexpr (digest_b_stages(NI) == 2) { if (more) issue(ir + 1, stage ^ 1); }
            else { if (ir > 0) issue(ir, 0); }            // single stage: the copy cannot overlap the previous record
            if (stage == 0) { mbar_wait(&s_bar[0], phase0); phase0 ^= 1; }
            else { mbar_wait(&s_bar[1], phase1); phase1 ^= 1; }
            const double* src = s_dyn + (size_t)stage * (NI * 32) + (kb & 31);
            const bool ok = ok_cur;
            const bool canonical = (br.flags & 1) != 0;
            const bool flip = (LA < LB) || (LA == LB && !canonical);
            if (__any_sync(0xffffffffu, ok)) {
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    // tbd = Ps_bd, tdb = Pa_bd (and likewise for c): K_ac = (U + V)/2, K_ca = (U - V)/2 at the flush
                    double tbd[ND], tdb[ND], tbc[NC], tcb[NC];
#pragma unroll
                    for (int d2 = 0; d2 < ND; ++d2) { tbd[d2] = cur_bd[b][d2].x; tdb[d2] = cur_bd[b][d2].y; }
#pragma unroll
                    for (int c = 0; c < NC; ++c) { tbc[c] = cur_bc[b][c].x; tcb[c] = cur_bc[b][c].y; }
#pragma unroll
                    for (int a = 0; a < NA; ++a) {
                        const int i_ab = flip ? (a * NB + b) : (b * NA + a);
#pragma unroll
                        for (int d2 = 0; d2 < ND; ++d2)
#pragma unroll
                            for (int c = 0; c < NC; ++c) {
                                const int i = (d2 * NC + c) * (NA * NB) + i_ab;
                                const double x = src[i * 32];
                                Kac[a][c] = fma(x, tbd[d2], Kac[a][c]);
                                Kca[c][a] = fma(x, tdb[d2], Kca[c][a]);
                                Kad[a][d2] = fma(x, tbc[c], Kad[a][d2]);
                                Kda[d2][a] = fma(x, tcb[c], Kda[d2][a]);
                            }
                    }
                }
            }
            if constexpr (digest_b_stages(NI) == 2) stage ^= 1;
            if (!more) { if (ir + 1 < nrec) done = true; break; }
            ok_cur = lane_ok(ir + 1);
            gather(ir + 1, ok_cur, cur_bd, cur_bc);
        }
    }
    if (active) {
#pragma unroll
        for (int a = 0; a < NA; ++a) {
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                atomicAdd(FQ(aoA + a, aoC + c), -0.5 * cx * (Kac[a][c] + Kca[c][a]));
                atomicAdd(FQ(aoC + c, aoA + a), -0.5 * cx * (Kac[a][c] - Kca[c][a]));
            }
#pragma unroll
            for (int d2 = 0; d2 < ND; ++d2) {
                atomicAdd(FQ(aoA + a, aoD + d2), -0.5 * cx * (Kad[a][d2] + Kda[d2][a]));
                atomicAdd(FQ(aoD + d2, aoA + a), -0.5 * cx * (Kad[a][d2] - Kda[d2][a]));
            }
        }
    }
#undef TQ
#undef FQ
#undef PQ
}

// ---------------------------------------------------------------------------------------------------
// Exchange digestion, lean variant: same mapping as digest_b_kernel (block = one 32-ket batch x the a-list of one
// shell, a group of G lanes per ket, lane = density; the batch's integrals arrive through a block-wide TMA ring), but
//   * the stored integrals carry the degeneracy weights and are zero where no quartet exists (jk_eval.cu), so there
//     is no per-lane test in the loop: the block walks the first `nreach` records of the a-list (those whose batch
//     exists), found by one binary search per record tile;
//   * a ring stage holds KR records (KR bulk copies on one mbarrier), so the block barrier and the mbarrier wait are
//     paid once per KR records instead of once per record;
//   * the density pairs of record r+1 are gathered while record r is digested (two register sets, loop unrolled by 2).
constexpr int digest_k_recs(int ni) { return ni == 1 ? 16 : (ni == 3 ? 8 : (ni == 9 ? 4 : (ni == 27 ? 2 : 1))); }
constexpr size_t digest_k_smem(int ni) { return (size_t)2 * digest_k_recs(ni) * ni * 256; }

template <int NB, int NC, int ND>
struct KRec {
    double2 bd[NB][ND], bc[NB][NC];
};

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(256)
digest_k_kernel(DigestArgs g, int G, int KW)
{
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    constexpr int NI = NA * NB * NC * ND;
    constexpr int NAB = NA * NB;
    constexpr int KR = digest_k_recs(NI);
    constexpr bool PP = (NI < RTTDA_K_PP_MAXNI);                        // two register sets for the gathered density pairs
    const JKTables& tb = g.tb;
    const WorkItem wi = g.work[blockIdx.x >> 2];
    const AList al = tb.alists[wi.alist];
    const KetClass& kc = tb.kets[g.ketclass];
    const int q0 = wi.ket0 + 32 * (blockIdx.x & 3);      // first ket of this block's batch
    if (q0 >= kc.n) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kg = lane / G, v = lane - kg * G;
    const int kb = warp * KW + kg;                       // ket index inside the batch
    const int q = q0 + kb;
    const bool active = kg < KW && kb < 32 && q < kc.n && v < g.nvleft;
    const bool same_class = g.same != 0;
    const size_t nao = tb.nao;
    const int nvt = g.nvt;
    const size_t rs = nao * nvt;
    __shared__ unsigned long long s_ro[REC_TILE];        // row offset of shell b in the density-pair array | canonical bit
    __shared__ long long s_bb[REC_TILE];                 // offset of the record's batch in the staging buffer
    __shared__ double s_Q[REC_TILE];
    __shared__ int s_pos[REC_TILE];
    __shared__ __align__(8) uint64_t s_bar[2];
    extern __shared__ __align__(16) double s_dyn[];      // ring: 2 stages x KR records x NI x 32 doubles
    if (threadIdx.x == 0) { mbar_init(&s_bar[0], 1); mbar_init(&s_bar[1], 1); mbar_fence_init(); }

    const int qlast = min(q0 + 31, kc.n - 1);
    const double Qbatch = __ldg(kc.Q + q0);               // kets are sorted: the batch's largest bound
    const int qq = active ? q : q0;                       // idle lanes shadow a real ket (their results are dropped)
    const int aoC = __ldg(kc.ao_c + qq), aoD = __ldg(kc.ao_d + qq);
    const double2* PPv = reinterpret_cast<const double2*>(g.PPq) + g.v0 + (active ? v : 0);
    const double2* PD = PPv + (size_t)aoD * nvt;         // + (aoB + b) * rs + d2 * nvt
    const double2* PC = PPv + (size_t)aoC * nvt;
    const double* gbase = g.buf + (size_t)(q0 >> 5) * (NI * 32);
    const int kcol = active ? kb : 0;

    double Kac[NA][NC], Kca[NC][NA], Kad[NA][ND], Kda[ND][NA];
#pragma unroll
    for (int a = 0; a < NA; ++a) {
#pragma unroll
        for (int c = 0; c < NC; ++c) Kac[a][c] = Kca[c][a] = 0.0;
#pragma unroll
        for (int d2 = 0; d2 < ND; ++d2) Kad[a][d2] = Kda[d2][a] = 0.0;
    }
    using Rec = KRec<NB, NC, ND>;
    auto fetch = [&](int ir, Rec& r) {
        const size_t ro = (size_t)(s_ro[ir] >> 1);
#pragma unroll
        for (int b = 0; b < NB; ++b) {
#pragma unroll
            for (int d2 = 0; d2 < ND; ++d2) r.bd[b][d2] = __ldg(PD + ro + b * rs + d2 * nvt);
#pragma unroll
            for (int c = 0; c < NC; ++c) r.bc[b][c] = __ldg(PC + ro + b * rs + c * nvt);
        }
    };
    auto digest = [&](int ir, const double* src, const Rec& r) {
        const bool flip = (LA < LB) || (LA == LB && LA > 0 && !(s_ro[ir] & 1ull));
#pragma unroll
        for (int d2 = 0; d2 < ND; ++d2)
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                double x[NAB];
#pragma unroll
                for (int j = 0; j < NAB; ++j) x[j] = src[((d2 * NC + c) * NAB + j) * 32];
#pragma unroll
                for (int b = 0; b < NB; ++b)
#pragma unroll
                    for (int a = 0; a < NA; ++a) {
                        const double xi = flip ? x[a * NB + b] : x[b * NA + a];
                        Kac[a][c] = fma(xi, r.bd[b][d2].x, Kac[a][c]);
                        Kca[c][a] = fma(xi, r.bd[b][d2].y, Kca[c][a]);
                        Kad[a][d2] = fma(xi, r.bc[b][c].x, Kad[a][d2]);
                        Kda[d2][a] = fma(xi, r.bc[b][c].y, Kda[d2][a]);
                    }
            }
    };
    auto issue = [&](int r_begin, int r_end, int sidx) {  // thread 0: records [r_begin, r_end) of the tile into ring stage sidx
        mbar_expect_tx(&s_bar[sidx], (uint32_t)(r_end - r_begin) * NI * 256);
        for (int r = r_begin; r < r_end; ++r)
            tma_load_1d(s_dyn + ((size_t)sidx * KR + (r - r_begin)) * (NI * 32), gbase + s_bb[r], NI * 256, &s_bar[sidx]);
    };
    uint32_t phase0 = 0, phase1 = 0;
    bool done = false;                                    // block-uniform
    for (int r0 = al.rec_begin; r0 < al.rec_end && !done; r0 += REC_TILE) {
        const int nrec = min(REC_TILE, al.rec_end - r0);
        __syncthreads();
        for (int i = threadIdx.x; i < nrec; i += blockDim.x) {
            const BraRec b0 = tb.recs[r0 + i];
            s_ro[i] = ((unsigned long long)((size_t)b0.ao_b * rs) << 1) | (unsigned long long)(b0.flags & 1);
            s_bb[i] = (__ldg(g.batch_base + b0.pos) - (same_class ? (b0.pos >> 5) : 0)) * (long long)(NI * 32);
            s_Q[i] = b0.Q;
            s_pos[i] = b0.pos;
        }
        __syncthreads();
        // Records are sorted (bound descending, position ascending).  The batch of record p exists iff some ket q of
        // it has Q_p Q_q >= tau and (different classes or p <= q); the best candidate is q = max(p, q0), and
        // Q[p] = Q_p inside one class.  The records whose batch exists are a prefix of the list.
        int lo = 0, hi = nrec;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const double Qp = s_Q[mid];
            const int pos = s_pos[mid];
            const bool reach = same_class ? (pos <= qlast && Qp * (pos > q0 ? Qp : Qbatch) >= tb.tau)
                                          : (Qp * Qbatch >= tb.tau);
            if (reach) lo = mid + 1; else hi = mid;
        }
        const int nreach = lo;
        if (nreach < nrec) done = true;
        if (nreach == 0) break;
        const int nst = (nreach + KR - 1) / KR;
        if (threadIdx.x == 0) issue(0, min(KR, nreach), 0);
        Rec A, B;
        fetch(0, A);
        for (int st = 0; st < nst; ++st) {
            const int sidx = st & 1, rb = st * KR, re = min(rb + KR, nreach);
            if (threadIdx.x == 0 && st + 1 < nst) issue(re, min(re + KR, nreach), sidx ^ 1);
            if (sidx == 0) { mbar_wait(&s_bar[0], phase0); phase0 ^= 1; }
            else { mbar_wait(&s_bar[1], phase1); phase1 ^= 1; }
            const double* sbase = s_dyn + (size_t)sidx * KR * (NI * 32) + kcol;
            if (PP) {
                int ir = rb;
                for (; ir + 1 < re; ir += 2) {
                    fetch(ir + 1, B);
                    digest(ir, sbase + (size_t)(ir - rb) * (NI * 32), A);
                    if (ir + 2 < nreach) fetch(ir + 2, A);
                    digest(ir + 1, sbase + (size_t)(ir + 1 - rb) * (NI * 32), B);
                }
                if (ir < re) {                            // odd tail of the stage (KR == 1 or the last stage)
                    if (ir + 1 < nreach) fetch(ir + 1, B);
                    digest(ir, sbase + (size_t)(ir - rb) * (NI * 32), A);
                    if (ir + 1 < nreach) A = B;
                }
            } else {
                for (int ir = rb; ir < re; ++ir) {
                    if (ir > 0) fetch(ir, A);
                    digest(ir, sbase + (size_t)(ir - rb) * (NI * 32), A);
                }
            }
            __syncthreads();                              // every warp is done with this stage before it is refilled
        }
    }
    if (active) {
        const int aoA = al.ao_a;
        const double cx = g.cx;
        double* Fv = g.Fq + g.v0 + v;
        double* FA = Fv + (size_t)aoA * rs;
#pragma unroll
        for (int a = 0; a < NA; ++a) {
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                atomicAdd(FA + a * rs + (size_t)(aoC + c) * nvt, -0.5 * cx * (Kac[a][c] + Kca[c][a]));
                atomicAdd(Fv + (size_t)(aoC + c) * rs + (size_t)(aoA + a) * nvt, -0.5 * cx * (Kac[a][c] - Kca[c][a]));
            }
#pragma unroll
            for (int d2 = 0; d2 < ND; ++d2) {
                atomicAdd(FA + a * rs + (size_t)(aoD + d2) * nvt, -0.5 * cx * (Kad[a][d2] + Kda[d2][a]));
                atomicAdd(Fv + (size_t)(aoD + d2) * rs + (size_t)(aoA + a) * nvt, -0.5 * cx * (Kad[a][d2] - Kda[d2][a]));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
template <int LA, int LB, int LC, int LD, int NV>
static int launch_digest_j(Handle* h, const JKLaunch& L, const Segment& sg, const double* buf, int nvt, int v0,
                            const double* Tq, double* Fq, cudaStream_t st)
{
    DigestArgs g;
    g.tb = h->tabs;
    g.work = L.work;
    g.batch_base = sg.batch_base;
    g.buf = buf;
    g.Tq = Tq; g.PPq = nullptr; g.Fq = Fq; g.cx = h->pass_cx;
    g.ketclass = L.ketclass; g.same = (sg.kc_bra == sg.kc_ket); g.nvt = nvt; g.v0 = v0;
    constexpr int NI = (ncart(LA)) * (ncart(LB)) * (ncart(LC)) * (ncart(LD));
    constexpr size_t smem = digest_ring_bytes(NI);
    if (smem > 0)     // per launch: the attribute belongs to the current device's context, not to the process
        RT_CUDA(cudaFuncSetAttribute(digest_j_kernel<LA, LB, LC, LD, NV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    digest_j_kernel<LA, LB, LC, LD, NV><<<dim3(L.nwork), dim3(JK_BLOCK), smem, st>>>(g);
    h->kernel_launches++;
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

// One digestion launch group (ordered bra class x ket class) for the nvec (even) densities of the call:
//   Coulomb part  - digest_j_kernel over the canonical records, NVJ densities in registers per launch; launches of the
//                   flipped orientation (la < lb) hold no canonical record;
//   exchange part - digest_b_kernel, groups of G <= 8 lanes per ket (at most 8 warps per block), chunks of 8 densities.
template <int LA, int LB, int LC, int LD>
static int launch_digest(Handle* h, const JKLaunch& L, const Segment& sg, const double* buf, int nvt, int nvec,
                         const double* Tq, double* Fq, cudaStream_t st)
{
    constexpr int NC = ncart(LC), ND = ncart(LD);
    if (LA >= LB && h->pass_do_j) {
        constexpr int NVJ = (NC * ND <= 3) ? 8 : (NC * ND <= 9 ? 4 : 2);      // Scd and Jcd hold NC ND NVJ doubles each
        int v0 = 0;
        while (v0 < nvec) {
            const int left = nvec - v0;
            if (left >= NVJ) { RT_TRY((launch_digest_j<LA, LB, LC, LD, NVJ>(h, L, sg, buf, nvt, v0, Tq, Fq, st))); v0 += NVJ; }
            else if (NVJ == 8 && left >= 6) { RT_TRY((launch_digest_j<LA, LB, LC, LD, 6>(h, L, sg, buf, nvt, v0, Tq, Fq, st))); v0 += 6; }
            else if (left >= 4) { RT_TRY((launch_digest_j<LA, LB, LC, LD, 4>(h, L, sg, buf, nvt, v0, Tq, Fq, st))); v0 += 4; }
            else { RT_TRY((launch_digest_j<LA, LB, LC, LD, 2>(h, L, sg, buf, nvt, v0, Tq, Fq, st))); v0 += 2; }
        }
    }
    constexpr int NI = (ncart(LA)) * (ncart(LB)) * (ncart(LC)) * (ncart(LD));
    constexpr size_t smem = (size_t)digest_b_stages(NI) * NI * 256;
    if constexpr (NI > RTTDA_K_MAXNI)
        RT_CUDA(cudaFuncSetAttribute(digest_b_kernel<LA, LB, LC, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    else
        RT_CUDA(cudaFuncSetAttribute(digest_k_kernel<LA, LB, LC, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)digest_k_smem(NI)));
    if (!h->pass_do_k || h->pass_cx == 0.0) return RTTDA_OK;
    for (int v0 = 0; v0 < nvec; v0 += 8) {
        // lane groups of 2, 4 or 8 densities: a group then never straddles a quarter warp, so one 16-byte gather per
        // lane costs one L1 wavefront per ket (groups of 6 cost ~1.6); lanes beyond the call's densities work on the
        // zero padding slots and are not flushed
        const int left = nvec - v0, G = left > 4 ? 8 : (left > 2 ? 4 : 2);
        DigestArgs g;
        g.nvleft = left;
        g.tb = h->tabs; g.work = L.work; g.batch_base = sg.batch_base; g.buf = buf;
        g.Tq = Tq; g.PPq = h->wsP; g.Fq = Fq; g.cx = h->pass_cx;
        g.ketclass = L.ketclass; g.same = (sg.kc_bra == sg.kc_ket); g.nvt = nvt; g.v0 = v0;
        const int KW = 32 / G, nwarps = (32 + KW - 1) / KW;
        // one or three integrals per quartet: the multi-record ring (digest_k_kernel) wins; above that its larger
        // register footprint costs more occupancy than the saved barriers bring (profiles/README.md)
        if constexpr (NI > RTTDA_K_MAXNI) digest_b_kernel<LA, LB, LC, LD><<<dim3(4 * L.nwork), dim3(32 * nwarps), smem, st>>>(g, G, KW);
        else digest_k_kernel<LA, LB, LC, LD><<<dim3(4 * L.nwork), dim3(32 * nwarps), digest_k_smem(NI), st>>>(g, G, KW);
        h->kernel_launches++;
        RT_CUDA(cudaGetLastError());
    }
    return RTTDA_OK;
}

// All digestion work of one segment: the a-list launches of the s/p classes, or the general-path kernel.
int digest_segment(Handle* h, const Segment& sg, const double* buf, int nvt, int nvec, const double* Tq, double* Fq,
                   cudaStream_t st)
{
    if (sg.nlaunch == 0) return digest_segment_general(h, sg, buf, nvt, nvec, Tq, Fq, st);   // no a-list launches: general kernel
    for (int l = sg.first_launch; l < sg.first_launch + sg.nlaunch; ++l)
        RT_TRY(digest_launch(h, h->launches[l], sg, buf, nvt, nvec, Tq, Fq, st));
    return RTTDA_OK;
}

int digest_launch(Handle* h, const JKLaunch& L, const Segment& sg, const double* buf, int nvt, int nvec,
                  const double* Tq, double* Fq, cudaStream_t st)
{
    if (L.nwork == 0) return RTTDA_OK;
#define RT_DIGEST_CASE(A, B, C, D) \
    case ((A * 3 + B) * 3 + C) * 3 + D: return launch_digest<A, B, C, D>(h, L, sg, buf, nvt, nvec, Tq, Fq, st);
    switch (((L.la * 3 + L.lb) * 3 + L.lc) * 3 + L.ld) {
        RT_DIGEST_CASE(0, 0, 0, 0) RT_DIGEST_CASE(1, 0, 0, 0) RT_DIGEST_CASE(0, 1, 0, 0) RT_DIGEST_CASE(1, 0, 1, 0)
        RT_DIGEST_CASE(0, 1, 1, 0) RT_DIGEST_CASE(1, 1, 0, 0) RT_DIGEST_CASE(1, 1, 1, 0) RT_DIGEST_CASE(1, 1, 1, 1)
        // classes with a d shell (both orientations of the bra pair) up to DIGEST_ALIST_MAXNI integrals per quartet
        RT_DIGEST_CASE(2, 0, 0, 0) RT_DIGEST_CASE(0, 2, 0, 0) RT_DIGEST_CASE(2, 0, 1, 0) RT_DIGEST_CASE(0, 2, 1, 0)
        RT_DIGEST_CASE(2, 0, 1, 1) RT_DIGEST_CASE(0, 2, 1, 1) RT_DIGEST_CASE(2, 0, 2, 0) RT_DIGEST_CASE(0, 2, 2, 0)
        RT_DIGEST_CASE(2, 1, 0, 0) RT_DIGEST_CASE(1, 2, 0, 0) RT_DIGEST_CASE(2, 1, 1, 0) RT_DIGEST_CASE(1, 2, 1, 0)
        RT_DIGEST_CASE(2, 1, 1, 1) RT_DIGEST_CASE(1, 2, 1, 1) RT_DIGEST_CASE(2, 1, 2, 0) RT_DIGEST_CASE(1, 2, 2, 0)
        RT_DIGEST_CASE(2, 2, 0, 0) RT_DIGEST_CASE(2, 2, 1, 0) RT_DIGEST_CASE(2, 2, 1, 1)
        RT_DIGEST_CASE(2, 1, 2, 1) RT_DIGEST_CASE(1, 2, 2, 1) RT_DIGEST_CASE(2, 2, 2, 0) RT_DIGEST_CASE(2, 2, 2, 1)
        default: set_error("digest: unsupported class"); return RTTDA_EINVAL;
    }
#undef RT_DIGEST_CASE
}

// PP[mu][nu][v] = {T[mu][nu][v] + T[nu][mu][v], T[mu][nu][v] - T[nu][mu][v]}  (step a2 of DESIGN.md)
__global__ void symsplit_kernel(int nao, int nvt, const double* __restrict__ T, double2* __restrict__ PP)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = (long long)nao * nao * nvt;
    if (i >= n) return;
    const int v = (int)(i % nvt);
    const long long e = i / nvt;
    const int mu = (int)(e / nao), nu = (int)(e % nao);
    const double a = T[i], b = T[((long long)nu * nao + mu) * nvt + v];
    PP[i] = make_double2(a + b, a - b);
}

// One ERI pass: every segment is evaluated once into the staging buffer of its lane and then digested for all
// densities on the lane's stream; the lanes (Handle::lane_*) run side by side and join the caller's stream at the end
// (the Fock updates are atomic adds, so the lanes need no ordering among themselves).  Small molecules, whose kernels
// do not fill the GPU, run 8 lanes; large ones run the two-buffer pipeline below.  Fq must be zeroed by the caller; densities [0, nvec) of the nvt slots per
// element are processed (nvec even, nvt a multiple of 2 with 16-byte aligned slots).
int jk_build(Handle* h, int nvt, int nvec, const double* Tq, double* Fq, cudaStream_t st)
{
    RT_CHECK(nvec >= 2 && nvec % 2 == 0 && nvt >= nvec && nvt % 2 == 0, "jk_build: bad density slot counts");
    if (!h->incore) {
        for (int l = 0; l < h->nlanes; ++l) RT_TRY(ensure_ws(h, &h->eri_buf[l], &h->eri_buf_n[l], h->lane_need[l]));
        if (h->nlanes == 0)
            for (int b = 0; b < 2; ++b) RT_TRY(ensure_ws(h, &h->eri_buf[b], &h->eri_buf_n[b], h->eri_buf_need));
    }
    {                                   // the exchange kernel gathers {Ps, Pa} pairs: one 16-byte load per (T_mn, T_nm)
        const long long n = (long long)h->nao * h->nao * nvt;
        RT_TRY(ensure_ws(h, &h->wsP, &h->wsP_n, (size_t)2 * n));
        symsplit_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(h->nao, nvt, Tq, reinterpret_cast<double2*>(h->wsP));
        RT_CUDA(cudaGetLastError());
        h->kernel_launches++;
    }
    RT_CUDA(cudaMemsetAsync(h->d_primcount, 0, 8 * sizeof(unsigned long long), st));   // counters of THIS build
    const bool lr = (h->cx_lr != 0.0 && h->rs_omega > 0.0);
    RT_CHECK(!(lr && h->incore), "jk_build: the in-core store holds the integrals of ONE operator; switch RTTDA_OPT_INCORE off "
                                 "when range-separated exchange is on");
    // ERI passes of this build: the 1/r12 pass (Coulomb + c_x exchange), and, with range-separated exchange, a second
    // pass over the same quartets with the integrals of erf(omega r12)/r12, digested into the exchange part only
    const int npass = lr ? 2 : 1;
    for (int pass = 0; pass < npass; ++pass) {
    h->pass_w_extra = pass == 0 ? 0.0 : 36.0 / (h->rs_omega * h->rs_omega);
    h->pass_cx = pass == 0 ? h->cx : h->cx_lr;
    h->pass_do_j = (pass == 0);
    h->pass_do_k = true;
    if (h->incore) {
        // In-core mode (optional, off by default): every segment owns its part of one resident store; the first
        // pass fills it, later passes only digest.  This trades 8 bytes of HBM per integral for the evaluation.
        RT_TRY(ensure_ws(h, &h->eri_all, &h->eri_all_n, h->eri_all_need));
        for (const Segment& sg : h->segments) {
            if (sg.nitems == 0) continue;
            double* buf = h->eri_all + sg.incore_off;
            if (!h->incore_valid) RT_TRY(eval_segment(h, sg, buf, st));
            RT_TRY(digest_segment(h, sg, buf, nvt, nvec, Tq, Fq, st));
        }
        h->incore_valid = true;
        continue;
    }
    if (h->nlanes == 0) {
        // Pipeline mode (large molecules: every kernel fills the GPU on its own, and two kernels of the same kind
        // running side by side only fight over the FP64 pipe or over L1/L2): segments in order, evaluation of
        // segment k+1 on lane_st[0] beside the digestion of segment k on the caller's stream, two buffers.
        cudaStream_t se = h->lane_st[0];
        cudaEvent_t *evE = h->lane_ev, *evD = h->lane_ev + 2;
        RT_CUDA(cudaEventRecord(h->ev_fork, st));
        RT_CUDA(cudaStreamWaitEvent(se, h->ev_fork, 0));
        int k = 0;
        for (const Segment& sg : h->segments) {
            if (sg.nitems == 0) continue;
            const int b = k & 1;
            if (k >= 2) RT_CUDA(cudaStreamWaitEvent(se, evD[b], 0));
            RT_TRY(eval_segment(h, sg, h->eri_buf[b], se));
            RT_CUDA(cudaEventRecord(evE[b], se));
            RT_CUDA(cudaStreamWaitEvent(st, evE[b], 0));
            RT_TRY(digest_segment(h, sg, h->eri_buf[b], nvt, nvec, Tq, Fq, st));
            RT_CUDA(cudaEventRecord(evD[b], st));
            ++k;
        }
        // the evaluation stream's last kernels were consumed by the digestion above; a following pass reuses the buffers
        continue;
    }
    RT_CUDA(cudaEventRecord(h->ev_fork, st));
    for (int l = 0; l < h->nlanes; ++l) {
        if (h->lane_segs[l].empty()) continue;
        cudaStream_t ls = h->lane_st[l];
        RT_CUDA(cudaStreamWaitEvent(ls, h->ev_fork, 0));
        for (int si : h->lane_segs[l]) {
            const Segment& sg = h->segments[si];
            RT_TRY(eval_segment(h, sg, h->eri_buf[l], ls));
            RT_TRY(digest_segment(h, sg, h->eri_buf[l], nvt, nvec, Tq, Fq, ls));
        }
        RT_CUDA(cudaEventRecord(h->lane_ev[l], ls));
        RT_CUDA(cudaStreamWaitEvent(st, h->lane_ev[l], 0));
    }
    }   // passes
    h->pass_w_extra = 0.0; h->pass_cx = h->cx; h->pass_do_j = h->pass_do_k = true;
    return RTTDA_OK;
}

// Timing instrumentation: ONE ERI pass with every segment's evaluation and digestion timed by its
// own pair of CUDA events, everything serialised on `st`.  rows[k][16] (host) = {segment, bra class, ket class, la, lb,
// lc, ld, bra primitive pairs, ket primitive pairs, quartets, 32-ket batches, evaluation ms, digestion ms, evaluation
// blocks, digestion launches, 0}.
int jk_profile(Handle* h, int nvt, int nvec, const double* Tq, double* Fq, cudaStream_t st, double* rows, int cap, int* nrows)
{
    RT_TRY(ensure_ws(h, &h->eri_buf[0], &h->eri_buf_n[0], h->eri_buf_need));
    const long long n = (long long)h->nao * h->nao * nvt;
    RT_TRY(ensure_ws(h, &h->wsP, &h->wsP_n, (size_t)2 * n));
    symsplit_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(h->nao, nvt, Tq, reinterpret_cast<double2*>(h->wsP));
    RT_CUDA(cudaGetLastError());
    cudaEvent_t e[3];
    for (auto& x : e) RT_CUDA(cudaEventCreate(&x));
    int k = 0;
    for (size_t si = 0; si < h->segments.size(); ++si) {
        const Segment& sg = h->segments[si];
        if (sg.nitems == 0 || k >= cap) continue;
        RT_CUDA(cudaEventRecord(e[0], st));
        RT_TRY(eval_segment(h, sg, h->eri_buf[0], st));
        RT_CUDA(cudaEventRecord(e[1], st));
        RT_TRY(digest_segment(h, sg, h->eri_buf[0], nvt, nvec, Tq, Fq, st));
        RT_CUDA(cudaEventRecord(e[2], st));
        RT_CUDA(cudaEventSynchronize(e[2]));
        float me = 0, md = 0;
        RT_CUDA(cudaEventElapsedTime(&me, e[0], e[1]));
        RT_CUDA(cudaEventElapsedTime(&md, e[1], e[2]));
        double* r = rows + (size_t)k * 16;
        r[0] = (double)si; r[1] = sg.kc_bra; r[2] = sg.kc_ket; r[3] = sg.la; r[4] = sg.lb; r[5] = sg.lc; r[6] = sg.ld;
        r[7] = h->tabs.kets[sg.kc_bra].np; r[8] = h->tabs.kets[sg.kc_ket].np; r[9] = (double)sg.nquartets;
        r[10] = (double)sg.nbatch; r[11] = me; r[12] = md; r[13] = sg.nitems; r[14] = sg.nlaunch; r[15] = 0.0;
        ++k;
    }
    for (auto& x : e) cudaEventDestroy(x);
    *nrows = k;
    return RTTDA_OK;
}

}  // namespace rttda
