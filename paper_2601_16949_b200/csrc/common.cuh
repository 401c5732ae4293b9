// Shared declarations of the rttda CUDA library (product path; shares nothing with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>
#include "../../include/rttda.h"

namespace rttda {

void set_error(const std::string& msg);

#define RT_CUDA(call)                                                                         \
    do {                                                                                      \
        cudaError_t e__ = (call);                                                             \
        if (e__ != cudaSuccess) {                                                             \
            ::rttda::set_error(std::string(#call) + ": " + cudaGetErrorString(e__));          \
            return RTTDA_ECUDA;                                                               \
        }                                                                                     \
    } while (0)

#define RT_CHECK(cond, msg)                                                                   \
    do {                                                                                      \
        if (!(cond)) {                                                                        \
            ::rttda::set_error(msg);                                                          \
            return RTTDA_EINVAL;                                                              \
        }                                                                                     \
    } while (0)

#define RT_TRY(expr)                                                                          \
    do {                                                                                      \
        int r__ = (expr);                                                                     \
        if (r__ != RTTDA_OK) return r__;                                                      \
    } while (0)

// ---------------------------------------------------------------------------------------------
// Shell-pair tables.
//
// A primitive pair record (12 doubles, one 96-byte row) of an ORDERED shell pair (first, second):
//   [0] p = a+b   [1..3] P   [4] c = sqrt(2) pi^(5/4) / p * coefA coefB exp(-mu |AB|^2)
//   [5] 1/(2p)    [6..8] P - A(first)   [9..11] P - B(second)
// so that c_bra * c_ket / sqrt(p+q) = 2 pi^(5/2) / (p q sqrt(p+q)) * K_ab K_cd * coefficients.
constexpr int PRIM_STRIDE = 12;

// Pair classes (higher l first): 0 = ss, 1 = ps, 2 = pp, 3 = ds, 4 = dp, 5 = dd; contraction sub-class by number of
// primitive pairs kept after primitive screening (setup.cu), rounded up to 1, 3, 6 or 9.
constexpr int NSUB = 4;                       // primitive pairs stored per shell pair: {1, 3, 6, 9}
constexpr int NPAIRCLASS = 6;
constexpr int NKETCLASS = NPAIRCLASS * NSUB;  // ket class id = pairclass * NSUB + sub
__host__ __device__ constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }     // Cartesian components of a shell
inline int pairclass_of(int l1, int l2) { return l1 * (l1 + 1) / 2 + l2; }       // l1 >= l2
inline int pairclass_l1(int pc) { return pc >= 3 ? 2 : (pc >= 1 ? 1 : 0); }
inline int pairclass_l2(int pc) { return pc - pairclass_l1(pc) * (pairclass_l1(pc) + 1) / 2; }
__host__ __device__ inline int sub_to_np(int sub) { return sub == 0 ? 1 : (sub == 1 ? 3 : (sub == 2 ? 6 : 9)); }

// Unique (unordered) pairs of one pair class (pair type x contraction sub-class), sorted by Schwarz bound
// descending.  The same list serves as the BRA list of the evaluation kernels (block-uniform side, AoS rows
// staged in shared memory) and as the KET list (thread-owned side, SoA so that consecutive kets coalesce).
// Primitive data SoA: prim[(k * PRIM_STRIDE + f) * n + q]; AoS: prim_aos[(q * np + k) * PRIM_STRIDE + f].
struct KetClass {
    int n;                 // number of pairs
    int np;                // primitive pairs per pair (1, 3, 9)
    const double* Q;       // [n] Schwarz bounds, descending
    const int* ao_c;       // [n] AO offset of the first (higher-l) shell
    const int* ao_d;       // [n] AO offset of the second shell
    const int* same;       // [n] 1 if both shells are the same shell
    const double* prim;    // [np][PRIM_STRIDE][n]
    const double* prim_aos;// [n][np][PRIM_STRIDE]
    const float* qp;       // [np][n]  primitive-pair bounds q_k = sqrt(max (kk|kk)), rounded up, descending in k
    const float* qp_aos;   // [n][np]
};

// Ordered bra record of the digestion kernels (block-uniform side): shell a fixed by the list, partner b varies.
struct BraRec {
    double Q;              // Schwarz bound of the pair
    int ao_b;              // AO offset of partner shell b
    int pos;               // position of the unordered pair inside its class list
    int flags;             // bit0: canonical orientation (a is the pair's first shell; does the J work), bit1: a == b
    int pad;
};

// All partners b of shell a with given l_b and contraction sub-class, sorted by Q descending.
struct AList {
    double Qmax;
    int ao_a;
    int rec_begin, rec_end;   // into BraRec array
    int jrec_begin, jrec_end; // into the array of canonical records only (J-only digestion)
    int ketclass;             // class id of the (unordered) pairs in this list
    int np;                   // primitive pairs per record
};

struct WorkItem {
    int alist;
    int ket0;                 // first ket (thread 0) of this block
};

// One block of the evaluation kernel: JK_BLOCK consecutive kets x bra pairs [p_begin, p_end) of the bra list.
struct EvalItem {
    int k0, p_begin, p_end;
};

// A segment = all unique quartets (bra pair class x ket pair class).  The evaluation kernel writes the
// contracted integrals of the segment to the staging buffer in HBM, batch by batch; a batch is one bra pair
// x 32 consecutive kets, laid out [component][lane] so that both sides coalesce:
//   value(pair p, ket q, component i) at  ((batch_base[p] + (q >> 5) - (same ? p >> 5 : 0)) * NI + i) * 32 + (q & 31)
// A quartet exists iff Q_p Q_q >= tau and (bra class != ket class or p <= q).
struct Segment {
    int kc_bra, kc_ket;       // class ids (pair type * NSUB + sub) of the bra and ket lists
    int la, lb, lc, ld;       // canonical angular momenta (la >= lb, lc >= ld)
    int ni;                   // integrals per quartet
    long long nbatch;         // 32-ket batches in the segment
    size_t incore_off;        // offset (doubles) of this segment in the in-core integral store
    long long nquartets;      // quartets actually evaluated (unique, screened)
    const long long* batch_base;   // device [n_bra]
    const EvalItem* items;    // device
    int nitems;
    int first_launch, nlaunch;     // digestion launches that read this segment
};

struct JKLaunch {             // one digestion kernel instantiation: ordered bra class x ket class
    int la, lb, lc, ld, ketclass;
    int seg;
    int nwork;
    const WorkItem* work;     // device
};

struct JKTables {
    KetClass kets[NKETCLASS];
    const BraRec* recs;
    const BraRec* jrecs;      // the canonical records of every a-list, in the same order
    const AList* alists;
    const double2* boys[9];   // per total angular momentum L (0..8): rows {F_{L+k}(j/8)/k!, k < 8; exp(-j/8); pad}
    double tau;
    int nao;
};

constexpr int JK_BLOCK = 128;
constexpr int EVAL_MAX_ROWS = 144;     // bra primitive rows staged per evaluation block (16 pairs x 9 prims)

// Boys grid: T0 = j / 8, j = 0..BOYS_NROW-1; BOYS_ROW doubles per row (eri_eval.cuh)
constexpr int BOYS_ROW = 10;
constexpr double BOYS_TMAX = 36.0;
constexpr int BOYS_NROW = 289 + 1;
void boys_table_host(int L, std::vector<double>& tab);

// ---------------------------------------------------------------------------------------------
struct Handle {
    int device = 0;
    int nao = 0, nocc = 0, nvirt = 0, ncsf = 0, nshells = 0;
    unsigned long long* d_primcount = nullptr; // [8] primitive quartets evaluated in the last ERI pass: [0..4] s/p classes by total L
                                               // (jk_eval.cu), [5] all classes of the general path (eri_generic.cu), [6] their model flops
    double cx = 1.0, tau = 0.0;
    // range-separated exchange (NEXT-4): A -= cx_lr (ij| erf(omega r12)/r12 |ab); rs_omega <= 0 or cx_lr == 0: off
    double cx_lr = 0.0, rs_omega = 0.0;
    // operator and digestion mode of the ERI pass being enqueued (set by jk_build, read by eval_segment / digest_launch)
    double pass_w_extra = 0.0;                 // 36 / omega^2 added to w = 36/p + 36/q: integrals of erf(omega r)/r
    double pass_cx = 1.0;                      // exchange factor of this pass
    bool pass_do_j = true, pass_do_k = true;
    // device-resident inputs
    double *C_occ = nullptr, *C_virt = nullptr, *deps = nullptr;
    double* D_ao = nullptr;                    // [3][nao][nao]
    double *D_oo = nullptr, *D_vv = nullptr, *D_ov = nullptr;   // [3][..]
    double D_00[3] = {0, 0, 0};
    // J/K tables
    JKTables tabs{};
    std::vector<JKLaunch> launches;
    std::vector<Segment> segments;
    // HBM staging buffers: the segments are dealt to `nlanes` lanes (setup.cu, longest first onto the least loaded
    // lane); a lane owns one stream and one buffer of the size of its largest segment and runs evaluate -> digest ->
    // evaluate -> ... for its segments, so kernels of different lanes overlap (the FP64-bound evaluation of one
    // segment beside the L1/L2-bound digestion of another, and each other's tails).
    static constexpr int MAXLANES = 8;
    int nlanes = 0;
    std::vector<int> lane_segs[MAXLANES];
    double* eri_buf[MAXLANES] = {nullptr};
    size_t eri_buf_n[MAXLANES] = {0};          // doubles allocated
    size_t lane_need[MAXLANES] = {0};          // doubles needed by the lane's largest segment
    size_t eri_buf_need = 0;                   // doubles needed by the largest segment
    cudaStream_t lane_st[MAXLANES] = {nullptr};
    cudaEvent_t lane_ev[MAXLANES] = {nullptr};
    cudaEvent_t ev_fork = nullptr;
    // optional in-core mode (rttda_set_option): all segments' integrals kept in HBM after the first pass
    bool incore = false, incore_valid = false;
    double* eri_all = nullptr;
    size_t eri_all_n = 0, eri_all_need = 0;
    std::vector<void*> dev_allocs;             // everything to free
    // workspaces (grown on demand)
    double *wsY = nullptr, *wsT = nullptr, *wsF = nullptr, *wsZ = nullptr, *wsP = nullptr;
    size_t wsY_n = 0, wsT_n = 0, wsF_n = 0, wsZ_n = 0, wsP_n = 0;
    double* prop_ws = nullptr;
    size_t prop_ws_n = 0;
    // CUDA graph of one RK4 step (propagate.cu): device-side control block, cached executable graph and its key
    void* d_ctl = nullptr;
    cudaGraphExec_t step_graph = nullptr;
    cudaStream_t graph_st = nullptr;
    cudaEvent_t graph_ev = nullptr;
    struct GraphKey { int ntraj = 0; const double* y = nullptr; unsigned active = 0; int nlanes = -1; long long epoch = -1; } graph_key;
    long long ws_epoch = 0;                    // bumped whenever a workspace is reallocated
    long long graph_launches = 0;              // kernels inside one replay of step_graph
    double graph_dt = 0.0;
    bool use_graph = false, capturing = false;
    // propagator state kept across calls: polarisations of the cached D_d matrices, reference state of R(t)
    bool dd_valid = false;
    int dd_ntraj = 0, yref_ntraj = 0;
    double dd_dir[8][3] = {{0}};
    // info
    double info[16] = {0};
    long long kernel_launches = 0;
    cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false;
    // pairs of events around every J/K build since the last rttda_jk_time query
    std::vector<cudaEvent_t> jk_ev;
    size_t jk_ev_used = 0;
};

int jk_mark(Handle* h, cudaStream_t st);
int assign_lanes(Handle* h, int nlanes);
// Primitive-level screening threshold: three orders below the shell-level one, and never looser than 1e-15, so that its
// error stays far below both the shell screening error and the 1e-10 sigma tolerance at any tau.
inline double prim_threshold(double tau) { return tau * 1e-3 < 1e-15 ? tau * 1e-3 : 1e-15; }
double flops_prim(int la, int lb, int lc, int ld);
double flops_prim_L(int L);                // flop model of one primitive quartet of total angular momentum L   // record the next event of the J/K timing log

// jk_eval.cu / jk_digest.cu
// F += 2 J[T] - cx K[T] for all nvt (even) interleaved densities; F zeroed by the caller.
int jk_build(Handle* h, int nvt, int nvec, const double* Tq, double* Fq, cudaStream_t st);
int jk_profile(Handle* h, int nvt, int nvec, const double* Tq, double* Fq, cudaStream_t st, double* rows, int cap, int* nrows);
int eval_segment(Handle* h, const Segment& sg, double* buf, cudaStream_t st);
int digest_launch(Handle* h, const JKLaunch& L, const Segment& sg, const double* buf, int nvt, int nvec, const double* Tq,
                  double* Fq, cudaStream_t st);
inline int padded_nvec(int nvec) { return nvec <= 2 ? 2 : (nvec <= 4 ? 4 : ((nvec + 7) & ~7)); }
int schwarz_device(int pairclass, int npairs, const int* d_np, const int* d_off, const double* d_prim,
                   const double2* d_boys /* table for L = 2 * pairclass */, double* d_Q, cudaStream_t st);
// eri_generic.cu: the general-angular-momentum path (classes with a d shell)
bool segment_is_general(const Segment& sg);
// the a-list digestion kernels (jk_digest.cu) are instantiated for the s/p classes and for these d classes
inline bool digest_has_alist_kernels(const Segment& sg)
{
    if (sg.la <= 1) return true;                                   // s/p (canonical order: la is the largest)
    if (getenv("RTTDA_GENERIC_DIGEST")) return false;
    const int bra = sg.la * 3 + sg.lb, ket = sg.lc * 3 + sg.ld;    // (2,0) = 6, (2,1) = 7, (2,2) = 8
    if (bra == 6) return ket == 0 || ket == 3 || ket == 4 || ket == 6;
    if (bra == 7) return ket == 0 || ket == 3 || ket == 4 || ket == 6 || ket == 7;
    if (bra == 8) return ket == 0 || ket == 3 || ket == 4 || ket == 6 || ket == 7;
    return false;
}
int eval_segment_general(Handle* h, const Segment& sg, double* buf, cudaStream_t st);
// jk_eval_d.cu: unrolled kernels for the d classes up to L = 5 (*handled = false: not one of them)
int eval_segment_d(Handle* h, const Segment& sg, double* buf, cudaStream_t st, bool* handled);
int digest_segment_general(Handle* h, const Segment& sg, const double* buf, int nvt, int nvec, const double* Tq, double* Fq,
                           cudaStream_t st);
int schwarz_general(int la, int lb, int npairs, const int* d_np, const int* d_off, const double* d_prim,
                    const double2* d_boys /* table for L = 2 (la + lb) */, double* d_Q, cudaStream_t st);
// evaluate + digest one segment (fast or general path)
int digest_segment(Handle* h, const Segment& sg, const double* buf, int nvt, int nvec, const double* Tq, double* Fq,
                   cudaStream_t st);

// gemm_f64.cu: C(m,n) = alpha * sum_k A(m,k) B(k,n) + beta * C(m,n), fully strided, batched.
struct GemmDesc {
    int M, N, K, batch;
    const double* A; long long sam, sak, sabatch;
    const double* B; long long sbk, sbn, sbbatch;
    double* C;       long long scm, scn, scbatch;
    double alpha, beta;
    const double* alpha_dev;   // optional DEVICE scalar multiplying alpha (read at run time: CUDA-graph friendly)
};
int gemm_f64(const GemmDesc& g, cudaStream_t st);

// propagate.cu
int propagate_impl(Handle* h, int ntraj, double* C, const rttda_field_t* fields, double t_start,
                   double dt, int nsteps, double* log, cudaStream_t st);
int propagate_sso_impl(Handle* h, int ntraj, double* C, const rttda_field_t* fields, double t_start,
                       double dt, int nsteps, double* log, cudaStream_t st);
int lanczos_impl(Handle* h, int m, const double* v0, double* alpha, double* beta, double* V, cudaStream_t st);
int spectrum_impl(int ntraj, int n, const double* R0, const double* log, double dt, int pad, int nout, double* omega,
                  double* inten, cudaStream_t st);
int populations_impl(Handle* h, int ntraj, const double* y, int nstates, const double* Xs, double* P, cudaStream_t st);
int sigma_impl(Handle* h, int nvec, const double* X, long long ldx, double* sigma, long long lds,
               cudaStream_t st);
int ensure_ws(Handle* h, double** p, size_t* cur, size_t need);
int sigma_reserve(Handle* h, int nvec);
int project_out(long long n, int nv, const double* V, double* w, double* dots, cudaStream_t st);
// eigs.cu
int eigs_impl(Handle* h, int k, int nblock, double tol, int maxiter, double* omega, double* X, double* resid, int* niter,
              int* nsigma, cudaStream_t st);

}  // namespace rttda
