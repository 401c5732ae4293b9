/* rttda.h -- C-ABI boundary of the B200-native RT-TDA sigma-vector / propagation library.
 *
 * What it computes (citations: P:NNN = /root/reference/PAPER.md line NNN, arXiv 2601.16949;
 * Rn = reading n in DESIGN.md):
 *   sigma = A X,  A_{ia,jb} = d_ij d_ab (eps_a - eps_i) + 2 (ia|jb) - c_x (ij|ab)     eq. 3 P:59 (R1), eq. 11
 *   index ia = i*nvirt + a (virtuals run fastest)
 *   direct CI through AO-basis Coulomb/exchange builds on the GPU
 *   i dC/dt = H(t) C,  H(t) = A_ext + E(t) M_d  (M_d from MO dipoles, Slater-Condon;    eq. 1, eq. 16 P:134,
 *   dipole origin = electronic centroid of the ground state, R6)
 *                                                                                       eq. 19 P:161-173 (R3-R5)
 *   C = q + i p, ground-state element first                                             eq. 12
 *   pulses                                                                              eq. 18a-d P:146-153 (R8, R9)
 *   R(t) = C(t0+)^dagger C(t)                                                           eq. 20
 *
 * Conventions
 *   - every call returns RTTDA_OK (0) or a negative RTTDA_E* code; the message of the last failure of the
 *     calling thread is available from rttda_last_error().  No C++ exception crosses the boundary.
 *   - "DEVICE" pointers are CUDA device memory on the handle's device; "host" pointers are ordinary host
 *     memory.  The caller owns every buffer it passes; the handle copies what it keeps.
 *   - rttda_sigma / rttda_fock / rttda_propagate only ENQUEUE work on `stream` (a cudaStream_t cast to void*,
 *     NULL = the legacy default stream) and return without synchronising; the *_host variants copy in,
 *     run, copy out and synchronise the stream before returning.
 *   - all floating point is IEEE binary64; all matrices are row-major.
 *   - a handle is bound to the device current at rttda_create; concurrent calls on one handle are not supported.
 *   - there is no CPU fallback: without a CUDA device every compute call fails with RTTDA_ECUDA.
 */
#ifndef RTTDA_H
#define RTTDA_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RTTDA_OK      0
#define RTTDA_EINVAL -1   /* bad shapes, l > 1, nocc + nvirt != nao, nvec < 1, NULL pointer, ... */
#define RTTDA_ENOMEM -2
#define RTTDA_ECUDA  -3   /* CUDA runtime error; string in rttda_last_error() */
#define RTTDA_ENOCONV -4  /* iterative solver stopped at maxiter; outputs hold the current iterate */

typedef struct rttda_handle_s* rttda_handle_t;   /* opaque; owns all internal device memory */

/* One contracted Cartesian Gaussian shell: l = 0 (s), 1 (p: components x, y, z) or 2 (d: the six Cartesian components
 * xx, xy, xz, yy, yz, zz, each normalised to <phi|phi> = 1, "6-31G*").  AO order = shell
 * order, so nao = sum over shells of (l+1)(l+2)/2. */
typedef struct {
    int32_t center;     /* index into centers */
    int32_t l;          /* 0, 1 or 2 */
    int32_t nprim;      /* 1..RTTDA_MAX_NPRIM */
    int32_t prim_off;   /* offset of this shell's primitives in exps / coefs */
} rttda_shell_t;

#define RTTDA_MAX_NPRIM 3

typedef struct {
    const double* centers;        /* host, [ncenters][3], bohr */
    int32_t ncenters, nshells;
    const rttda_shell_t* shells;  /* host, [nshells] */
    const double* exps;           /* host, [sum nprim] Gaussian exponents */
    const double* coefs;          /* host, [sum nprim]; multiply NORMALISED primitives; the library rescales
                                     each contracted function to <phi|phi> = 1 (R11) */
} rttda_basis_t;

/* Pulse shapes, eq. 18a-d.  SIN2 is config 4's envelope (R9):
 *   DELTA  linearised kick of area E0 applied at t_start: C <- (1 - i E0 M_d) C, then field free (R8)
 *   CW     E0 sin(omega t)
 *   TL     E0 exp(-(t-t0)^2 / (2 sigma^2)) sin(omega (t-t0))
 *   CHIRP  E0 exp(-(t-t0)^2 / (2 sigma^2)) sin((omega + beta (t-t0)/2)(t-t0))
 *   SIN2   E0 sin^2(pi t / T_env) sin(omega t) for 0 <= t <= T_env, else 0 */
typedef enum { RTTDA_NONE = 0, RTTDA_DELTA = 1, RTTDA_CW = 2, RTTDA_TL = 3, RTTDA_CHIRP = 4,
               RTTDA_SIN2 = 5 } rttda_pulse_t;

#define RTTDA_FIELD_CONTINUE 1   /* flags bit: this call CONTINUES the previous rttda_propagate / _sso call of the handle:
                                  no delta kick is applied and R(t) stays relative to the reference state of that call */
typedef struct {
    int32_t type;                               /* rttda_pulse_t */
    int32_t flags;                              /* 0 or RTTDA_FIELD_CONTINUE (setting it in any record marks the call) */
    double E0, omega, t0, sigma, beta, T_env;
    double dir[3];                              /* polarisation d (used as given, not renormalised) */
} rttda_field_t;

/* ---- host-only helpers (no GPU needed) ------------------------------------------------------------ */

/* Overlap matrix S [nao][nao] (host) of the renormalised contracted basis; used by callers to build
 * orthonormal MOs (C = S^-1/2 Q).  EINVAL if nao does not match the shell table. */
int rttda_overlap(const rttda_basis_t* basis, int32_t nao, double* S);

/* Position-operator matrices D^k_{mu nu} = <mu| r_k |nu> about the coordinate origin (0,0,0); D host [3][nao][nao].
 * (A handle shifts its own copies to the electronic centroid of the ground state, R6.) */
int rttda_dipole_ao(const rttda_basis_t* basis, int32_t nao, double* D);

/* ---- handle -------------------------------------------------------------------------------------- */

/* Once per molecule: normalise shells, build the Schwarz-sorted shell-pair tables and work lists,
 * MO-basis dipole blocks and eps_a - eps_i.  Synchronises `stream` before returning.
 *   C_occ  DEVICE [nao][nocc], C_virt DEVICE [nao][nvirt] (copied), eps host [nocc+nvirt] occupied first,
 *   cx = exact-exchange fraction c_x (1.0 in every config), schwarz_tau: a shell quartet (ab|cd) is skipped
 *   iff Q_ab Q_cd < tau, Q_ab = sqrt(max (mu nu|mu nu)) (R14); tau = 0 keeps everything. */
int rttda_create(rttda_handle_t* h, const rttda_basis_t* basis, int32_t nao, int32_t nocc, int32_t nvirt,
                 const double* C_occ, const double* C_virt, const double* eps, double cx,
                 double schwarz_tau, void* stream);

int rttda_destroy(rttda_handle_t h);

/* sigma_v = A x_v for v < nvec (singles block only, R16).  X, sigma DEVICE [nvec][nocc*nvirt]; must not
 * alias.  Steps a1-a5 of DESIGN.md: MO->AO transform (FP64 tensor-core GEMM), Schwarz-screened direct J/K
 * (ONE evaluation pass serves all densities of the call), AO->MO transform + (eps_a - eps_i) x. */
int rttda_sigma(rttda_handle_t h, int32_t nvec, const double* X, double* sigma, void* stream);

/* Same with HOST buffers: H2D copy of X, sigma build, D2H copy of sigma, stream synchronised. */
int rttda_sigma_host(rttda_handle_t h, int32_t nvec, const double* X, double* sigma, void* stream);

/* The AO-direct build alone (steps a3-a4): F_v = 2 J[T_v] - c_x K[T_v] for arbitrary (non-symmetric)
 * AO matrices T_v; J_{mn} = sum_{ls} (mn|ls) T_ls, K_{ml} = sum_{ns} (mn|ls) T_ns.
 * T, F DEVICE [nvec][nao][nao]. */
int rttda_fock(rttda_handle_t h, int32_t nvec, const double* T, double* F, void* stream);

/* rttda_fock for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same inputs, same result, but every workspace - interleaved densities and results,
 * the symmetry-split density pairs, the integral staging buffer - lives in ONE file-scope device array of
 * RTTDA_STATIC_SCRATCH_BYTES inside the library (csrc/fock_static.cu), and the call runs no cudaMalloc / cudaFree /
 * allocating library routine.  Every GPU that loads the library holds that array until the process exits.
 *   nvec   1..RTTDA_STATIC_MAX_NVEC;  T, F DEVICE [nvec][nao][nao] as for rttda_fock, must not alias
 *   EINVAL (with the byte counts in rttda_last_error) when 4 * nao^2 * nvt * 8 bytes + the handle's staging buffer
 *          (RTTDA_INFO_ERI_BUF_BYTES) exceed the array: about 250 basis functions with s/p shells; use rttda_fock beyond
 *   All calls on one device share the array and it keeps the last call's contents (the call clears what must start at
 *   zero): calls that overlap on the GPU - two streams, or two handles on one device - RACE; serialise them.  The
 *   segments run one after the other on `stream` (no lanes), so small molecules are slower here than through rttda_fock.
 *   The first call on a device resolves the array's device address (cudaGetSymbolAddress) and must not be captured. */
#define RTTDA_STATIC_SCRATCH_BYTES 134217728
#define RTTDA_STATIC_MAX_NVEC 8
int rttda_fock_static(rttda_handle_t h, int32_t nvec, const double* T, double* F, void* stream);

/* Fixed-step RK4 (R7) on i dC/dt = H(t) C for ntraj independent trajectories sharing every ERI pass.
 *   C      DEVICE in/out [ntraj][2][1 + nocc*nvirt]: plane 0 = q (Re), plane 1 = p (Im); element 0 = KS
 *          ground state
 *   fields host [ntraj]
 *   log    DEVICE or NULL, [nsteps][ntraj][3]: |C|^2, Re R, Im R after each step, R relative to the state
 *          at t_start (after the kick, if any)
 * Re-entrant in time: call again with t_start += nsteps*dt to continue; set RTTDA_FIELD_CONTINUE in the field
 * records of the continued call, otherwise a DELTA field kicks again and R(t) restarts from the state at t_start.
 * (The state C is the whole checkpoint; the reference state of R(t) lives in the handle until the next fresh call.) */
int rttda_propagate(rttda_handle_t h, int32_t ntraj, double* C, const rttda_field_t* fields,
                    double t_start, double dt, int32_t nsteps, double* log, void* stream);

/* The paper's own propagator (NEXT-1 of DESIGN.md): second-order symplectic split operator, P:126-130, 2 sigma
 * builds per step.  The text names it without formulas; reading R22 = Stoermer-Verlet on (q', p') = (H p, -H q):
 *   p_half = p_n - dt/2 H(t_n) q_n;  q_{n+1} = q_n + dt H(t_n + dt/2) p_half;  p_{n+1} = p_half - dt/2 H(t_{n+1}) q_{n+1},
 * H(t_{n+1}) q_{n+1} being reused by the next step.  Arguments, layout, kick (R8), log and re-entrancy as
 * rttda_propagate (a continued call recomputes H(t_start) q once). */
int rttda_propagate_sso(rttda_handle_t h, int32_t ntraj, double* C, const rttda_field_t* fields,
                        double t_start, double dt, int32_t nsteps, double* log, void* stream);

/* Same with HOST buffers for C and log (copies inside, stream synchronised on return). */
int rttda_propagate_host(rttda_handle_t h, int32_t ntraj, double* C, const rttda_field_t* fields,
                         double t_start, double dt, int32_t nsteps, double* log, void* stream);

/* Counters and timings.  Keys: */
#define RTTDA_INFO_NPAIRS_TOTAL      0   /* unique shell pairs a >= b */
#define RTTDA_INFO_NPAIRS_KEPT       1   /* pairs with Q_ab Q_max >= tau */
#define RTTDA_INFO_NQUARTETS         2   /* unique shell quartets with Q_ab Q_cd >= tau (R14) */
#define RTTDA_INFO_NPRIM_QUARTETS    3   /* primitive quartets inside those */
#define RTTDA_INFO_NQUARTETS_EVAL    4   /* contracted quartet evaluations the kernels perform per ERI pass */
#define RTTDA_INFO_NPRIM_EVAL        5   /* primitive quartets evaluated by the LAST ERI build, counted on the device (after
                                            primitive screening: a primitive quartet (kb, kk) of a shell quartet is
                                            evaluated iff q_kb Q_ket >= tau_p and q_kk Q_bra >= tau_p, tau_p = min(1e-3 tau, 1e-15), q_k the
                                            primitive pair's own Schwarz bound); synchronises the device */
#define RTTDA_INFO_FLOPS_EVAL        6   /* FP64 flop model of one ERI pass, evaluation part: on the primitive quartets
                                            actually evaluated (RTTDA_INFO_NPRIM_EVAL) */
#define RTTDA_INFO_FLOPS_DIGEST_PER_VEC 7 /* FP64 flop model, digestion per density */
#define RTTDA_INFO_JK_LAUNCHES       8   /* kernel launches of one ERI pass */
#define RTTDA_INFO_KERNEL_LAUNCHES   9   /* kernels launched by this handle so far (all entry points) */
#define RTTDA_INFO_CREATE_MS        10   /* wall time of rttda_create */
#define RTTDA_INFO_QMAX             11   /* largest Schwarz bound */
#define RTTDA_INFO_NVEC_CHUNK       12   /* 0: every ERI pass serves all densities of the call */
#define RTTDA_INFO_ERI_BUF_BYTES    13   /* HBM staging buffer between ERI evaluation and J/K digestion */
#define RTTDA_INFO_ERI_ALL_BYTES    14   /* bytes of ALL contracted integrals of one pass (the in-core store) */
int rttda_get_info(rttda_handle_t h, int32_t key, double* out);

/* TI-TDA eigenvalues through the same sigma builds (NEXT-3 of DESIGN.md): m steps of the symmetric Lanczos process on
 * the singles block A (A X = omega X, eq. 2), one sigma vector per step, full reorthogonalisation.
 *   v0 DEVICE [nocc*nvirt] start vector (any norm), alpha, beta HOST [m], V DEVICE [m+1][nocc*nvirt] (the Lanczos
 *   vectors; must not alias v0).  The Ritz values are the eigenvalues of tridiag(alpha, beta[0..m-2]); the caller
 *   diagonalises that small matrix.  Synchronises `stream` every step (alpha_j, beta_j are read back). */
int rttda_lanczos(rttda_handle_t h, int32_t m, const double* v0, double* alpha, double* beta, double* V, void* stream);

/* TI-TDA eigenpairs (NEXT-3 of DESIGN.md): the k lowest solutions of A X = omega X (eq. 2; the reference method
 * the paper compares its spectra with, Table 1) by block Davidson on the singles block: each iteration applies
 * A to a block of up to max(nblock, k) new directions in ONE multi-vector sigma build; start vectors are unit vectors on
 * the smallest eps_a - eps_i, the preconditioner is 1 / (theta - (eps_a - eps_i)).
 *   omega HOST [k] ascending, X DEVICE [k][nocc*nvirt] orthonormal eigenvectors, resid HOST [k] or NULL: |A x - omega x|_2,
 *   niter / nsigma (may be NULL): iterations and sigma vectors built.  Converged when every residual norm <= tol;
 *   RTTDA_ENOCONV after maxiter iterations (outputs then hold the current Ritz pairs).  Synchronises `stream`. */
int rttda_eigs(rttda_handle_t h, int32_t k, int32_t nblock, double tol, int32_t maxiter, double* omega, double* X,
               double* resid, int32_t* niter, int32_t* nsigma, void* stream);

/* Populations of stationary states (NEXT-2 of DESIGN.md): P[t][i] = |X_i^dagger C_t|^2, eq. 22, the projection
 * of every trajectory's vector onto supplied stationary states (e.g. TI-TDA eigenvectors; the ground state is e_0).
 *   C  DEVICE [ntraj][2][1 + nocc*nvirt] (layout of rttda_propagate), Xs DEVICE [nstates][1 + nocc*nvirt] real,
 *   P  DEVICE [ntraj][nstates].  Enqueued on `stream`. */
int rttda_populations(rttda_handle_t h, int32_t ntraj, const double* C, int32_t nstates, const double* Xs, double* P,
                      void* stream);

/* Absorption spectrum from the time-correlation function (NEXT-2 of DESIGN.md): eq. 21 R(omega) ~ omega F[R(t)]
 * with the recipe of P:212 (mirroring R(-t) = R(t)^*, Hann window over the 2n+1 mirrored points, `pad` zeros; the
 * paper pads 50,000), and the angular average of eq. 23 over the ntraj trajectories.
 *   log  DEVICE [n][ntraj][3], the log rttda_propagate wrote (entries 1, 2 of a row = Re, Im R((k+1) dt)); may be
 *        NULL if n == 0.  R0 HOST [ntraj][2] = R(0) of each trajectory (1 + 0i for a normalised start).
 *   omega DEVICE [nout], intensity DEVICE [ntraj + 1][nout] with nout = (2n + 1 + pad) / 2 (anything else is
 *        RTTDA_EINVAL): omega[i] = 2 pi (i+1) / ((2n+1+pad) dt); row t < ntraj = omega |F_t|, row ntraj = their mean.
 *   No normalisation to the highest peak (P:214 does that for plotting).  The transform is a direct DFT evaluated on
 *   the device.  Needs no handle.  Enqueued on `stream`. */
int rttda_spectrum(int32_t ntraj, int32_t n, const double* R0, const double* log, double dt, int32_t pad, int32_t nout,
                   double* omega, double* intensity, void* stream);

/* Options.  RTTDA_OPT_INCORE (value != 0 switches it on; default off): keep the contracted integrals of all
 * segments resident in HBM (RTTDA_INFO_ERI_ALL_BYTES: 61 GB for the 1280-AO molecule at tau = 1e-12) so that, after
 * the first ERI pass of the handle, later passes skip the evaluation and only digest.  This is NOT the paper's direct
 * method (P:130 re-evaluates every integral in every sigma build; that is the default and what bench.py reports as
 * `value`); it is offered because 180 GB of HBM3e can hold what the paper's GPUs could not.  RTTDA_ENOMEM if the
 * store does not fit: the handle then stays in direct mode. */
#define RTTDA_OPT_INCORE 1
/* RTTDA_OPT_GRAPH (value != 0 on): rttda_propagate captures ONE RK4 step (4 sigma builds, field coupling, stage
 * combination, observables; E(t) and the step counter live in device memory) in a CUDA graph and replays it nsteps times.
 * Default: on for small molecules (whose ERI pass is a few hundred short kernels), off for large ones.  While it is on
 * the per-pass event timings of rttda_jk_time / rttda_last_timings are not recorded by rttda_propagate. */
#define RTTDA_OPT_GRAPH 2
/* Range-separated exchange (NEXT-4 of DESIGN.md; the paper's functional is CAM-B3LYP):
 *   A_{ia,jb} = d_ij d_ab (eps_a - eps_i) + 2 (ia|jb) - c_x (ij|ab) - c_x^LR (ij| erf(omega r12)/r12 |ab)
 * RTTDA_OPT_CX_LR sets c_x^LR (default 0), RTTDA_OPT_RS_OMEGA sets omega in 1/bohr (default 0 = off).  When both are
 * non-zero every sigma build runs a second ERI pass over the same screened quartets with the integrals of the
 * attenuated operator (1/r12 with alpha -> alpha omega^2 / (alpha + omega^2)), digested into the exchange part only.
 * (CAM-B3LYP's exchange kernel is c_x = 0.19, c_x^LR = 0.46, omega = 0.33; its f_xc grid term stays out of scope.) */
#define RTTDA_OPT_CX_LR 3
#define RTTDA_OPT_RS_OMEGA 4
int rttda_set_option(rttda_handle_t h, int32_t option, double value);

/* Time the last rttda_sigma/rttda_fock call spent in the J/K kernels, from CUDA events recorded on its
 * stream (synchronises those events).  ms_out[0] = J/K build, [1] = MO->AO GEMMs, [2] = AO->MO GEMMs. */
int rttda_last_timings(rttda_handle_t h, double* ms_out);

/* Device time spent in the J/K builds (steps a3-a4) of every rttda_sigma / rttda_fock / rttda_propagate call
 * since the previous query: *sum_ms = total of the CUDA-event intervals recorded on the callers' streams
 * around each ERI pass, *count = number of passes.  Synchronises on those events and resets the log (which
 * holds at most 32768 passes; later ones are not recorded). */
int rttda_jk_time(rttda_handle_t h, double* sum_ms, double* count);

/* Timing instrumentation: runs ONE extra ERI pass (steps a3-a4) on the densities left by the last rttda_sigma /
 * rttda_fock call of the same nvec, with the evaluation and the digestion of every segment (bra pair class x ket pair
 * class) timed by CUDA events, serialised on `stream` (no overlap: the sum exceeds the time of a normal pass).
 *   rows HOST [cap][16]: segment, bra class id, ket class id, la, lb, lc, ld, bra primitive pairs, ket primitive
 *   pairs, quartets evaluated, 32-ket batches, evaluation ms, digestion ms, evaluation blocks, digestion launches, 0.
 *   *nrows = rows written.  Synchronises.  The Fock workspace of the handle is overwritten. */
int rttda_profile_pass(rttda_handle_t h, int32_t nvec, double* rows, int32_t cap, int32_t* nrows, void* stream);

/* The FP64 tensor-core (DMMA) GEMM behind the MO<->AO transforms and the field coupling (steps a1, a5, a6; the paper
 * uses cuBLAS for them), exposed for unit tests and callers:
 *   C_b(m,n) = alpha * sum_k A_b(m,k) B_b(k,n) + beta * C_b(m,n),  b < batch, element strides in doubles:
 *   A_b(m,k) = A[b*sabatch + m*sam + k*sak], B_b(k,n) = B[b*sbbatch + k*sbk + n*sbn], C likewise.  All DEVICE.
 *   beta == 0 does not read C.  K == 0 gives C = beta * C.  Enqueued on `stream`. */
int rttda_gemm_f64(int32_t M, int32_t N, int32_t K, int32_t batch, double alpha, const double* A, int64_t sam, int64_t sak,
                   int64_t sabatch, const double* B, int64_t sbk, int64_t sbn, int64_t sbbatch, double beta, double* C,
                   int64_t scm, int64_t scn, int64_t scbatch, void* stream);

/* Sustained FP64 FMA throughput of the device (TFLOP/s) from a dependent-chain DFMA kernel run for about
 * `seconds`; the roofline denominator of the ALU-bound J/K kernels. */
int rttda_fp64_peak(double seconds, double* tflops_out, void* stream);

const char* rttda_last_error(void);
const char* rttda_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RTTDA_H */
