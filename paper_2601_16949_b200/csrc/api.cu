// C-ABI entry points (include/rttda.h).  Argument checking and marshalling only; every step of the path
// runs in the kernels of this library.
#include <chrono>
#include <cstring>
#include "common.cuh"

namespace rttda {

static thread_local std::string g_err;
void set_error(const std::string& msg) { g_err = msg; }

int create_impl(Handle* h, const rttda_basis_t* basis, const double* C_occ, const double* C_virt,
                const double* eps, cudaStream_t st);
int overlap_host(const rttda_basis_t* basis, int nao, double* S, double* D);

// [nvec][N][N] <-> [N][N][nvt] (nvt >= nvec slots per element; the padding slots are written as zeros)
__global__ void interleave_kernel(long long nn, int nvec, int nvt, const double* __restrict__ in,
                                  double* __restrict__ out, int to_interleaved)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (to_interleaved) {
        if (i >= nn * nvt) return;
        const long long e = i / nvt; const int v = (int)(i % nvt);
        out[i] = v < nvec ? in[(long long)v * nn + e] : 0.0;
    } else {
        if (i >= nn * nvec) return;
        const int v = (int)(i / nn); const long long e = i % nn;
        out[i] = in[e * nvt + v];
    }
}

// dependent DFMA chains: 8 independent accumulators per thread, 2 flops per FMA
__global__ void fp64_peak_kernel(double* out, int iters, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

}  // namespace rttda

using namespace rttda;

// A handle is bound to the device current at rttda_create: every entry point makes that device current.
#define RT_DEVICE(h) RT_CUDA(cudaSetDevice((h)->device))

extern "C" {

const char* rttda_last_error(void) { return g_err.c_str(); }
const char* rttda_version(void) { return "rttda-b200 0.1 (sm_100a)"; }

int rttda_overlap(const rttda_basis_t* basis, int32_t nao, double* S)
{
    RT_CHECK(S != nullptr, "rttda_overlap: NULL output");
    return overlap_host(basis, nao, S, nullptr);
}

int rttda_dipole_ao(const rttda_basis_t* basis, int32_t nao, double* D)
{
    RT_CHECK(D != nullptr, "rttda_dipole_ao: NULL output");
    return overlap_host(basis, nao, nullptr, D);
}

int rttda_create(rttda_handle_t* out, const rttda_basis_t* basis, int32_t nao, int32_t nocc, int32_t nvirt,
                 const double* C_occ, const double* C_virt, const double* eps, double cx, double schwarz_tau,
                 void* stream)
{
    RT_CHECK(out && basis && C_occ && C_virt && eps, "rttda_create: NULL pointer");
    RT_CHECK(nao > 0 && nocc > 0 && nvirt > 0 && nocc + nvirt == nao, "rttda_create: need nocc + nvirt == nao > 0");
    RT_CHECK(schwarz_tau >= 0.0, "rttda_create: negative Schwarz threshold");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        set_error(std::string("rttda_create: no CUDA device (") + cudaGetErrorString(e) + "); there is no CPU fallback");
        return RTTDA_ECUDA;
    }
    Handle* h = new (std::nothrow) Handle();
    if (!h) { set_error("rttda_create: out of host memory"); return RTTDA_ENOMEM; }
    if (cudaGetDevice(&h->device) != cudaSuccess) { delete h; set_error("rttda_create: cudaGetDevice failed"); return RTTDA_ECUDA; }
    h->nao = nao; h->nocc = nocc; h->nvirt = nvirt; h->ncsf = nocc * nvirt;
    h->cx = cx; h->tau = schwarz_tau;
    const int r = create_impl(h, basis, C_occ, C_virt, eps, (cudaStream_t)stream);
    if (r != RTTDA_OK) { rttda_destroy((rttda_handle_t)h); return r; }
    *out = (rttda_handle_t)h;
    return RTTDA_OK;
}

int rttda_destroy(rttda_handle_t hh)
{
    Handle* h = (Handle*)hh;
    if (!h) return RTTDA_OK;
    cudaSetDevice(h->device);
    cudaDeviceSynchronize();
    for (void* p : h->dev_allocs) cudaFree(p);
    for (double* p : {h->wsY, h->wsT, h->wsF, h->wsZ, h->wsP, h->prop_ws, h->eri_all}) if (p) cudaFree(p);
    for (int l = 0; l < Handle::MAXLANES; ++l) {
        if (h->eri_buf[l]) cudaFree(h->eri_buf[l]);
        if (h->lane_st[l]) cudaStreamDestroy(h->lane_st[l]);
        if (h->lane_ev[l]) cudaEventDestroy(h->lane_ev[l]);
    }
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->step_graph) cudaGraphExecDestroy(h->step_graph);
    if (h->d_ctl) cudaFree(h->d_ctl);
    if (h->graph_st) cudaStreamDestroy(h->graph_st);
    if (h->graph_ev) cudaEventDestroy(h->graph_ev);
    for (auto& e : h->ev) if (e) cudaEventDestroy(e);
    for (auto& e : h->jk_ev) cudaEventDestroy(e);
    delete h;
    return RTTDA_OK;
}

int rttda_sigma(rttda_handle_t hh, int32_t nvec, const double* X, double* sigma, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && X && sigma, "rttda_sigma: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(nvec >= 1, "rttda_sigma: nvec < 1");
    RT_CHECK(X != sigma, "rttda_sigma: X and sigma must not alias");
    return sigma_impl(h, nvec, X, h->ncsf, sigma, h->ncsf, (cudaStream_t)stream);
}

int rttda_sigma_host(rttda_handle_t hh, int32_t nvec, const double* X, double* sigma, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && X && sigma, "rttda_sigma_host: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(nvec >= 1, "rttda_sigma_host: nvec < 1");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)nvec * h->ncsf;
    RT_TRY(ensure_ws(h, &h->wsZ, &h->wsZ_n, 2 * n));
    RT_CUDA(cudaMemcpyAsync(h->wsZ, X, n * sizeof(double), cudaMemcpyHostToDevice, st));
    RT_TRY(sigma_impl(h, nvec, h->wsZ, h->ncsf, h->wsZ + n, h->ncsf, st));
    RT_CUDA(cudaMemcpyAsync(sigma, h->wsZ + n, n * sizeof(double), cudaMemcpyDeviceToHost, st));
    RT_CUDA(cudaStreamSynchronize(st));
    return RTTDA_OK;
}

int rttda_fock(rttda_handle_t hh, int32_t nvec, const double* T, double* F, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && T && F, "rttda_fock: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(nvec >= 1, "rttda_fock: nvec < 1");
    cudaStream_t st = (cudaStream_t)stream;
    const long long nn = (long long)h->nao * h->nao;
    const int nvt = padded_nvec(nvec);
    RT_TRY(ensure_ws(h, &h->wsT, &h->wsT_n, (size_t)nvt * nn));
    RT_TRY(ensure_ws(h, &h->wsF, &h->wsF_n, (size_t)nvt * nn));
    RT_CUDA(cudaEventRecord(h->ev[0], st));
    interleave_kernel<<<(unsigned)((nn * nvt + 255) / 256), 256, 0, st>>>(nn, nvec, nvt, T, h->wsT, 1);
    RT_CUDA(cudaGetLastError());
    RT_CUDA(cudaEventRecord(h->ev[1], st));
    RT_TRY(jk_mark(h, st));
    RT_CUDA(cudaMemsetAsync(h->wsF, 0, (size_t)nvt * nn * sizeof(double), st));
    RT_TRY(jk_build(h, nvt, (nvec + 1) & ~1, h->wsT, h->wsF, st));
    RT_TRY(jk_mark(h, st));
    RT_CUDA(cudaEventRecord(h->ev[2], st));
    interleave_kernel<<<(unsigned)((nn * nvec + 255) / 256), 256, 0, st>>>(nn, nvec, nvt, h->wsF, F, 0);
    RT_CUDA(cudaGetLastError());
    RT_CUDA(cudaEventRecord(h->ev[3], st));
    h->ev_valid = true;
    h->kernel_launches += 2;
    return RTTDA_OK;
}

int rttda_propagate(rttda_handle_t hh, int32_t ntraj, double* C, const rttda_field_t* fields, double t_start,
                    double dt, int32_t nsteps, double* log, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && C && fields, "rttda_propagate: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(ntraj >= 1 && ntraj <= 8, "rttda_propagate: ntraj must be in 1..8");
    RT_CHECK(nsteps >= 0, "rttda_propagate: negative step count");
    for (int t = 0; t < ntraj; ++t)
        RT_CHECK(fields[t].type >= RTTDA_NONE && fields[t].type <= RTTDA_SIN2, "rttda_propagate: bad pulse type");
    return propagate_impl(h, ntraj, C, fields, t_start, dt, nsteps, log, (cudaStream_t)stream);
}

int rttda_propagate_sso(rttda_handle_t hh, int32_t ntraj, double* C, const rttda_field_t* fields, double t_start,
                        double dt, int32_t nsteps, double* log, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && C && fields, "rttda_propagate_sso: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(ntraj >= 1 && ntraj <= 8, "rttda_propagate_sso: ntraj must be in 1..8");
    RT_CHECK(nsteps >= 0, "rttda_propagate_sso: negative step count");
    for (int t = 0; t < ntraj; ++t)
        RT_CHECK(fields[t].type >= RTTDA_NONE && fields[t].type <= RTTDA_SIN2, "rttda_propagate_sso: bad pulse type");
    return propagate_sso_impl(h, ntraj, C, fields, t_start, dt, nsteps, log, (cudaStream_t)stream);
}

int rttda_propagate_host(rttda_handle_t hh, int32_t ntraj, double* C, const rttda_field_t* fields,
                         double t_start, double dt, int32_t nsteps, double* log, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && C && fields, "rttda_propagate_host: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(ntraj >= 1 && ntraj <= 8 && nsteps >= 0, "rttda_propagate_host: bad ntraj / nsteps");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t ns = (size_t)ntraj * 2 * ((size_t)h->ncsf + 1), nl = (size_t)nsteps * ntraj * 3;
    RT_TRY(ensure_ws(h, &h->wsZ, &h->wsZ_n, ns + nl));
    RT_CUDA(cudaMemcpyAsync(h->wsZ, C, ns * sizeof(double), cudaMemcpyHostToDevice, st));
    RT_TRY(rttda_propagate(hh, ntraj, h->wsZ, fields, t_start, dt, nsteps, log ? h->wsZ + ns : nullptr, stream));
    RT_CUDA(cudaMemcpyAsync(C, h->wsZ, ns * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (log && nl) RT_CUDA(cudaMemcpyAsync(log, h->wsZ + ns, nl * sizeof(double), cudaMemcpyDeviceToHost, st));
    RT_CUDA(cudaStreamSynchronize(st));
    return RTTDA_OK;
}

int rttda_lanczos(rttda_handle_t hh, int32_t m, const double* v0, double* alpha, double* beta, double* V, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && v0 && alpha && beta && V, "rttda_lanczos: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(m >= 1 && m < h->ncsf, "rttda_lanczos: need 1 <= m < nocc*nvirt");
    RT_CHECK(v0 < V || v0 >= V + (size_t)(m + 1) * h->ncsf, "rttda_lanczos: v0 must not alias V");
    return lanczos_impl(h, m, v0, alpha, beta, V, (cudaStream_t)stream);
}

int rttda_eigs(rttda_handle_t hh, int32_t k, int32_t nblock, double tol, int32_t maxiter, double* omega, double* X,
               double* resid, int32_t* niter, int32_t* nsigma, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && omega && X, "rttda_eigs: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(k >= 1 && k <= h->ncsf && nblock >= 1, "rttda_eigs: need 1 <= k <= nocc*nvirt and nblock >= 1");
    RT_CHECK(tol > 0.0 && maxiter >= 1, "rttda_eigs: need tol > 0 and maxiter >= 1");
    return eigs_impl(h, k, nblock, tol, maxiter, omega, X, resid, niter, nsigma, (cudaStream_t)stream);
}

int rttda_populations(rttda_handle_t hh, int32_t ntraj, const double* C, int32_t nstates, const double* Xs, double* P,
                      void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && C && Xs && P, "rttda_populations: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(ntraj >= 1 && nstates >= 1, "rttda_populations: ntraj and nstates must be positive");
    return populations_impl(h, ntraj, C, nstates, Xs, P, (cudaStream_t)stream);
}

int rttda_spectrum(int32_t ntraj, int32_t n, const double* R0, const double* log, double dt, int32_t pad, int32_t nout,
                   double* omega, double* intensity, void* stream)
{
    RT_CHECK(ntraj >= 1 && n >= 0 && pad >= 0 && dt > 0.0, "rttda_spectrum: need ntraj >= 1, n >= 0, pad >= 0, dt > 0");
    const long long npad = 2LL * n + 1 + pad;
    RT_CHECK(npad < (1LL << 31), "rttda_spectrum: 2n + 1 + pad must be below 2^31");
    RT_CHECK((long long)nout == npad / 2, "rttda_spectrum: nout must be (2n + 1 + pad) / 2");
    if (nout == 0) return RTTDA_OK;                         // a single sample without padding has no frequency grid
    RT_CHECK(R0 && omega && intensity && (log || n == 0), "rttda_spectrum: NULL pointer");
    return spectrum_impl(ntraj, n, R0, log, dt, pad, nout, omega, intensity, (cudaStream_t)stream);
}

int rttda_set_option(rttda_handle_t hh, int32_t option, double value)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h != nullptr, "rttda_set_option: NULL handle");
    RT_DEVICE(h);
    RT_CHECK(option == RTTDA_OPT_INCORE || option == RTTDA_OPT_GRAPH || option == RTTDA_OPT_CX_LR || option == RTTDA_OPT_RS_OMEGA,
             "rttda_set_option: unknown option");
    const bool on = value != 0.0;
    if (option == RTTDA_OPT_GRAPH) { h->use_graph = on; return RTTDA_OK; }
    if (option == RTTDA_OPT_CX_LR || option == RTTDA_OPT_RS_OMEGA) {
        RT_CHECK(option == RTTDA_OPT_CX_LR || value >= 0.0, "rttda_set_option: negative range-separation parameter");
        (option == RTTDA_OPT_CX_LR ? h->cx_lr : h->rs_omega) = value;
        if (h->step_graph) { cudaGraphExecDestroy(h->step_graph); h->step_graph = nullptr; }   // the captured step has one pass structure
        return RTTDA_OK;
    }
    if (on && !h->incore) {
        const int r = ensure_ws(h, &h->eri_all, &h->eri_all_n, h->eri_all_need);
        if (r != RTTDA_OK) return r;                       // not enough HBM: the handle stays in direct mode
    }
    if (!on && h->eri_all) { cudaDeviceSynchronize(); cudaFree(h->eri_all); h->eri_all = nullptr; h->eri_all_n = 0; }
    h->incore = on;
    h->incore_valid = false;
    return RTTDA_OK;
}

int rttda_get_info(rttda_handle_t hh, int32_t key, double* out)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && out, "rttda_get_info: NULL pointer");
    RT_CHECK(key >= 0 && key < 16, "rttda_get_info: unknown key");
    *out = (key == RTTDA_INFO_KERNEL_LAUNCHES) ? (double)h->kernel_launches : h->info[key];
    if (key == RTTDA_INFO_NPRIM_EVAL || key == RTTDA_INFO_FLOPS_EVAL) {
        // counted by the evaluation kernels of the last ERI build (all its passes); before the first build the
        // host-side count of the stored primitive pairs stands in (an upper bound)
        RT_DEVICE(h);
        unsigned long long c[8];
        RT_CUDA(cudaDeviceSynchronize());
        RT_CUDA(cudaMemcpy(c, h->d_primcount, sizeof c, cudaMemcpyDeviceToHost));
        double n = 0.0, fl = 0.0;
        for (int L = 0; L <= 4; ++L) { n += (double)c[L]; fl += (double)c[L] * flops_prim_L(L); }
        n += (double)c[5]; fl += (double)c[6];              // classes with a d shell (eri_generic.cu)
        if (n > 0.0) *out = (key == RTTDA_INFO_NPRIM_EVAL) ? n : fl;
    }
    return RTTDA_OK;
}

int rttda_last_timings(rttda_handle_t hh, double* ms)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && ms, "rttda_last_timings: NULL pointer");
    RT_DEVICE(h);
    RT_CHECK(h->ev_valid, "rttda_last_timings: no sigma/fock call yet");
    RT_CUDA(cudaEventSynchronize(h->ev[3]));
    float a = 0, b = 0, c = 0;
    RT_CUDA(cudaEventElapsedTime(&a, h->ev[1], h->ev[2]));
    RT_CUDA(cudaEventElapsedTime(&b, h->ev[0], h->ev[1]));
    RT_CUDA(cudaEventElapsedTime(&c, h->ev[2], h->ev[3]));
    ms[0] = a; ms[1] = b; ms[2] = c;
    return RTTDA_OK;
}

int rttda_jk_time(rttda_handle_t hh, double* sum_ms, double* count)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && sum_ms && count, "rttda_jk_time: NULL pointer");
    RT_DEVICE(h);
    double tot = 0.0;
    const size_t n = h->jk_ev_used / 2;
    for (size_t i = 0; i < n; ++i) {
        RT_CUDA(cudaEventSynchronize(h->jk_ev[2 * i + 1]));
        float ms = 0;
        RT_CUDA(cudaEventElapsedTime(&ms, h->jk_ev[2 * i], h->jk_ev[2 * i + 1]));
        tot += ms;
    }
    *sum_ms = tot; *count = (double)n;
    h->jk_ev_used = 0;
    return RTTDA_OK;
}

int rttda_profile_pass(rttda_handle_t hh, int32_t nvec, double* rows, int32_t cap, int32_t* nrows, void* stream)
{
    Handle* h = (Handle*)hh;
    RT_CHECK(h && rows && nrows && cap > 0, "rttda_profile_pass: bad arguments");
    RT_DEVICE(h);
    RT_CHECK(nvec >= 1, "rttda_profile_pass: nvec < 1");
    const int nvt = padded_nvec(nvec);
    const size_t nn = (size_t)h->nao * h->nao;
    RT_CHECK(h->wsT && h->wsT_n >= nn * nvt && h->wsF_n >= nn * nvt,
             "rttda_profile_pass: call rttda_sigma / rttda_fock with the same nvec first (its densities are reused)");
    cudaStream_t st = (cudaStream_t)stream;
    RT_CUDA(cudaMemsetAsync(h->wsF, 0, nn * nvt * sizeof(double), st));
    RT_CUDA(cudaMemsetAsync(h->d_primcount, 0, 8 * sizeof(unsigned long long), st));
    return jk_profile(h, nvt, (nvec + 1) & ~1, h->wsT, h->wsF, st, rows, cap, nrows);
}

int rttda_gemm_f64(int32_t M, int32_t N, int32_t K, int32_t batch, double alpha, const double* A, int64_t sam, int64_t sak,
                   int64_t sabatch, const double* B, int64_t sbk, int64_t sbn, int64_t sbbatch, double beta, double* C,
                   int64_t scm, int64_t scn, int64_t scbatch, void* stream)
{
    RT_CHECK(M >= 0 && N >= 0 && K >= 0 && batch >= 0, "rttda_gemm_f64: negative size");
    RT_CHECK(A && B && C, "rttda_gemm_f64: NULL pointer");
    GemmDesc g{};
    g.M = M; g.N = N; g.K = K; g.batch = batch; g.alpha = alpha; g.beta = beta;
    g.A = A; g.sam = sam; g.sak = sak; g.sabatch = sabatch;
    g.B = B; g.sbk = sbk; g.sbn = sbn; g.sbbatch = sbbatch;
    g.C = C; g.scm = scm; g.scn = scn; g.scbatch = scbatch;
    return gemm_f64(g, (cudaStream_t)stream);
}

int rttda_fp64_peak(double seconds, double* tflops, void* stream)
{
    RT_CHECK(tflops && seconds > 0.0, "rttda_fp64_peak: bad arguments");
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, nsm = 0;
    RT_CUDA(cudaGetDevice(&dev));
    RT_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = nsm * 8, threads = 256, iters = 4096;
    double* buf = nullptr;
    RT_CUDA(cudaMalloc((void**)&buf, (size_t)blocks * threads * sizeof(double)));
    cudaEvent_t e0, e1;
    RT_CUDA(cudaEventCreate(&e0));
    RT_CUDA(cudaEventCreate(&e1));
    fp64_peak_kernel<<<blocks, threads, 0, st>>>(buf, 64, 0.999999, 1e-9);   // warm-up
    RT_CUDA(cudaStreamSynchronize(st));
    const double flops_per_launch = (double)blocks * threads * iters * 16.0 * 8.0 * 2.0;
    double best = 0.0, elapsed = 0.0;
    while (elapsed < seconds) {
        RT_CUDA(cudaEventRecord(e0, st));
        fp64_peak_kernel<<<blocks, threads, 0, st>>>(buf, iters, 0.999999, 1e-9);
        RT_CUDA(cudaEventRecord(e1, st));
        RT_CUDA(cudaEventSynchronize(e1));
        float ms = 0;
        RT_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        elapsed += ms * 1e-3;
        best = flops_per_launch / (ms * 1e-3) * 1e-12;   // sustained: keep the LAST launch's rate
    }
    *tflops = best;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf);
    return RTTDA_OK;
}

}  // extern "C"
