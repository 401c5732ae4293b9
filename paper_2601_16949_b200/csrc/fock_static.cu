// rttda_fock_static: the AO-direct Fock build (steps a3-a4 of DESIGN.md, F = 2 J[T] - c_x K[T]) for callers that
// cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  rttda_fock takes its workspaces - interleaved densities and results, the {T+T^T, T-T^T} pairs, the
// integral staging buffer - from buffers the handle grows on demand with cudaMalloc; this variant takes them from ONE
// file-scope device array of fixed size instead and calls no cudaMalloc / cudaFree / allocating library routine.
//
// The array (RTTDA_STATIC_SCRATCH_BYTES = 128 MiB) is part of the library image: every GPU that loads librttda.so holds
// it until the process exits.  Every call on a device shares it, and it keeps the last call's contents: the result part
// is cleared at the start of each call, everything else is fully overwritten before it is read.  Two calls that overlap
// on the GPU (different streams, or different handles on one device) race on it - callers serialise them.
//
// In host code the array's NAME is a host-side stand-in, not a device address; the address comes from
// cudaGetSymbolAddress, asked once per device with that device current (first call on the device; that first call
// is not capturable - make one call before starting a capture).
#include "common.cuh"

namespace rttda {

namespace {

constexpr size_t STATIC_SCRATCH_DOUBLES = RTTDA_STATIC_SCRATCH_BYTES / sizeof(double);
static __device__ __align__(256) double g_static_scratch[STATIC_SCRATCH_DOUBLES];

constexpr int MAX_DEVICES = 64;
double* g_scratch_addr[MAX_DEVICES] = {nullptr};      // device address of g_static_scratch on each device

// T [nvec][N][N] -> Tq [N][N][nvt] (v fastest; padding slots zero) and PP [N][N][nvt] = {T + T^T, T - T^T}:
// the interleave and symmetry-split steps of rttda_fock (interleave_kernel + symsplit_kernel) in one pass,
// writing into the static scratch.
__global__ void interleave_split_static_kernel(int nao, int nvec, int nvt, const double* __restrict__ T,
                                               double* __restrict__ Tq, double2* __restrict__ PP)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nn = (long long)nao * nao;
    if (i >= nn * nvt) return;
    const int v = (int)(i % nvt);
    const long long e = i / nvt;
    const int mu = (int)(e / nao), nu = (int)(e % nao);
    const double a = v < nvec ? T[(long long)v * nn + e] : 0.0;
    const double b = v < nvec ? T[(long long)v * nn + (long long)nu * nao + mu] : 0.0;
    Tq[i] = a;
    PP[i] = make_double2(a + b, a - b);
}

// Fq [N][N][nvt] -> F [nvec][N][N]
__global__ void deinterleave_static_kernel(long long nn, int nvec, int nvt, const double* __restrict__ Fq,
                                           double* __restrict__ F)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nn * nvec) return;
    const int v = (int)(i / nn);
    const long long e = i % nn;
    F[i] = Fq[e * nvt + v];
}

inline size_t round_up_32(size_t n) { return (n + 31) & ~(size_t)31; }      // 256-byte aligned parts

int fock_static_impl(Handle* h, int nvec, const double* T, double* F, cudaStream_t st)
{
    RT_CHECK(nvec >= 1 && nvec <= RTTDA_STATIC_MAX_NVEC, "rttda_fock_static: nvec must be in 1..8");
    RT_CHECK(h->device >= 0 && h->device < MAX_DEVICES, "rttda_fock_static: device index out of range");
    const size_t nn = (size_t)h->nao * h->nao;
    const int nvt = padded_nvec(nvec);
    // parts of the scratch: Tq | Fq | PP | integral staging buffer of the largest segment
    const size_t n_t = round_up_32(nn * nvt), n_pp = round_up_32(2 * nn * nvt), n_buf = round_up_32(h->eri_buf_need);
    const size_t need = 2 * n_t + n_pp + n_buf;
    if (need > STATIC_SCRATCH_DOUBLES) {
        char msg[256];
        snprintf(msg, sizeof msg,
                 "rttda_fock_static: this molecule and nvec need %zu bytes of scratch (%zu of them for the integral staging "
                 "buffer), the static array holds %zu; use rttda_fock",
                 need * sizeof(double), n_buf * sizeof(double), (size_t)RTTDA_STATIC_SCRATCH_BYTES);
        set_error(msg);
        return RTTDA_EINVAL;
    }
    if (!g_scratch_addr[h->device]) {                // once per device, with that device current (RT_DEVICE in the caller)
        double* p = nullptr;
        RT_CUDA(cudaGetSymbolAddress((void**)&p, g_static_scratch));
        g_scratch_addr[h->device] = p;
    }
    double* Tq = g_scratch_addr[h->device];
    double* Fq = Tq + n_t;
    double* PP = Fq + n_t;
    double* buf = PP + n_pp;

    RT_CUDA(cudaMemsetAsync(Fq, 0, nn * nvt * sizeof(double), st));       // the result accumulates by atomic adds
    interleave_split_static_kernel<<<(unsigned)((nn * nvt + 255) / 256), 256, 0, st>>>(h->nao, nvec, nvt, T, Tq,
                                                                                       reinterpret_cast<double2*>(PP));
    RT_CUDA(cudaGetLastError());
    RT_CUDA(cudaMemsetAsync(h->d_primcount, 0, 8 * sizeof(unsigned long long), st));
    // The digestion kernels read the density pairs through the handle's workspace pointer: lend it the static part for
    // the launches enqueued here (kernel arguments are captured at launch), then give it back.
    double* const wsP_saved = h->wsP;
    h->wsP = PP;
    const bool lr = (h->cx_lr != 0.0 && h->rs_omega > 0.0);
    const int nvec2 = (nvec + 1) & ~1;
    int rc = RTTDA_OK;
    for (int pass = 0; pass < (lr ? 2 : 1) && rc == RTTDA_OK; ++pass) {
        // pass 0: 1/r12, Coulomb + c_x exchange; pass 1 (range-separated exchange): erf(omega r12)/r12, exchange only
        h->pass_w_extra = pass == 0 ? 0.0 : 36.0 / (h->rs_omega * h->rs_omega);
        h->pass_cx = pass == 0 ? h->cx : h->cx_lr;
        h->pass_do_j = (pass == 0);
        h->pass_do_k = true;
        for (const Segment& sg : h->segments) {      // one stream, one staging buffer: evaluate, digest, next segment
            if (sg.nitems == 0) continue;
            rc = eval_segment(h, sg, buf, st);
            if (rc == RTTDA_OK) rc = digest_segment(h, sg, buf, nvt, nvec2, Tq, Fq, st);
            if (rc != RTTDA_OK) break;
        }
    }
    h->wsP = wsP_saved;
    h->pass_w_extra = 0.0; h->pass_cx = h->cx; h->pass_do_j = h->pass_do_k = true;
    RT_TRY(rc);
    deinterleave_static_kernel<<<(unsigned)((nn * nvec + 255) / 256), 256, 0, st>>>((long long)nn, nvec, nvt, Fq, F);
    RT_CUDA(cudaGetLastError());
    h->kernel_launches += 2;
    return RTTDA_OK;
}

}  // namespace

}  // namespace rttda

extern "C" int rttda_fock_static(rttda_handle_t hh, int32_t nvec, const double* T, double* F, void* stream)
{
    using namespace rttda;
    Handle* h = (Handle*)hh;
    RT_CHECK(h && T && F, "rttda_fock_static: NULL pointer");
    RT_CUDA(cudaSetDevice(h->device));
    return fock_static_impl(h, nvec, T, F, (cudaStream_t)stream);
}
