// sigma = A X (steps a1-a5), field coupling (a6, eq. 16/19) and the RK4 propagator (a7, eq. 1, 12-15).
#include <cmath>
#include <vector>
#include "common.cuh"

namespace rttda {

int ensure_ws(Handle* h, double** p, size_t* cur, size_t need)
{
    if (*cur >= need) return RTTDA_OK;
    if (*p) cudaFree(*p);
    *p = nullptr; *cur = 0;
    cudaError_t e = cudaMalloc((void**)p, need * sizeof(double));
    if (e != cudaSuccess) { set_error(std::string("workspace cudaMalloc: ") + cudaGetErrorString(e)); return RTTDA_ENOMEM; }
    *cur = need;
    h->ws_epoch++;                               // pointers baked into a captured graph are stale now
    return RTTDA_OK;
}

// sigma[v][ia] = deps[ia] * X[v][ia]   (the diagonal term of eq. 3; the GEMM then accumulates onto it)
__global__ void diag_kernel(int ncsf, int nvec, const double* __restrict__ deps, const double* __restrict__ X,
                            long long ldx, double* __restrict__ S, long long lds)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)ncsf * nvec) return;
    const int v = (int)(i / ncsf), k = (int)(i % ncsf);
    S[v * lds + k] = deps[k] * X[v * ldx + k];
}

int jk_mark(Handle* h, cudaStream_t st)
{
    constexpr size_t CAP = 1 << 16;
    if (h->jk_ev_used >= CAP) return RTTDA_OK;
    if (h->jk_ev_used == h->jk_ev.size()) {
        cudaEvent_t e;
        RT_CUDA(cudaEventCreate(&e));
        h->jk_ev.push_back(e);
    }
    RT_CUDA(cudaEventRecord(h->jk_ev[h->jk_ev_used++], st));
    return RTTDA_OK;
}

// Every workspace a sigma build of nvec vectors needs (must not be grown while a stream is being captured)
int sigma_reserve(Handle* h, int nvec)
{
    const size_t N = h->nao, no = h->nocc;
    const int nvt = padded_nvec(nvec);
    RT_TRY(ensure_ws(h, &h->wsY, &h->wsY_n, (size_t)nvec * no * N));
    RT_TRY(ensure_ws(h, &h->wsT, &h->wsT_n, (size_t)nvt * N * N));
    RT_TRY(ensure_ws(h, &h->wsF, &h->wsF_n, (size_t)nvt * N * N));
    RT_TRY(ensure_ws(h, &h->wsP, &h->wsP_n, (size_t)2 * nvt * N * N));
    if (!h->incore) {
        for (int l = 0; l < h->nlanes; ++l) RT_TRY(ensure_ws(h, &h->eri_buf[l], &h->eri_buf_n[l], h->lane_need[l]));
        if (h->nlanes == 0)
            for (int b = 0; b < 2; ++b) RT_TRY(ensure_ws(h, &h->eri_buf[b], &h->eri_buf_n[b], h->eri_buf_need));
    }
    return RTTDA_OK;
}

int sigma_impl(Handle* h, int nvec, const double* X, long long ldx, double* sigma, long long lds,
               cudaStream_t st)
{
    const size_t N = h->nao, no = h->nocc, nv = h->nvirt;
    const int nvt = padded_nvec(nvec);          // density slots: 16, 32 or multiples of 64 bytes (sector aligned)
    const bool timed = !h->capturing;           // event timings cannot be taken inside a captured graph
    if (timed) RT_TRY(sigma_reserve(h, nvec));
    if (timed) RT_CUDA(cudaEventRecord(h->ev[0], st));
    if (nvt != nvec) RT_CUDA(cudaMemsetAsync(h->wsT, 0, (size_t)nvt * N * N * sizeof(double), st));
    // a1: Y_v = X_v C_v^T  [no][N];  T[mu][nu][v] = sum_j C_o[mu][j] Y_v[j][nu]
    GemmDesc g{};
    g.alpha = 1.0; g.beta = 0.0; g.batch = nvec;
    g.M = (int)no; g.N = (int)N; g.K = (int)nv;
    g.A = X; g.sam = nv; g.sak = 1; g.sabatch = ldx;
    g.B = h->C_virt; g.sbk = 1; g.sbn = nv; g.sbbatch = 0;
    g.C = h->wsY; g.scm = N; g.scn = 1; g.scbatch = no * N;
    RT_TRY(gemm_f64(g, st));
    g.M = (int)N; g.N = (int)N; g.K = (int)no;
    g.A = h->C_occ; g.sam = no; g.sak = 1; g.sabatch = 0;
    g.B = h->wsY; g.sbk = N; g.sbn = 1; g.sbbatch = no * N;
    g.C = h->wsT; g.scm = N * nvt; g.scn = nvt; g.scbatch = 1;
    RT_TRY(gemm_f64(g, st));
    if (timed) { RT_CUDA(cudaEventRecord(h->ev[1], st)); RT_TRY(jk_mark(h, st)); }
    // a3-a4: F = 2 J[T] - cx K[T], interleaved layout; one ERI pass serves all densities
    RT_CUDA(cudaMemsetAsync(h->wsF, 0, (size_t)nvt * N * N * sizeof(double), st));
    RT_TRY(jk_build(h, nvt, (nvec + 1) & ~1, h->wsT, h->wsF, st));
    if (timed) { RT_TRY(jk_mark(h, st)); RT_CUDA(cudaEventRecord(h->ev[2], st)); }
    // a5: Z_v = C_o^T F_v [no][N];  sigma_v = deps o X_v + Z_v C_v
    g.M = (int)no; g.N = (int)N; g.K = (int)N; g.batch = nvec;
    g.A = h->C_occ; g.sam = 1; g.sak = no; g.sabatch = 0;
    g.B = h->wsF; g.sbk = N * nvt; g.sbn = nvt; g.sbbatch = 1;
    g.C = h->wsY; g.scm = N; g.scn = 1; g.scbatch = no * N;
    RT_TRY(gemm_f64(g, st));
    const long long tot = (long long)h->ncsf * nvec;
    diag_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(h->ncsf, nvec, h->deps, X, ldx, sigma, lds);
    RT_CUDA(cudaGetLastError());
    g.M = (int)no; g.N = (int)nv; g.K = (int)N; g.beta = 1.0;
    g.A = h->wsY; g.sam = N; g.sak = 1; g.sabatch = no * N;
    g.B = h->C_virt; g.sbk = nv; g.sbn = 1; g.sbbatch = 0;
    g.C = sigma; g.scm = nv; g.scn = 1; g.scbatch = lds;
    RT_TRY(gemm_f64(g, st));
    if (timed) { RT_CUDA(cudaEventRecord(h->ev[3], st)); h->ev_valid = true; }
    h->kernel_launches += 5;
    return RTTDA_OK;
}

// ---------------------------------------------------------------------------------------------- field
static double field_value(const rttda_field_t& f, double t)
{
    switch (f.type) {
        case RTTDA_CW: return f.E0 * std::sin(f.omega * t);
        case RTTDA_TL: {
            const double s = t - f.t0;
            return f.E0 * std::exp(-s * s / (2.0 * f.sigma * f.sigma)) * std::sin(f.omega * s);
        }
        case RTTDA_CHIRP: {
            const double s = t - f.t0;
            return f.E0 * std::exp(-s * s / (2.0 * f.sigma * f.sigma)) * std::sin((f.omega + 0.5 * f.beta * s) * s);
        }
        case RTTDA_SIN2: {
            if (t < 0.0 || t > f.T_env) return 0.0;
            const double e = std::sin(M_PI * t / f.T_env);
            return f.E0 * e * e * std::sin(f.omega * t);
        }
        default: return 0.0;
    }
}

// out[i] = d0 in0[i] + d1 in1[i] + d2 in2[i]   (D_d = sum_k d_k D^k)
__global__ void combine3_kernel(long long n, const double* __restrict__ in, double d0, double d1, double d2,
                                double* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = d0 * in[i] + d1 * in[n + i] + d2 * in[2 * n + i];
}

struct FieldArgs {
    double E[8];        // E(t) (or kick area) per trajectory
    double D00[8];      // D_00 along the trajectory's polarisation
};

// One block per (trajectory, plane): element 0 and the elementwise part of E * M y (eq. 19a-c):
//   hy_0  (+)= E (D_00 y_0 + sqrt2 sum_ia D_ov[ia] Y[ia])
//   hy_ia  += E (sqrt2 D_ov[ia] y_0 + D_00 Y[ia])
// `assign0`: hy_0 is assigned (sigma never writes element 0), singles are always accumulated.
__global__ void __launch_bounds__(1024)
field_elem_kernel(int ncsf, const double* __restrict__ ys, double* __restrict__ hy,
                  const double* __restrict__ Dov /* [ntraj][ncsf] */, FieldArgs fa)
{
    const int b = blockIdx.x, traj = b >> 1;
    const long long n1 = (long long)ncsf + 1;
    const double* y = ys + b * n1;
    double* h = hy + b * n1;
    const double* d = Dov + (long long)traj * ncsf;
    const double E = fa.E[traj], D00 = fa.D00[traj], y0 = y[0];
    const double s2 = 1.41421356237309504880;
    double dot = 0.0;
    if (E != 0.0) {
        for (int i = threadIdx.x; i < ncsf; i += blockDim.x) {
            const double Y = y[1 + i], dv = d[i];
            dot = fma(dv, Y, dot);
            h[1 + i] += E * fma(s2 * dv, y0, D00 * Y);
        }
    }
    __shared__ double red[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = dot;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) h[0] = E * fma(D00, y0, s2 * v);
    }
}

// hy (+)= E_traj * M_d ys for all trajectories/planes.  Singles of hy must already hold A ys (or zeros).
static int apply_field(Handle* h, int ntraj, const double* ys, double* hy, const double* Dd_oo,
                       const double* Dd_vv, const double* Dd_ov, const FieldArgs& fa, cudaStream_t st)
{
    const size_t no = h->nocc, nv = h->nvirt, n1 = (size_t)h->ncsf + 1;
    field_elem_kernel<<<2 * ntraj, 1024, 0, st>>>(h->ncsf, ys, hy, Dd_ov, fa);
    RT_CUDA(cudaGetLastError());
    h->kernel_launches++;
    for (int t = 0; t < ntraj; ++t) {
        if (fa.E[t] == 0.0) continue;
        GemmDesc g{};
        g.batch = 2; g.beta = 1.0;
        // + E Y D_vv
        g.alpha = fa.E[t];
        g.M = (int)no; g.N = (int)nv; g.K = (int)nv;
        g.A = ys + (size_t)t * 2 * n1 + 1; g.sam = nv; g.sak = 1; g.sabatch = n1;
        g.B = Dd_vv + (size_t)t * nv * nv; g.sbk = nv; g.sbn = 1; g.sbbatch = 0;
        g.C = hy + (size_t)t * 2 * n1 + 1; g.scm = nv; g.scn = 1; g.scbatch = n1;
        RT_TRY(gemm_f64(g, st));
        // - E D_oo Y
        g.alpha = -fa.E[t];
        g.M = (int)no; g.N = (int)nv; g.K = (int)no;
        g.A = Dd_oo + (size_t)t * no * no; g.sam = no; g.sak = 1; g.sabatch = 0;
        g.B = ys + (size_t)t * 2 * n1 + 1; g.sbk = nv; g.sbn = 1; g.sbbatch = n1;
        RT_TRY(gemm_f64(g, st));
        h->kernel_launches += 2;
    }
    return RTTDA_OK;
}

// ---------------------------------------------------------------------------------------------- device-side stepping
// Control block of a graph-replayed run: pulse parameters, start time, step counter and log pointer live in device
// memory, so that the captured step holds no per-step host value.
struct PropCtl {
    double t_start, dt;
    double* log;                    // [nsteps][ntraj][3] or NULL
    int step, ntraj;
    rttda_field_t f[8];
    double E[8], mE[8], D00[8];     // E(t) of the current stage, its negative, D_00 along the polarisation
};

__device__ double field_value_dev(const rttda_field_t& f, double t)
{
    switch (f.type) {
        case RTTDA_CW: return f.E0 * sin(f.omega * t);
        case RTTDA_TL: {
            const double s = t - f.t0;
            return f.E0 * exp(-s * s / (2.0 * f.sigma * f.sigma)) * sin(f.omega * s);
        }
        case RTTDA_CHIRP: {
            const double s = t - f.t0;
            return f.E0 * exp(-s * s / (2.0 * f.sigma * f.sigma)) * sin((f.omega + 0.5 * f.beta * s) * s);
        }
        case RTTDA_SIN2: {
            if (t < 0.0 || t > f.T_env) return 0.0;
            const double e = sin(3.14159265358979323846 * t / f.T_env);
            return f.E0 * e * e * sin(f.omega * t);
        }
        default: return 0.0;
    }
}

// E(t_stage) of every trajectory, t_stage = t_start + (step + off) dt
__global__ void field_eval_kernel(PropCtl* c, double off)
{
    const int t = threadIdx.x;
    if (t >= c->ntraj) return;
    const double ts = c->t_start + ((double)c->step + off) * c->dt;
    const double E = field_value_dev(c->f[t], ts);
    c->E[t] = E;
    c->mE[t] = -E;
}

__global__ void step_advance_kernel(PropCtl* c) { c->step += 1; }

// field_elem_kernel with E and D_00 read from the control block
__global__ void __launch_bounds__(1024)
field_elem_dev_kernel(int ncsf, const double* __restrict__ ys, double* __restrict__ hy,
                      const double* __restrict__ Dov, const PropCtl* __restrict__ c)
{
    const int b = blockIdx.x, traj = b >> 1;
    const long long n1 = (long long)ncsf + 1;
    const double* y = ys + b * n1;
    double* h = hy + b * n1;
    const double* d = Dov + (long long)traj * ncsf;
    const double E = c->E[traj], D00 = c->D00[traj], y0 = y[0];
    const double s2 = 1.41421356237309504880;
    double dot = 0.0;
    for (int i = threadIdx.x; i < ncsf; i += blockDim.x) {
        const double Y = y[1 + i], dv = d[i];
        dot = fma(dv, Y, dot);
        h[1 + i] += E * fma(s2 * dv, y0, D00 * Y);
    }
    __shared__ double red[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = dot;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) h[0] = E * fma(D00, y0, s2 * v);
    }
}

// ---------------------------------------------------------------------------------------------- RK4
// k = -i H ys: (k_q, k_p) = (hy_p, -hy_q)  (eq. 14-15).  One fused pass per stage:
//   ksum  = (first ? 0 : ksum) + w k
//   ys    = y + c k                      (next stage input)       if !last
//   y     = y + (dt/6) ksum                                       if last
__global__ void rk4_stage_kernel(long long n1, int ntraj, const double* __restrict__ hy, double* __restrict__ y,
                                 double* __restrict__ ys, double* __restrict__ ksum, double w, double c,
                                 double dt6, int first, int last)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n1 * ntraj) return;
    const long long t = i / n1, e = i % n1;
    const long long iq = (2 * t) * n1 + e, ip = (2 * t + 1) * n1 + e;
    const double kq = hy[ip], kp = -hy[iq];
    double sq = w * kq, sp = w * kp;
    if (!first) { sq += ksum[iq]; sp += ksum[ip]; }
    if (last) {
        y[iq] = fma(dt6, sq, y[iq]);
        y[ip] = fma(dt6, sp, y[ip]);
    } else {
        ksum[iq] = sq; ksum[ip] = sp;
        ys[iq] = fma(c, kq, y[iq]);
        ys[ip] = fma(c, kp, y[ip]);
    }
}

// delta kick (R8): y <- y - i kappa M y, hy holds kappa M y:  q += hy_p, p -= hy_q
__global__ void kick_kernel(long long n1, int ntraj, const double* __restrict__ hy, double* __restrict__ y,
                            FieldArgs fa)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n1 * ntraj) return;
    const long long t = i / n1, e = i % n1;
    if (fa.E[t] == 0.0) return;
    const long long iq = (2 * t) * n1 + e, ip = (2 * t + 1) * n1 + e;
    y[iq] += hy[ip];
    y[ip] -= hy[iq];
}

// log[traj] = (|y|^2, Re <yref|y>, Im <yref|y>)   (eq. 20)
__global__ void __launch_bounds__(1024)
observe_kernel(long long n1, const double* __restrict__ y, const double* __restrict__ yref, double* __restrict__ out)
{
    const int t = blockIdx.x;
    const double *q = y + 2 * t * n1, *p = q + n1, *qr = yref + 2 * t * n1, *pr = qr + n1;
    double a = 0, b = 0, c = 0;
    for (long long i = threadIdx.x; i < n1; i += blockDim.x) {
        const double qi = q[i], pi = p[i], qri = qr[i], pri = pr[i];
        a = fma(qi, qi, fma(pi, pi, a));
        b = fma(qri, qi, fma(pri, pi, b));
        c = fma(qri, pi, fma(-pri, qi, c));
    }
    __shared__ double red[3][32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
        c += __shfl_xor_sync(0xffffffffu, c, o);
    }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = a; red[1][threadIdx.x >> 5] = b; red[2][threadIdx.x >> 5] = c; }
    __syncthreads();
    if (threadIdx.x < 32) {
        const int nw = blockDim.x >> 5;
        a = threadIdx.x < nw ? red[0][threadIdx.x] : 0.0;
        b = threadIdx.x < nw ? red[1][threadIdx.x] : 0.0;
        c = threadIdx.x < nw ? red[2][threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_xor_sync(0xffffffffu, a, o);
            b += __shfl_xor_sync(0xffffffffu, b, o);
            c += __shfl_xor_sync(0xffffffffu, c, o);
        }
        if (threadIdx.x == 0) { out[3 * t] = a; out[3 * t + 1] = b; out[3 * t + 2] = c; }
    }
}

// Common prologue of both propagators: workspace carving, D_d = sum_k d_k D^k per trajectory (recomputed only when the
// polarisations change), the linearised delta kick (R8) and the reference state of R(t).  A field record with
// RTTDA_FIELD_CONTINUE set marks a CONTINUED run: no kick, and R(t) stays relative to the reference state of the
// previous call on this handle (which must have had the same ntraj).
struct PropWs {
    double *ys, *hy, *ksum, *yref, *Dd_oo, *Dd_vv, *Dd_ov;
    FieldArgs fa;
    unsigned eg;
};

static int prop_prologue(Handle* h, int ntraj, double* y, const rttda_field_t* fields, PropWs& w, cudaStream_t st)
{
    const size_t no = h->nocc, nv = h->nvirt, ncsf = h->ncsf, n1 = ncsf + 1;
    const size_t nstate = (size_t)ntraj * 2 * n1;
    const size_t need = 4 * nstate + (size_t)ntraj * (no * no + nv * nv + no * nv);
    if (h->prop_ws_n < need) { h->dd_valid = false; h->yref_ntraj = 0; }
    RT_TRY(ensure_ws(h, &h->prop_ws, &h->prop_ws_n, need));
    w.ys = h->prop_ws;
    w.hy = w.ys + nstate;
    w.ksum = w.hy + nstate;
    w.yref = w.ksum + nstate;
    w.Dd_oo = w.yref + nstate;
    w.Dd_vv = w.Dd_oo + (size_t)ntraj * no * no;
    w.Dd_ov = w.Dd_vv + (size_t)ntraj * nv * nv;
    w.fa = FieldArgs{};
    w.eg = (unsigned)((n1 * ntraj + 255) / 256);
    bool same_dirs = h->dd_valid && h->dd_ntraj == ntraj;
    for (int t = 0; t < ntraj && same_dirs; ++t)
        for (int k = 0; k < 3; ++k) same_dirs = same_dirs && (h->dd_dir[t][k] == fields[t].dir[k]);
    for (int t = 0; t < ntraj; ++t) {
        const double* d = fields[t].dir;
        w.fa.D00[t] = d[0] * h->D_00[0] + d[1] * h->D_00[1] + d[2] * h->D_00[2];
        if (same_dirs) continue;
        const long long a = no * no, b = nv * nv, c = no * nv;
        combine3_kernel<<<(unsigned)((a + 255) / 256), 256, 0, st>>>(a, h->D_oo, d[0], d[1], d[2], w.Dd_oo + t * a);
        combine3_kernel<<<(unsigned)((b + 255) / 256), 256, 0, st>>>(b, h->D_vv, d[0], d[1], d[2], w.Dd_vv + t * b);
        combine3_kernel<<<(unsigned)((c + 255) / 256), 256, 0, st>>>(c, h->D_ov, d[0], d[1], d[2], w.Dd_ov + t * c);
        h->kernel_launches += 3;
        for (int k = 0; k < 3; ++k) h->dd_dir[t][k] = d[k];
    }
    RT_CUDA(cudaGetLastError());
    h->dd_valid = true; h->dd_ntraj = ntraj;
    bool cont = false;
    for (int t = 0; t < ntraj; ++t) cont = cont || (fields[t].flags & RTTDA_FIELD_CONTINUE);
    if (cont) {
        RT_CHECK(h->yref_ntraj == ntraj, "propagate: RTTDA_FIELD_CONTINUE without a previous call of the same ntraj on this handle");
        return RTTDA_OK;
    }
    bool any_kick = false;
    for (int t = 0; t < ntraj; ++t) {
        w.fa.E[t] = fields[t].type == RTTDA_DELTA ? fields[t].E0 : 0.0;
        any_kick |= w.fa.E[t] != 0.0;
    }
    if (any_kick) {
        RT_CUDA(cudaMemsetAsync(w.hy, 0, nstate * sizeof(double), st));
        RT_TRY(apply_field(h, ntraj, y, w.hy, w.Dd_oo, w.Dd_vv, w.Dd_ov, w.fa, st));
        kick_kernel<<<w.eg, 256, 0, st>>>((long long)n1, ntraj, w.hy, y, w.fa);
        RT_CUDA(cudaGetLastError());
        h->kernel_launches++;
    }
    RT_CUDA(cudaMemcpyAsync(w.yref, y, nstate * sizeof(double), cudaMemcpyDeviceToDevice, st));
    h->yref_ntraj = ntraj;
    return RTTDA_OK;
}

// observe_kernel writing to the control block's log row of the current step (no-op without a log)
__global__ void __launch_bounds__(1024)
observe_dev_kernel(long long n1, const double* __restrict__ y, const double* __restrict__ yref, const PropCtl* __restrict__ c)
{
    if (c->log == nullptr) return;
    const int t = blockIdx.x;
    double* out = c->log + ((long long)c->step * c->ntraj + t) * 3;
    const double *q = y + 2 * t * n1, *p = q + n1, *qr = yref + 2 * t * n1, *pr = qr + n1;
    double a = 0, b = 0, cc = 0;
    for (long long i = threadIdx.x; i < n1; i += blockDim.x) {
        const double qi = q[i], pi = p[i], qri = qr[i], pri = pr[i];
        a = fma(qi, qi, fma(pi, pi, a));
        b = fma(qri, qi, fma(pri, pi, b));
        cc = fma(qri, pi, fma(-pri, qi, cc));
    }
    __shared__ double red[3][32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
        cc += __shfl_xor_sync(0xffffffffu, cc, o);
    }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = a; red[1][threadIdx.x >> 5] = b; red[2][threadIdx.x >> 5] = cc; }
    __syncthreads();
    if (threadIdx.x < 32) {
        const int nw = blockDim.x >> 5;
        a = threadIdx.x < nw ? red[0][threadIdx.x] : 0.0;
        b = threadIdx.x < nw ? red[1][threadIdx.x] : 0.0;
        cc = threadIdx.x < nw ? red[2][threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_xor_sync(0xffffffffu, a, o);
            b += __shfl_xor_sync(0xffffffffu, b, o);
            cc += __shfl_xor_sync(0xffffffffu, cc, o);
        }
        if (threadIdx.x == 0) { out[0] = a; out[1] = b; out[2] = cc; }
    }
}

// One RK4 step with every per-step quantity read from the control block: the body of the captured graph.
static int rk4_step_dev(Handle* h, int ntraj, double* y, const PropWs& w, unsigned active, double dt, cudaStream_t st)
{
    const size_t no = h->nocc, nv = h->nvirt, n1 = (size_t)h->ncsf + 1;
    PropCtl* c = (PropCtl*)h->d_ctl;
    const double ts_off[4] = {0.0, 0.5, 0.5, 1.0}, wgt[4] = {1.0, 2.0, 2.0, 1.0}, cnext[4] = {0.5 * dt, 0.5 * dt, dt, 0.0};
    for (int s = 0; s < 4; ++s) {
        const double* in = (s == 0) ? y : w.ys;
        RT_TRY(sigma_impl(h, 2 * ntraj, in + 1, (long long)n1, w.hy + 1, (long long)n1, st));
        field_eval_kernel<<<1, 32, 0, st>>>(c, ts_off[s]);
        field_elem_dev_kernel<<<2 * ntraj, 1024, 0, st>>>(h->ncsf, in, w.hy, w.Dd_ov, c);
        RT_CUDA(cudaGetLastError());
        h->kernel_launches += 2;
        for (int t = 0; t < ntraj; ++t) {
            if (!(active >> t & 1u)) continue;               // NONE / DELTA: E(t) is identically zero
            GemmDesc g{};
            g.batch = 2; g.beta = 1.0; g.alpha = 1.0;
            g.alpha_dev = c->E + t;                           // + E Y D_vv
            g.M = (int)no; g.N = (int)nv; g.K = (int)nv;
            g.A = in + (size_t)t * 2 * n1 + 1; g.sam = nv; g.sak = 1; g.sabatch = n1;
            g.B = w.Dd_vv + (size_t)t * nv * nv; g.sbk = nv; g.sbn = 1; g.sbbatch = 0;
            g.C = w.hy + (size_t)t * 2 * n1 + 1; g.scm = nv; g.scn = 1; g.scbatch = n1;
            RT_TRY(gemm_f64(g, st));
            g.alpha_dev = c->mE + t;                          // - E D_oo Y
            g.M = (int)no; g.N = (int)nv; g.K = (int)no;
            g.A = w.Dd_oo + (size_t)t * no * no; g.sam = no; g.sak = 1; g.sabatch = 0;
            g.B = in + (size_t)t * 2 * n1 + 1; g.sbk = nv; g.sbn = 1; g.sbbatch = n1;
            RT_TRY(gemm_f64(g, st));
            h->kernel_launches += 2;
        }
        rk4_stage_kernel<<<w.eg, 256, 0, st>>>((long long)n1, ntraj, w.hy, y, w.ys, w.ksum, wgt[s], cnext[s], dt / 6.0,
                                                s == 0, s == 3);
        RT_CUDA(cudaGetLastError());
        h->kernel_launches++;
    }
    observe_dev_kernel<<<ntraj, 1024, 0, st>>>((long long)n1, y, w.yref, c);
    step_advance_kernel<<<1, 1, 0, st>>>(c);
    RT_CUDA(cudaGetLastError());
    h->kernel_launches += 2;
    return RTTDA_OK;
}

// Graph-replayed RK4 run (RTTDA_OPT_GRAPH): upload the control block, capture one step if the cached graph does not
// fit (trajectory count, state pointer, set of trajectories with a field, lane layout), replay it nsteps times.
static int propagate_graph(Handle* h, int ntraj, double* y, const rttda_field_t* fields, double t_start, double dt,
                           int nsteps, double* log, const PropWs& w, cudaStream_t st)
{
    if (!h->d_ctl) RT_CUDA(cudaMalloc(&h->d_ctl, sizeof(PropCtl)));
    PropCtl hc{};
    hc.t_start = t_start; hc.dt = dt; hc.log = log; hc.step = 0; hc.ntraj = ntraj;
    unsigned active = 0;
    for (int t = 0; t < ntraj; ++t) {
        hc.f[t] = fields[t];
        hc.D00[t] = w.fa.D00[t];
        if (fields[t].type != RTTDA_NONE && fields[t].type != RTTDA_DELTA) active |= 1u << t;
    }
    // The legacy default stream cannot be captured, so the step is captured on and replayed from the handle's own stream,
    // which is ordered after the caller's stream here and joined back into it at the end.
    cudaStream_t user = st;
    if (!h->graph_st) {
        RT_CUDA(cudaStreamCreateWithFlags(&h->graph_st, cudaStreamNonBlocking));
        RT_CUDA(cudaEventCreateWithFlags(&h->graph_ev, cudaEventDisableTiming));
    }
    st = h->graph_st;
    RT_CUDA(cudaEventRecord(h->graph_ev, user));
    RT_CUDA(cudaStreamWaitEvent(st, h->graph_ev, 0));
    RT_CUDA(cudaMemcpyAsync(h->d_ctl, &hc, sizeof(PropCtl), cudaMemcpyHostToDevice, st));   // pageable source: staged before return
    Handle::GraphKey key;
    RT_TRY(sigma_reserve(h, 2 * ntraj));
    key.ntraj = ntraj; key.y = y; key.active = active; key.nlanes = h->nlanes; key.epoch = h->ws_epoch;
    const Handle::GraphKey& k0 = h->graph_key;
    if (!h->step_graph || k0.ntraj != key.ntraj || k0.y != key.y || k0.active != key.active || k0.nlanes != key.nlanes ||
        k0.epoch != key.epoch || h->graph_dt != dt) {
        if (h->step_graph) { cudaGraphExecDestroy(h->step_graph); h->step_graph = nullptr; }
        const long long l0 = h->kernel_launches;
        cudaGraph_t graph = nullptr;
        RT_CUDA(cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed));
        h->capturing = true;
        const int rc = rk4_step_dev(h, ntraj, y, w, active, dt, st);
        h->capturing = false;
        const cudaError_t e = cudaStreamEndCapture(st, &graph);
        if (rc != RTTDA_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
        RT_CUDA(e);
        const cudaError_t e2 = cudaGraphInstantiate(&h->step_graph, graph, 0);
        cudaGraphDestroy(graph);
        RT_CUDA(e2);
        h->graph_launches = h->kernel_launches - l0;
        h->kernel_launches = l0;
        h->graph_key = key;
        h->graph_dt = dt;
    }
    for (int n = 0; n < nsteps; ++n) RT_CUDA(cudaGraphLaunch(h->step_graph, st));
    RT_CUDA(cudaEventRecord(h->graph_ev, st));
    RT_CUDA(cudaStreamWaitEvent(user, h->graph_ev, 0));
    h->kernel_launches += h->graph_launches * nsteps;
    return RTTDA_OK;
}

int propagate_impl(Handle* h, int ntraj, double* y, const rttda_field_t* fields, double t_start, double dt,
                   int nsteps, double* log, cudaStream_t st)
{
    const size_t n1 = (size_t)h->ncsf + 1;
    PropWs w;
    RT_TRY(prop_prologue(h, ntraj, y, fields, w, st));
    if (h->use_graph && nsteps > 0) return propagate_graph(h, ntraj, y, fields, t_start, dt, nsteps, log, w, st);
    double *ys = w.ys, *hy = w.hy, *ksum = w.ksum, *yref = w.yref, *Dd_oo = w.Dd_oo, *Dd_vv = w.Dd_vv, *Dd_ov = w.Dd_ov;
    FieldArgs& fa = w.fa;
    const unsigned eg = w.eg;

    const double ts_off[4] = {0.0, 0.5, 0.5, 1.0};
    const double wgt[4] = {1.0, 2.0, 2.0, 1.0};
    const double cnext[4] = {0.5 * dt, 0.5 * dt, dt, 0.0};
    for (int n = 0; n < nsteps; ++n) {
        const double t0 = t_start + n * dt;
        for (int s = 0; s < 4; ++s) {
            const double* in = (s == 0) ? y : ys;
            // hy singles = A in (both planes of every trajectory in one batched sigma)
            RT_TRY(sigma_impl(h, 2 * ntraj, in + 1, (long long)n1, hy + 1, (long long)n1, st));
            const double ts = t0 + ts_off[s] * dt;
            for (int t = 0; t < ntraj; ++t) fa.E[t] = field_value(fields[t], ts);
            RT_TRY(apply_field(h, ntraj, in, hy, Dd_oo, Dd_vv, Dd_ov, fa, st));
            rk4_stage_kernel<<<eg, 256, 0, st>>>((long long)n1, ntraj, hy, y, ys, ksum, wgt[s], cnext[s],
                                                 dt / 6.0, s == 0, s == 3);
            RT_CUDA(cudaGetLastError());
            h->kernel_launches++;
        }
        if (log) {
            observe_kernel<<<ntraj, 1024, 0, st>>>((long long)n1, y, yref, log + (size_t)n * ntraj * 3);
            RT_CUDA(cudaGetLastError());
            h->kernel_launches++;
        }
    }
    return RTTDA_OK;
}

// ---------------------------------------------------------------------------------------------- SSO
// y[t][dst_plane][e] += c * hy[t][src_plane][e]
__global__ void plane_axpy_kernel(long long n1, int ntraj, double c, const double* __restrict__ hy, int src_plane,
                                  double* __restrict__ y, int dst_plane)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n1 * ntraj) return;
    const long long t = i / n1, e = i % n1;
    y[(2 * t + dst_plane) * n1 + e] = fma(c, hy[(2 * t + src_plane) * n1 + e], y[(2 * t + dst_plane) * n1 + e]);
}

// Second-order symplectic split-operator propagator (the paper's SSO; Stoermer-Verlet reading R22 of
// DESIGN.md): p_half = p - dt/2 H(t_n) q; q += dt H(t_n + dt/2) p_half; p = p_half - dt/2 H(t_n + dt) q, with the
// last H q reused by the next step: two applications of H to one REAL plane per step, i.e. two sigma builds of
// ntraj vectors each (RK4: four builds of 2 ntraj).
int propagate_sso_impl(Handle* h, int ntraj, double* y, const rttda_field_t* fields, double t_start, double dt,
                       int nsteps, double* log, cudaStream_t st)
{
    const size_t n1 = (size_t)h->ncsf + 1;
    const size_t nstate = (size_t)ntraj * 2 * n1;
    PropWs w;
    RT_TRY(prop_prologue(h, ntraj, y, fields, w, st));
    double *hy = w.hy, *yref = w.yref, *Dd_oo = w.Dd_oo, *Dd_vv = w.Dd_vv, *Dd_ov = w.Dd_ov;
    FieldArgs& fa = w.fa;
    const unsigned eg = w.eg;

    // hy[:, plane, :] = H(t) y[:, plane, :]; the other plane of hy is scratch of the field kernels
    auto apply_H = [&](int plane, double t) -> int {
        RT_CUDA(cudaMemsetAsync(hy, 0, nstate * sizeof(double), st));
        RT_TRY(sigma_impl(h, ntraj, y + plane * n1 + 1, (long long)(2 * n1), hy + plane * n1 + 1, (long long)(2 * n1), st));
        for (int k = 0; k < ntraj; ++k) fa.E[k] = field_value(fields[k], t);
        RT_TRY(apply_field(h, ntraj, y, hy, Dd_oo, Dd_vv, Dd_ov, fa, st));
        return RTTDA_OK;
    };
    auto axpy = [&](double c, int src_plane, int dst_plane) -> int {
        plane_axpy_kernel<<<eg, 256, 0, st>>>((long long)n1, ntraj, c, hy, src_plane, y, dst_plane);
        RT_CUDA(cudaGetLastError());
        h->kernel_launches++;
        return RTTDA_OK;
    };
    if (nsteps > 0) RT_TRY(apply_H(0, t_start));                         // H(t_0) q_0
    for (int n = 0; n < nsteps; ++n) {
        const double t0 = t_start + n * dt;
        RT_TRY(axpy(-0.5 * dt, 0, 1));                                   // p_half = p - dt/2 H q
        RT_TRY(apply_H(1, t0 + 0.5 * dt));
        RT_TRY(axpy(dt, 1, 0));                                          // q += dt H p_half
        RT_TRY(apply_H(0, t0 + dt));
        RT_TRY(axpy(-0.5 * dt, 0, 1));                                   // p = p_half - dt/2 H q   (H q kept for the next step)
        if (log) {
            observe_kernel<<<ntraj, 1024, 0, st>>>((long long)n1, y, yref, log + (size_t)n * ntraj * 3);
            RT_CUDA(cudaGetLastError());
            h->kernel_launches++;
        }
    }
    return RTTDA_OK;
}

// ---------------------------------------------------------------------------------------------- populations
// P[t][i] = |X_i^dagger y_t|^2 (eq. 22) for real stationary-state vectors X_i [nstates][n1]; one block per (t, i)
__global__ void __launch_bounds__(256)
populations_kernel(long long n1, int nstates, const double* __restrict__ y, const double* __restrict__ Xs,
                   double* __restrict__ P)
{
    const int t = blockIdx.x / nstates, i = blockIdx.x % nstates;
    const double *q = y + 2 * t * n1, *p = q + n1, *x = Xs + (long long)i * n1;
    double re = 0.0, im = 0.0;
    for (long long e = threadIdx.x; e < n1; e += blockDim.x) {
        const double xv = x[e];
        re = fma(xv, q[e], re);
        im = fma(xv, p[e], im);
    }
    __shared__ double red[2][8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        re += __shfl_xor_sync(0xffffffffu, re, o);
        im += __shfl_xor_sync(0xffffffffu, im, o);
    }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = re; red[1][threadIdx.x >> 5] = im; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { a += red[0][w]; b += red[1][w]; }
        P[blockIdx.x] = a * a + b * b;
    }
}

int populations_impl(Handle* h, int ntraj, const double* y, int nstates, const double* Xs, double* P, cudaStream_t st)
{
    populations_kernel<<<ntraj * nstates, 256, 0, st>>>((long long)h->ncsf + 1, nstates, y, Xs, P);
    RT_CUDA(cudaGetLastError());
    h->kernel_launches++;
    return RTTDA_OK;
}

// ---------------------------------------------------------------------------------------------- spectrum
// eq. 21 with the recipe of P:212: the correlation function of one trajectory, R(k dt) for k = 0..n, is
// mirrored (R(-t) = R(t)^*), multiplied by the Hann window over its 2n+1 points, padded with `pad` zeros and Fourier
// transformed; the spectrum is omega |F| on the grid omega_j = 2 pi j / (npad dt), j = 1..npad/2.  The transform is
// a direct DFT (n is a few thousand steps: 1e8 phase factors): thread = one frequency, block = SPEC_TILE of them;
// the windowed signal is built tile by tile in shared memory, the phase index (j m mod npad) is kept as an integer
// so that sincospi sees an argument reduced exactly.
constexpr int SPEC_TILE = 128;

__global__ void __launch_bounds__(SPEC_TILE)
spectrum_kernel(int ntraj, int n, const double* __restrict__ log, double r0re, double r0im, int traj0, double dt,
                long long npad, int nout, double* __restrict__ omega, double* __restrict__ inten)
{
    __shared__ double2 s_x[SPEC_TILE];
    const int traj = traj0 + blockIdx.y;
    const long long M = 2LL * n + 1;
    const int i = blockIdx.x * SPEC_TILE + threadIdx.x;
    const long long j = (long long)i + 1;                      // frequency index; also the phase increment per sample
    const double inv = 2.0 / (double)npad;
    double re = 0.0, im = 0.0;
    for (long long m0 = 0; m0 < M; m0 += SPEC_TILE) {
        const long long m = m0 + threadIdx.x;
        double2 x = make_double2(0.0, 0.0);
        if (m < M) {
            const long long k = m - n;                          // sample time k dt
            const long long a = k < 0 ? -k : k;
            double xr, xi;
            if (a == 0) { xr = r0re; xi = r0im; }
            else {
                const double* e = log + ((a - 1) * ntraj + traj) * 3;
                xr = e[1]; xi = e[2];
            }
            if (k < 0) xi = -xi;
            const double w = (M > 1) ? 0.5 - 0.5 * cospi(2.0 * (double)m / (double)(M - 1)) : 1.0;
            x = make_double2(w * xr, w * xi);
        }
        __syncthreads();
        s_x[threadIdx.x] = x;
        __syncthreads();
        if (i < nout) {
            const int cnt = (int)((M - m0 < SPEC_TILE) ? (M - m0) : SPEC_TILE);
            long long r = (j * (m0 % npad)) % npad;             // j, m0 % npad < 2^31
            for (int t = 0; t < cnt; ++t) {
                double sn, cs;
                sincospi((double)r * inv, &sn, &cs);            // exp(+2 pi i j m / npad): numpy's bin npad - j
                const double2 v = s_x[t];
                re = fma(v.x, cs, fma(-v.y, sn, re));
                im = fma(v.x, sn, fma(v.y, cs, im));
                r += j;
                if (r >= npad) r -= npad;
            }
        }
    }
    if (i < nout) {
        const double om = 6.283185307179586476925 * (double)j / ((double)npad * dt);
        if (blockIdx.y == 0) omega[i] = om;
        inten[(long long)traj * nout + i] = om * sqrt(re * re + im * im);
    }
}

// eq. 23: mean of the ntraj spectra (x, y, z polarisation) into row ntraj
__global__ void spectrum_mean_kernel(int ntraj, int nout, double* __restrict__ inten)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nout) return;
    double s = 0.0;
    for (int t = 0; t < ntraj; ++t) s += inten[(long long)t * nout + i];
    inten[(long long)ntraj * nout + i] = s / (double)ntraj;
}

int spectrum_impl(int ntraj, int n, const double* R0, const double* log, double dt, int pad, int nout, double* omega,
                  double* inten, cudaStream_t st)
{
    const long long npad = 2LL * n + 1 + pad;
    dim3 grid((nout + SPEC_TILE - 1) / SPEC_TILE, 1);
    for (int t = 0; t < ntraj; ++t) {                           // R(0) of each trajectory is a kernel argument
        spectrum_kernel<<<grid, SPEC_TILE, 0, st>>>(ntraj, n, log, R0[2 * t], R0[2 * t + 1], t, dt, npad, nout, omega,
                                                    inten);
        RT_CUDA(cudaGetLastError());
    }
    spectrum_mean_kernel<<<(nout + 255) / 256, 256, 0, st>>>(ntraj, nout, inten);
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

// ---------------------------------------------------------------------------------------------- Lanczos
// out[i] = sum_e V[i][e] w[e] for i < nv (one block per i)
__global__ void __launch_bounds__(256)
multi_dot_kernel(long long n, const double* __restrict__ V, const double* __restrict__ w, double* __restrict__ out)
{
    const double* v = V + (long long)blockIdx.x * n;
    double s = 0.0;
    for (long long e = threadIdx.x; e < n; e += blockDim.x) s = fma(v[e], w[e], s);
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) a += red[k];
        out[blockIdx.x] = a;
    }
}
// w[e] -= sum_i c[i] V[i][e]
__global__ void multi_axpy_kernel(long long n, int nv, const double* __restrict__ V, const double* __restrict__ c,
                                  double* __restrict__ w)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    double s = w[e];
    for (int i = 0; i < nv; ++i) s = fma(-c[i], V[(long long)i * n + e], s);
    w[e] = s;
}
// w -= V^T (V w) for the nv rows of V (coefficients through `dots`, DEVICE [nv])
int project_out(long long n, int nv, const double* V, double* w, double* dots, cudaStream_t st)
{
    if (nv <= 0) return RTTDA_OK;
    multi_dot_kernel<<<nv, 256, 0, st>>>(n, V, w, dots);
    multi_axpy_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, nv, V, dots, w);
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

__global__ void scale_to_kernel(long long n, double a, const double* __restrict__ in, double* __restrict__ out)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n) out[e] = a * in[e];
}

// m steps of symmetric Lanczos on the singles block A through sigma_impl (one sigma vector per step), with full
// reorthogonalisation (twice) against all previous Lanczos vectors.  alpha, beta: host [m]; V: DEVICE [m+1][ncsf].
int lanczos_impl(Handle* h, int m, const double* v0, double* alpha, double* beta, double* V, cudaStream_t st)
{
    const long long n = h->ncsf;
    const unsigned eg = (unsigned)((n + 255) / 256);
    RT_TRY(ensure_ws(h, &h->wsZ, &h->wsZ_n, (size_t)n + (size_t)m + 2));
    double* w = h->wsZ;
    double* dots = h->wsZ + n;                              // [m+1] device scalars
    std::vector<double> hd((size_t)m + 2);
    // v_1 = v0 / |v0|
    multi_dot_kernel<<<1, 256, 0, st>>>(n, v0, v0, dots);
    RT_CUDA(cudaMemcpyAsync(hd.data(), dots, sizeof(double), cudaMemcpyDeviceToHost, st));
    RT_CUDA(cudaStreamSynchronize(st));
    RT_CHECK(hd[0] > 0.0, "rttda_lanczos: zero start vector");
    scale_to_kernel<<<eg, 256, 0, st>>>(n, 1.0 / std::sqrt(hd[0]), v0, V);
    h->kernel_launches += 2;
    for (int j = 0; j < m; ++j) {
        double* vj = V + (size_t)j * n;
        RT_TRY(sigma_impl(h, 1, vj, n, w, n, st));                              // w = A v_j
        // one pass of coefficients against v_0..v_j removes alpha_j v_j and beta_{j-1} v_{j-1} (and, in exact
        // arithmetic, nothing else); alpha_j is the coefficient of v_j in that first pass
        for (int pass = 0; pass < 3; ++pass) {
            multi_dot_kernel<<<j + 1, 256, 0, st>>>(n, V, w, dots);
            if (pass == 0) RT_CUDA(cudaMemcpyAsync(hd.data(), dots + j, sizeof(double), cudaMemcpyDeviceToHost, st));
            multi_axpy_kernel<<<eg, 256, 0, st>>>(n, j + 1, V, dots, w);
            h->kernel_launches += 2;
        }
        multi_dot_kernel<<<1, 256, 0, st>>>(n, w, w, dots);
        RT_CUDA(cudaMemcpyAsync(hd.data() + 1, dots, sizeof(double), cudaMemcpyDeviceToHost, st));
        RT_CUDA(cudaStreamSynchronize(st));
        alpha[j] = hd[0];
        beta[j] = std::sqrt(hd[1]);
        RT_CHECK(beta[j] > 0.0, "rttda_lanczos: breakdown (invariant subspace reached)");
        scale_to_kernel<<<eg, 256, 0, st>>>(n, 1.0 / beta[j], w, V + (size_t)(j + 1) * n);
        h->kernel_launches += 2;
    }
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

}  // namespace rttda
