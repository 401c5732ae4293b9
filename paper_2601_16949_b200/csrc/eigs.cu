// TI-TDA eigenpairs A X = omega X (eq. 2; the paper's reference method for Table 1) by block Davidson
// on the same multi-vector sigma builds: every iteration applies A to a BLOCK of new directions in one rttda sigma call
// (one ERI pass serving all of them), i.e. the large-nvec regime of config 5 in a real algorithm (NEXT-3 of DESIGN.md).
//
//   V (m x n) orthonormal search space, W = A V;  H = V W^T (m x m, host, Jacobi);  Ritz pairs (theta_j, y_j), lowest k;
//   x_j = sum_i y_ij V_i,  r_j = sum_i y_ij W_i - theta_j x_j;  converged when max_j |r_j|_2 <= tol;
//   new directions t_j = r_j / (theta_j - d_eps) (diagonal preconditioner: d_eps is the diagonal of A up to the
//   two-electron part, eq. 3), orthonormalised against V and each other (two passes of Gram-Schmidt), appended.
//   The space is collapsed onto the current Ritz vectors when it reaches mmax.
// All vectors live on the device; only H, y and a few norms cross to the host.
#include <algorithm>
#include <cmath>
#include <vector>
#include "common.cuh"

namespace rttda {

// Cyclic Jacobi for a symmetric m x m matrix (row-major, destroyed); eigenvalues ascending in w, eigenvectors as
// COLUMNS of Y (row-major m x m).
static void jacobi_eigh(int m, std::vector<double>& H, std::vector<double>& w, std::vector<double>& Y)
{
    Y.assign((size_t)m * m, 0.0);
    for (int i = 0; i < m; ++i) Y[(size_t)i * m + i] = 1.0;
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0.0, diag = 0.0;
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < m; ++j) (i == j ? diag : off) += H[(size_t)i * m + j] * H[(size_t)i * m + j];
        if (off <= 1e-30 * std::max(diag, 1e-300)) break;
        for (int p = 0; p < m - 1; ++p)
            for (int q = p + 1; q < m; ++q) {
                const double apq = H[(size_t)p * m + q];
                if (apq == 0.0) continue;
                const double app = H[(size_t)p * m + p], aqq = H[(size_t)q * m + q];
                const double th = 0.5 * (aqq - app) / apq;
                const double t = (th >= 0.0 ? 1.0 : -1.0) / (std::fabs(th) + std::sqrt(th * th + 1.0));
                const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
                for (int k = 0; k < m; ++k) {
                    const double hkp = H[(size_t)k * m + p], hkq = H[(size_t)k * m + q];
                    H[(size_t)k * m + p] = c * hkp - s * hkq;
                    H[(size_t)k * m + q] = s * hkp + c * hkq;
                }
                for (int k = 0; k < m; ++k) {
                    const double hpk = H[(size_t)p * m + k], hqk = H[(size_t)q * m + k];
                    H[(size_t)p * m + k] = c * hpk - s * hqk;
                    H[(size_t)q * m + k] = s * hpk + c * hqk;
                }
                for (int k = 0; k < m; ++k) {
                    const double ykp = Y[(size_t)k * m + p], ykq = Y[(size_t)k * m + q];
                    Y[(size_t)k * m + p] = c * ykp - s * ykq;
                    Y[(size_t)k * m + q] = s * ykp + c * ykq;
                }
            }
    }
    std::vector<int> order(m);
    for (int i = 0; i < m; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int a, int b) { return H[(size_t)a * m + a] < H[(size_t)b * m + b]; });
    w.resize(m);
    std::vector<double> Ys((size_t)m * m);
    for (int j = 0; j < m; ++j) {
        w[j] = H[(size_t)order[j] * m + order[j]];
        for (int i = 0; i < m; ++i) Ys[(size_t)i * m + j] = Y[(size_t)i * m + order[j]];
    }
    Y.swap(Ys);
}

// t[j][e] = r[j][e] / (theta_j - deps[e]), denominators kept away from zero
__global__ void davidson_precond_kernel(long long n, int nb, const double* __restrict__ r, const double* __restrict__ theta,
                                        const double* __restrict__ deps, double* __restrict__ t)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * nb) return;
    const int j = (int)(i / n);
    const long long e = i % n;
    double d = theta[j] - deps[e];
    if (fabs(d) < 1e-4) d = d < 0.0 ? -1e-4 : 1e-4;
    t[i] = r[i] / d;
}

// r[j][e] -= theta_j x[j][e]
__global__ void davidson_resid_kernel(long long n, int nb, const double* __restrict__ theta, const double* __restrict__ x,
                                      double* __restrict__ r)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * nb) return;
    r[i] = fma(-theta[i / n], x[i], r[i]);
}

__global__ void unit_vector_kernel(long long n, int nb, const int* __restrict__ pos, double* __restrict__ v)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * nb) return;
    v[i] = (i % n == pos[i / n]) ? 1.0 : 0.0;
}

__global__ void scale_rows_kernel(long long n, int nb, const double* __restrict__ s, double* __restrict__ v)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n * nb) v[i] *= s[i / n];
}

// out[j] = a[j] . b[j] for j < nb (one block per row)
__global__ void __launch_bounds__(256)
row_dot_kernel(long long n, const double* __restrict__ a, const double* __restrict__ b, double* __restrict__ out)
{
    const double *x = a + (long long)blockIdx.x * n, *y = b + (long long)blockIdx.x * n;
    double s = 0.0;
    for (long long e = threadIdx.x; e < n; e += blockDim.x) s = fma(x[e], y[e], s);
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 8; ++k) t += red[k];
        out[blockIdx.x] = t;
    }
}

static int gemm_simple(int M, int N, int K, double alpha, const double* A, long long sam, long long sak, const double* B,
                       long long sbk, long long sbn, double beta, double* C, long long scm, long long scn, cudaStream_t st)
{
    GemmDesc g{};
    g.M = M; g.N = N; g.K = K; g.batch = 1; g.alpha = alpha; g.beta = beta;
    g.A = A; g.sam = sam; g.sak = sak; g.sabatch = 0;
    g.B = B; g.sbk = sbk; g.sbn = sbn; g.sbbatch = 0;
    g.C = C; g.scm = scm; g.scn = scn; g.scbatch = 0;
    return gemm_f64(g, st);
}

int eigs_impl(Handle* h, int k, int nblock, double tol, int maxiter, double* omega, double* X, double* resid, int* niter,
              int* nsigma, cudaStream_t st)
{
    const long long n = h->ncsf;
    const int nb = std::min<long long>(std::max(nblock, k), n);
    const int mmax = (int)std::min<long long>(n, std::max(8 * nb, 3 * k + nb));
    // workspace: V, W (mmax rows), Xr, R, T (nb rows each), small: H (mmax^2), Y (mmax x nb), theta, scal (nb), coef (mmax x nb)
    const size_t small = (size_t)mmax * mmax + 2 * (size_t)mmax * nb + 4 * (size_t)nb + 64;
    const size_t need = (2 * (size_t)mmax + 3 * (size_t)nb) * n + small;
    double* ws = nullptr;
    {
        cudaError_t e = cudaMalloc((void**)&ws, need * sizeof(double));
        if (e != cudaSuccess) { set_error(std::string("rttda_eigs: workspace cudaMalloc: ") + cudaGetErrorString(e)); return RTTDA_ENOMEM; }
    }
    struct Free { double* p; ~Free() { cudaFree(p); } } guard{ws};
    double* V = ws;
    double* W = V + (size_t)mmax * n;
    double* Xr = W + (size_t)mmax * n;
    double* R = Xr + (size_t)nb * n;
    double* T = R + (size_t)nb * n;
    double* dH = T + (size_t)nb * n;
    double* dY = dH + (size_t)mmax * mmax;
    double* dC = dY + (size_t)mmax * nb;
    double* dth = dC + (size_t)mmax * nb;
    double* dsc = dth + nb;
    int* dpos = reinterpret_cast<int*>(dsc + 2 * nb);

    // start: unit vectors on the nb smallest orbital-energy differences
    std::vector<double> de((size_t)n);
    RT_CUDA(cudaMemcpyAsync(de.data(), h->deps, n * sizeof(double), cudaMemcpyDeviceToHost, st));
    RT_CUDA(cudaStreamSynchronize(st));
    std::vector<int> order((size_t)n);
    for (long long i = 0; i < n; ++i) order[i] = (int)i;
    std::partial_sort(order.begin(), order.begin() + nb, order.end(), [&](int a, int b) { return de[a] < de[b] || (de[a] == de[b] && a < b); });
    RT_CUDA(cudaMemcpyAsync(dpos, order.data(), nb * sizeof(int), cudaMemcpyHostToDevice, st));
    const unsigned gb = (unsigned)((n * nb + 255) / 256);
    unit_vector_kernel<<<gb, 256, 0, st>>>(n, nb, dpos, V);
    RT_CUDA(cudaGetLastError());
    int m = 0, mnew = nb, nsig = 0, it = 0;
    std::vector<double> H, Y, w, hsc(2 * (size_t)nb), rn(k, 0.0), th(nb);
    bool converged = false;
    for (it = 0; it < maxiter; ++it) {
        // W_new = A V_new: one multi-vector sigma build
        RT_TRY(sigma_impl(h, mnew, V + (size_t)m * n, n, W + (size_t)m * n, n, st));
        nsig += mnew;
        m += mnew;
        // H = V W^T, symmetrised on the host
        RT_TRY(gemm_simple(m, m, (int)n, 1.0, V, n, 1, W, 1, n, 0.0, dH, m, 1, st));
        H.resize((size_t)m * m);
        RT_CUDA(cudaMemcpyAsync(H.data(), dH, H.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
        RT_CUDA(cudaStreamSynchronize(st));
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < i; ++j) H[(size_t)i * m + j] = H[(size_t)j * m + i] = 0.5 * (H[(size_t)i * m + j] + H[(size_t)j * m + i]);
        jacobi_eigh(m, H, w, Y);
        const int kk = std::min(nb, m);
        std::vector<double> Yk((size_t)m * kk);
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < kk; ++j) Yk[(size_t)i * kk + j] = Y[(size_t)i * m + j];
        for (int j = 0; j < kk; ++j) th[j] = w[j];
        RT_CUDA(cudaMemcpyAsync(dY, Yk.data(), Yk.size() * sizeof(double), cudaMemcpyHostToDevice, st));
        RT_CUDA(cudaMemcpyAsync(dth, th.data(), kk * sizeof(double), cudaMemcpyHostToDevice, st));
        // Ritz vectors Xr = Y^T V and residuals R = Y^T W - theta Xr  (rows j < kk)
        RT_TRY(gemm_simple(kk, (int)n, m, 1.0, dY, 1, kk, V, n, 1, 0.0, Xr, n, 1, st));
        RT_TRY(gemm_simple(kk, (int)n, m, 1.0, dY, 1, kk, W, n, 1, 0.0, R, n, 1, st));
        davidson_resid_kernel<<<(unsigned)((n * kk + 255) / 256), 256, 0, st>>>(n, kk, dth, Xr, R);
        // residual norms
        row_dot_kernel<<<kk, 256, 0, st>>>(n, R, R, dC);
        RT_CUDA(cudaGetLastError());
        std::vector<double> G((size_t)kk);
        RT_CUDA(cudaMemcpyAsync(G.data(), dC, G.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
        RT_CUDA(cudaStreamSynchronize(st));
        double worst = 0.0;
        for (int j = 0; j < k; ++j) { rn[j] = std::sqrt(std::max(G[j], 0.0)); worst = std::max(worst, rn[j]); }
        if (worst <= tol) { converged = true; ++it; break; }
        if (m >= n) { ++it; break; }                          // the space is the whole singles space: nothing to add
        // collapse when the next block would not fit: restart from the current Ritz vectors (W follows by linearity)
        if (m + kk > mmax) {
            RT_TRY(gemm_simple(kk, (int)n, m, 1.0, dY, 1, kk, W, n, 1, 0.0, T, n, 1, st));   // A Xr
            RT_CUDA(cudaMemcpyAsync(V, Xr, (size_t)kk * n * sizeof(double), cudaMemcpyDeviceToDevice, st));
            RT_CUDA(cudaMemcpyAsync(W, T, (size_t)kk * n * sizeof(double), cudaMemcpyDeviceToDevice, st));
            m = kk;
        }
        // preconditioned residuals of the unconverged roots (and of the guard vectors beyond k), orthonormalised
        davidson_precond_kernel<<<(unsigned)((n * kk + 255) / 256), 256, 0, st>>>(n, kk, R, dth, h->deps, T);
        RT_CUDA(cudaGetLastError());
        int added = 0;
        for (int j = 0; j < kk && m + added < mmax; ++j) {
            if (j < k && rn[j] <= tol) continue;
            double* t = V + (size_t)(m + added) * n;
            RT_CUDA(cudaMemcpyAsync(t, T + (size_t)j * n, n * sizeof(double), cudaMemcpyDeviceToDevice, st));
            const int mb = m + added;
            double nrm2 = 0.0;
            for (int pass = 0; pass < 2; ++pass) RT_TRY(project_out(n, mb, V, t, dC, st));   // t -= V^T (V t), twice
            row_dot_kernel<<<1, 256, 0, st>>>(n, t, t, dsc);
            RT_CUDA(cudaMemcpyAsync(&nrm2, dsc, sizeof(double), cudaMemcpyDeviceToHost, st));
            RT_CUDA(cudaStreamSynchronize(st));
            if (!(nrm2 > 1e-24)) continue;                   // direction already in the space
            const double s = 1.0 / std::sqrt(nrm2);
            RT_CUDA(cudaMemcpyAsync(dsc, &s, sizeof(double), cudaMemcpyHostToDevice, st));
            scale_rows_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, 1, dsc, t);
            RT_CUDA(cudaStreamSynchronize(st));              // `s` is a stack variable
            ++added;
        }
        if (added == 0) { ++it; break; }                      // nothing left to add: the space is exhausted
        mnew = added;
    }
    RT_CUDA(cudaMemcpyAsync(X, Xr, (size_t)k * n * sizeof(double), cudaMemcpyDeviceToDevice, st));
    RT_CUDA(cudaStreamSynchronize(st));
    for (int j = 0; j < k; ++j) { omega[j] = th[j]; if (resid) resid[j] = rn[j]; }
    if (niter) *niter = it;
    if (nsigma) *nsigma = nsig;
    if (!converged) { set_error("rttda_eigs: not converged within maxiter (results are the current Ritz pairs)"); return RTTDA_ENOCONV; }
    return RTTDA_OK;
}

}  // namespace rttda
