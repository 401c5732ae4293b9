// FP64 tensor-core GEMM (DMMA, mma.sync.m8n8k4.f64) for the MO<->AO transforms and the field coupling
// (DESIGN.md steps a1, a5, a6; the paper uses cuBLAS for these).  tcgen05 has no FP64 kind, so the
// FP64 tensor path on sm_100a is the warp-level DMMA instruction.
//
//   C(m,n) = alpha * sum_k A(m,k) B(k,n) + beta * C(m,n),   fully strided operands, batched over blockIdx.z.
// Block tile 64x64x16, 4 warps, each warp owns a 32x32 sub-tile = 4x4 DMMA tiles.  Shared tiles are stored
// k-fastest with a row pitch of 20 doubles, which makes both fragment reads bank-conflict free.
#include "common.cuh"

namespace rttda {

constexpr int BM = 64, BN = 64, BK = 16, LDS_PITCH = 20;

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(128) gemm_f64_kernel(GemmDesc g)
{
    __shared__ double As[2][BM][LDS_PITCH];
    __shared__ double Bs[2][BN][LDS_PITCH];
    const int bz = blockIdx.z;
    const double* __restrict__ A = g.A + (long long)bz * g.sabatch;
    const double* __restrict__ B = g.B + (long long)bz * g.sbbatch;
    double* __restrict__ C = g.C + (long long)bz * g.scbatch;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32;
    const int fr = lane >> 2, fc = lane & 3;

    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const bool a_kfast = (g.sak == 1), b_kfast = (g.sbk == 1);
    const double alpha = g.alpha_dev ? g.alpha * __ldg(g.alpha_dev) : g.alpha;
    double ra[8], rb[8];                       // register staging of the next tile (BM*BK/128 = 8 each)

    auto gload = [&](int k0) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int idx = tid + i * 128;
            int m, k;
            if (a_kfast) { k = idx % BK; m = idx / BK; } else { m = idx % BM; k = idx / BM; }
            const int gm = m0 + m, gka = k0 + k;
            ra[i] = (gm < g.M && gka < g.K) ? __ldg(A + (long long)gm * g.sam + (long long)gka * g.sak) : 0.0;
            int n;
            if (b_kfast) { k = idx % BK; n = idx / BK; } else { n = idx % BN; k = idx / BN; }
            const int gn = n0 + n, gkb = k0 + k;
            rb[i] = (gn < g.N && gkb < g.K) ? __ldg(B + (long long)gkb * g.sbk + (long long)gn * g.sbn) : 0.0;
        }
    };
    auto sstore = [&](int buf) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int idx = tid + i * 128;
            int m, k;
            if (a_kfast) { k = idx % BK; m = idx / BK; } else { m = idx % BM; k = idx / BM; }
            As[buf][m][k] = ra[i];
            int n;
            if (b_kfast) { k = idx % BK; n = idx / BK; } else { n = idx % BN; k = idx / BN; }
            Bs[buf][n][k] = rb[i];
        }
    };

    const int nk = (g.K + BK - 1) / BK;
    gload(0);
    sstore(0);
    __syncthreads();
    for (int kt = 0; kt < nk; ++kt) {
        const int buf = kt & 1;
        if (kt + 1 < nk) gload((kt + 1) * BK);
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double af[4], bf[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) af[i] = As[buf][wm + i * 8 + fr][kk + fc];
#pragma unroll
            for (int j = 0; j < 4; ++j) bf[j] = Bs[buf][wn + j * 8 + fr][kk + fc];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
        if (kt + 1 < nk) sstore(buf ^ 1);
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int gm = m0 + wm + i * 8 + fr, gn = n0 + wn + j * 8 + 2 * fc + e;
                if (gm < g.M && gn < g.N) {
                    double* p = C + (long long)gm * g.scm + (long long)gn * g.scn;
                    const double v = alpha * acc[i][j][e];
                    *p = (g.beta == 0.0) ? v : fma(g.beta, *p, v);
                }
            }
}

int gemm_f64(const GemmDesc& g, cudaStream_t st)
{
    if (g.M <= 0 || g.N <= 0 || g.batch <= 0) return RTTDA_OK;
    dim3 grid((g.N + BN - 1) / BN, (g.M + BM - 1) / BM, g.batch), block(128);
    gemm_f64_kernel<<<grid, block, 0, st>>>(g);
    RT_CUDA(cudaGetLastError());
    return RTTDA_OK;
}

}  // namespace rttda
