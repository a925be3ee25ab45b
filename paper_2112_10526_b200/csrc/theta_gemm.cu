// Base activations theta = sigma W^T + b  (W in C^{MxN}, b in C^M: PAPER.md Eq. (7)).
//   theta[s][m] = bg[m] + sum_k sigma[s][k] * Wg[m][k],   s < B, m < M_eff (M_eff is a multiple of 128)
// FP32 SIMT version: products with +-1 are exact; accumulation is fp32 in two levels (a fresh partial sum per
// 16-wide k tile, added to the running sum once per tile), which cuts the rounding error of a length-1024 sum by
// ~3.5x against plain sequential accumulation -- needed for the 1e-5 bound on ln psi at N = 1024 (Q12).
// 128x128x16 tiles, 256 threads, 8x8 outputs per thread, register-prefetched global loads.
#include "nk_internal.h"

namespace nk {

constexpr int BM = 128, BN = 128, BK = 16, GEMM_THREADS = 256;

__global__ void __launch_bounds__(GEMM_THREADS, 1)
theta_gemm_simt_kernel(const int8_t* __restrict__ sigma, int64_t B, int N, int M_eff, const float* __restrict__ Wg,
                       const float* __restrict__ bg, float* __restrict__ theta) {
    __shared__ __align__(16) float As[2][BK][BM];   // sigma tile, transposed: [k][sample]
    __shared__ __align__(16) float Bs[2][BK][BN];   // W tile, transposed:     [k][hidden]
    const int tid = threadIdx.x;
    const int64_t s0 = (int64_t)blockIdx.y * BM;
    const int m0 = blockIdx.x * BN;
    // loader mapping: 128 rows x 16 k = 2048 elements; thread t loads row (t >> 1), k half (t & 1) * 8 .. +8
    const int lrow = tid >> 1, lk = (tid & 1) * 8;
    const int8_t* ap = sigma + (s0 + lrow) * N;
    const float* bp = Wg + (size_t)(m0 + lrow) * N;
    const bool arow_ok = (s0 + lrow) < B;

    float areg[8], breg[8];
    auto load_tile = [&](int k0) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int k = k0 + lk + u;
            areg[u] = (arow_ok && k < N) ? (float)ap[k] : 0.f;
            breg[u] = (k < N) ? bp[k] : 0.f;
        }
    };
    auto store_tile = [&](int buf) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            As[buf][lk + u][lrow] = areg[u];
            Bs[buf][lk + u][lrow] = breg[u];
        }
    };

    // compute mapping: thread owns samples {ty*4..+3, 64+ty*4..+3} x hidden {tx*4..+3, 64+tx*4..+3}
    const int tx = tid & 15, ty = tid >> 4;
    float acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;

    const int n_kt = (N + BK - 1) / BK;
    load_tile(0);
    store_tile(0);
    __syncthreads();
    for (int kt = 0; kt < n_kt; ++kt) {
        const int buf = kt & 1;
        if (kt + 1 < n_kt) load_tile((kt + 1) * BK);
        float part[8][8];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) part[i][j] = 0.f;
#pragma unroll
        for (int k = 0; k < BK; ++k) {
            const float4 a0 = *reinterpret_cast<const float4*>(&As[buf][k][ty * 4]);
            const float4 a1 = *reinterpret_cast<const float4*>(&As[buf][k][64 + ty * 4]);
            const float4 b0 = *reinterpret_cast<const float4*>(&Bs[buf][k][tx * 4]);
            const float4 b1 = *reinterpret_cast<const float4*>(&Bs[buf][k][64 + tx * 4]);
            const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float bv[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j) part[i][j] = fmaf(av[i], bv[j], part[i][j]);
        }
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[i][j] += part[i][j];
        if (kt + 1 < n_kt) {
            store_tile(buf ^ 1);
            __syncthreads();
        }
    }

    const float4 bias0 = *reinterpret_cast<const float4*>(&bg[m0 + tx * 4]);
    const float4 bias1 = *reinterpret_cast<const float4*>(&bg[m0 + 64 + tx * 4]);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int64_t s = s0 + (i < 4 ? ty * 4 + i : 64 + ty * 4 + (i - 4));
        if (s < B) {
            float* row = theta + s * M_eff + m0;
            float4 o0 = {acc[i][0] + bias0.x, acc[i][1] + bias0.y, acc[i][2] + bias0.z, acc[i][3] + bias0.w};
            float4 o1 = {acc[i][4] + bias1.x, acc[i][5] + bias1.y, acc[i][6] + bias1.z, acc[i][7] + bias1.w};
            *reinterpret_cast<float4*>(row + tx * 4) = o0;
            *reinterpret_cast<float4*>(row + 64 + tx * 4) = o1;
        }
    }
}

cudaError_t launch_theta_gemm(const int8_t* sigma, int64_t B, int N, int M_eff, const float* Wg, const float* bg,
                              float* theta, cudaStream_t st) {
    if (B <= 0) return cudaSuccess;
    dim3 grid(M_eff / BN, (unsigned)((B + BM - 1) / BM));
    theta_gemm_simt_kernel<<<grid, GEMM_THREADS, 0, st>>>(sigma, B, N, M_eff, Wg, bg, theta);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
