// Sample statistics of the local energies:  E[A~] ~ (1/N_s) sum_i A~(s_i)  (Eq. (17)
// L675) and the population variance mean |E - mean|^2 (Q10).  One CTA, fp64, fixed reduction order:
// the result does not depend on chunk_size and is bit-reproducible.
#include "nk_internal.h"

namespace nk {

constexpr int ST = 1024;

__device__ double block_sum(double v, double* sh) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    v = (threadIdx.x < ST / 32) ? sh[threadIdx.x] : 0.0;
    if (warp == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) sh[0] = v;
    }
    __syncthreads();
    return sh[0];
}

__global__ void __launch_bounds__(ST) stats_kernel(const float* __restrict__ eloc, int64_t B, int cplx,
                                                   double* __restrict__ out) {
    __shared__ double sh[ST / 32];
    double sr = 0.0, si = 0.0;
    for (int64_t n = threadIdx.x; n < B; n += ST) {
        if (cplx) { sr += (double)eloc[2 * n]; si += (double)eloc[2 * n + 1]; }
        else sr += (double)eloc[n];
    }
    const double mr = block_sum(sr, sh) / (double)B;
    const double mi = cplx ? block_sum(si, sh) / (double)B : 0.0;
    double m2 = 0.0;
    for (int64_t n = threadIdx.x; n < B; n += ST) {
        const double dr = (double)(cplx ? eloc[2 * n] : eloc[n]) - mr;
        const double di = cplx ? (double)eloc[2 * n + 1] - mi : 0.0;
        m2 += dr * dr + di * di;
    }
    const double var = block_sum(m2, sh) / (double)B;
    if (threadIdx.x == 0) { out[0] = mr; out[1] = mi; out[2] = var; out[3] = (double)B; }
}

cudaError_t launch_stats(const void* eloc, int64_t B, int dtype, double* stats_out, cudaStream_t st) {
    if (B <= 0) return cudaMemsetAsync(stats_out, 0, 4 * sizeof(double), st);
    stats_kernel<<<1, ST, 0, st>>>((const float*)eloc, B, dtype == NK_C64, stats_out);
    count_launch();
    return cudaGetLastError();
}

// NK_CHECK_SPINS: *flag |= 1 if any entry of sigma is not +1 or -1 (the spin encoding of PAPER.md L178)
__global__ void check_spins_kernel(const int8_t* __restrict__ sigma, int64_t n, int* __restrict__ flag) {
    int bad = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int v = sigma[i];
        bad |= (v != 1 && v != -1);
    }
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(flag, 1);
}

cudaError_t launch_check_spins(const int8_t* sigma, int64_t n, int* flag, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(flag, 0, sizeof(int), st);
    if (e != cudaSuccess || n <= 0) return e;
    int64_t blocks = (n + 255) / 256;
    if (blocks > 2368) blocks = 2368;
    check_spins_kernel<<<(unsigned)blocks, 256, 0, st>>>(sigma, n, flag);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
