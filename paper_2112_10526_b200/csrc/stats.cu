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

}  // namespace nk
