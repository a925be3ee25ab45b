// Pipe-peak microbenchmarks for the roofline denominators of bench.py ("MUFU-only / FMA-only
// microbenchmark on the box"): three tiny kernels, each saturating ONE pipe of every SM with independent dependency
// chains and nothing else in the loop —
//   MUFU.EX2      (the log-cosh form's bound: 1 exponential per (amplitude, hidden unit) pair)
//   FFMA          (the product form's arithmetic: 2 FP32 operations per pair)
//   LDS.128       (the product form's measured bound: 4 B of the tanh(delta) table per pair through shared memory)
// nk_pipe_peaks times them with CUDA events and returns lanes (or bytes) per clock per SM at the SM clock it measures
// with clock64 / globaltimer inside the same launches.  Nothing of the hot path runs here.
#include "nk_internal.h"
#include "ptx_helpers.cuh"

namespace nk {

constexpr int PK_THREADS = 512, PK_ITERS = 4096, PK_ILP = 8;

// SM clock seen by a busy kernel: cycles per nanosecond, clock64 against globaltimer on one thread of block 0
struct ClockProbe {
    unsigned long long t0; long long c0;
    __device__ __forceinline__ void start() {
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
        c0 = clock64();
    }
    __device__ __forceinline__ void stop(double* ghz) const {
        const long long c1 = clock64();
        unsigned long long t1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        if (blockIdx.x == 0 && threadIdx.x == 0) *ghz = (double)(c1 - c0) / (double)(t1 - t0);
    }
};

__global__ void __launch_bounds__(PK_THREADS) peak_mufu_kernel(float* out, float seed, double* ghz) {
    ClockProbe cp; cp.start();
    float x[PK_ILP];
#pragma unroll
    for (int i = 0; i < PK_ILP; ++i) x[i] = seed + 1e-3f * (float)(threadIdx.x + i);
    for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < PK_ILP; ++i) x[i] = ex2_approx(-x[i]);    // the negation is an operand modifier; stays in (0, 1]
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PK_ILP; ++i) s += x[i];
    if (s == 12345.678f) out[0] = s;                                   // keeps the chains alive
    cp.stop(ghz);
}

__global__ void __launch_bounds__(PK_THREADS) peak_ffma_kernel(float* out, float a, float b, double* ghz) {
    ClockProbe cp; cp.start();
    float x[PK_ILP];
#pragma unroll
    for (int i = 0; i < PK_ILP; ++i) x[i] = a + (float)(threadIdx.x + i);
    for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < PK_ILP; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PK_ILP; ++i) s += x[i];
    if (s == 12345.678f) out[0] = s;
    cp.stop(ghz);
}

__global__ void __launch_bounds__(PK_THREADS) peak_lds_kernel(float* out, double* ghz) {
    ClockProbe cp; cp.start();
    __shared__ float4 buf[PK_THREADS * 2];
    buf[threadIdx.x] = make_float4(1.f, 2.f, 3.f, 4.f);                  // 1024 float4 = 32 rows of 512 B
    buf[threadIdx.x + PK_THREADS] = make_float4(1.f, 2.f, 3.f, 4.f);
    __syncthreads();
    float4 acc[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) acc[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    // conflict-free: a warp reads 32 consecutive float4 (512 B = 4 wavefronts of 128 B).  The loads are volatile asm so
    // that the compiler can neither hoist them nor keep the 16 distinct values in registers
    const uint32_t base = smem_u32(buf) + (threadIdx.x & 31) * 16;
    for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            float4 v;
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                         : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                         : "r"(base + (uint32_t)(((it * 4 + i) & 31) * 512)));
            acc[i].x += v.x; acc[i].y += v.y; acc[i].z += v.z; acc[i].w += v.w;
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) s += acc[i].x + acc[i].y + acc[i].z + acc[i].w;
    if (s == 12345.678f) out[0] = s;
    cp.stop(ghz);
}

}  // namespace nk

using namespace nk;

extern "C" int nk_pipe_peaks(double* out8_host, void* scratch_dev, nk_stream_t stream) {
    if (!out8_host || !scratch_dev) return NK_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return NK_ERR_CUDA;
    float* fout = (float*)scratch_dev;
    double* ghz = (double*)((uint8_t*)scratch_dev + 64);
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return NK_ERR_CUDA;
    const int grid = sms * 4;                                          // 4 resident CTAs of 512 threads = 64 warps per SM
    float ms[3] = {0.f, 0.f, 0.f};
    for (int which = 0; which < 3; ++which) {
        for (int rep = 0; rep < 3; ++rep) {                            // two warm-ups, the third is timed
            cudaEventRecord(e0, st);
            if (which == 0) peak_mufu_kernel<<<grid, PK_THREADS, 0, st>>>(fout, 0.5f, ghz + 0);
            else if (which == 1) peak_ffma_kernel<<<grid, PK_THREADS, 0, st>>>(fout, 0.999f, 1e-3f, ghz + 1);
            else peak_lds_kernel<<<grid, PK_THREADS, 0, st>>>(fout, ghz + 2);
            cudaEventRecord(e1, st);
        }
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms[which], e0, e1) != cudaSuccess) {
            cudaEventDestroy(e0); cudaEventDestroy(e1);
            return NK_ERR_CUDA;
        }
    }
    double clk[3] = {0.0, 0.0, 0.0};
    cudaError_t e = cudaMemcpyAsync(clk, ghz, sizeof(clk), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess) return NK_ERR_CUDA;
    count_launch(9);
    for (int k = 0; k < 3; ++k) if (!(clk[k] > 0.0)) return NK_ERR_CUDA;
    const double per_sm_threads = 4.0 * PK_THREADS;
    const double mufu_ops = per_sm_threads * PK_ITERS * PK_ILP, ffma_ops = mufu_ops;
    const double lds_bytes = per_sm_threads * PK_ITERS * 4.0 * 16.0;
    out8_host[0] = mufu_ops / (ms[0] * 1e6 * clk[0]);                  // MUFU.EX2 lanes per clock per SM
    out8_host[1] = ffma_ops / (ms[1] * 1e6 * clk[1]);                  // FFMA lanes per clock per SM
    out8_host[2] = lds_bytes / (ms[2] * 1e6 * clk[2]);                 // LDS.128 bytes per clock per SM
    out8_host[3] = clk[0]; out8_host[4] = clk[1]; out8_host[5] = clk[2];   // SM clock (GHz) inside each kernel
    out8_host[6] = (double)sms;
    out8_host[7] = (double)(ms[0] + ms[1] + ms[2]);
    return NK_OK;
}
