// Base log-amplitude  ln psi(s) = sum_i a_i s_i + sum_j ln cosh(theta_j)   (RBM: PAPER.md L575,
// ln cosh form Eq. (41)).  One warp per sample; theta comes from the fp32 contraction, every ln cosh term
// and both sums are evaluated in fp64 (at N = 1024 |ln psi| ~ 100, where one fp32 ulp is already 7.6e-6:
// DESIGN.md Q12), and ln 2 is applied once as M ln 2.
//   stable form (Q11): z <- z sign(Re z);  ln cosh z = z + log1p(exp(-2 z)) - ln 2
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "lncosh.cuh"
#include "nk_internal.h"

namespace nk {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

constexpr int LOGPSI_WARPS_REAL = 4;      // warps per block of the real kernel
// entries of a warp's compaction list (2 KB; the list is evaluated and emptied whenever the next 128 elements might not
// fit).  8 KB per block: small enough to run beside a CTA of the series form's tensor-core kernel (205 KB), which is
// what lets this pass over chunk c + 1 hide under the GEMM of chunk c (api.cu, the pipelined chunk loop)
constexpr int LOGPSI_LIST = 512;

__device__ __forceinline__ uint32_t pack_h2(float x, float y) {
    const __half2 h = __floats2half2_rn(x, y);
    return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ uint32_t pack_b2(float x, float y) {
    const __nv_bfloat162 h = __floats2bfloat162_rn(x, y);
    return *reinterpret_cast<const uint32_t*>(&h);
}

// series_ctl / series_Ap (real parameters only, may be NULL): when *series_ctl = K > 0 the same pass over theta also
// writes the sample-side operand rows of the tensor-core series form (series_tc.cu): per hidden unit t = tanh(theta)
// as fp16 hi + lo, t^2 as fp16 and t^3 .. t^K as bf16, in segments of M_pad — theta is read once for both.
template <bool CPLX>
__global__ void __launch_bounds__(256)
logpsi_kernel(const int8_t* __restrict__ sigma, int64_t B, int N, int M, int M_pad, int M_eff,
              const float* __restrict__ theta, const float* __restrict__ a, void* __restrict__ logpsi_out,
              int out_f64, float* __restrict__ theta_out, const unsigned* __restrict__ series_ctl,
              uint16_t* __restrict__ series_Ap) {
    const int lane = threadIdx.x & 31;
    const int64_t s = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= B) return;
    const float* th = theta + s * M_eff;
    double re = 0.0, im = 0.0;
    const int K = (!CPLX && series_ctl != nullptr) ? (int)*series_ctl : 0;
    if (logpsi_out == nullptr && K == 0) return;           // nothing asked of this launch
    if constexpr (!CPLX) {
        // 128-bit loads over the padded row (theta of a padded hidden unit is exactly 0 and contributes ln cosh 0 = 0),
        // four independent fp64 accumulators
        double r0 = 0.0, r1 = 0.0, r2 = 0.0, r3 = 0.0;
        // |t| < 1/2: the fp32 series, in place.  Larger arguments need the stable form in fp64 (exp + log1p: ~30 DFMA
        // each).  At config 5 theta ~ N(0, 0.32): an eighth of the elements, spread over every warp instruction, so a
        // branch per element made every warp pay the slow path 64 times per sample.  Instead the large arguments are
        // compacted into a per-warp list in shared memory (ballot + popc) and evaluated densely afterwards: ~8 slow
        // evaluations per lane and sample instead of 64, same fp64 formula.  (An fp32 expf / log1pf slow path was also
        // measured, 0.94 -> 0.53 ms per step, and rejected: ln psi error 2.9e-6 -> 3.6e-6.)
        __shared__ float big_list[LOGPSI_WARPS_REAL][LOGPSI_LIST];
        float* big = big_list[threadIdx.x >> 5];
        int n_big = 0;
        const unsigned lt = (1u << lane) - 1u;
        // (no branch on the ballot: with an eighth of the elements large, a warp almost always has one)
        auto take = [&](float x) -> float {
            const bool is_big = fabsf(x) >= 0.5f;
            const unsigned m = __ballot_sync(0xffffffffu, is_big);
            if (is_big) big[n_big + __popc(m & lt)] = x;
            n_big += __popc(m);
            return is_big ? 0.f : ln_cosh_small_f(x);
        };
        auto drain = [&]() {                                // the stable form, fp64, for the compacted large arguments
            __syncwarp();
            for (int k = lane; k < n_big; k += 32) {
                const double t = fabs((double)big[k]);
                r0 += t + log1p(exp(-2.0 * t)) - 0.69314718055994530942;
            }
            __syncwarp();
            n_big = 0;
        };
#pragma unroll 2
        for (int j = lane * 4; j < M_pad; j += 128) {
            if (n_big + 128 > LOGPSI_LIST) drain();         // warp-uniform
            const float4 x = *reinterpret_cast<const float4*>(th + j);
            if (theta_out) {
                if (j < M) theta_out[s * M + j] = x.x;
                if (j + 1 < M) theta_out[s * M + j + 1] = x.y;
                if (j + 2 < M) theta_out[s * M + j + 2] = x.z;
                if (j + 3 < M) theta_out[s * M + j + 3] = x.w;
            }
            // the four small-argument terms of a lane (each < 0.13) are added in fp32 first — one rounding of ~1e-8 per
            // group of four, 3e-7 over 2048 hidden units, against a conversion and an fp64 add per element
            const float q01 = take(x.x) + take(x.y), q23 = take(x.z) + take(x.w);
            if ((j >> 7) & 1) r1 += (double)(q01 + q23); else r0 += (double)(q01 + q23);
            if (K > 0) {
                const float t0 = tanh_f32(x.x), t1 = tanh_f32(x.y), t2 = tanh_f32(x.z), t3 = tanh_f32(x.w);   // < 2e-7 relative
                uint16_t* out = series_Ap + (size_t)s * SERIES_SEGS * M_pad + j;
                const __half2 h01 = __floats2half2_rn(t0, t1), h23 = __floats2half2_rn(t2, t3);
                const float2 f01 = __half22float2(h01), f23 = __half22float2(h23);
                *reinterpret_cast<uint2*>(out) = make_uint2(*reinterpret_cast<const uint32_t*>(&h01),
                                                            *reinterpret_cast<const uint32_t*>(&h23));
                *reinterpret_cast<uint2*>(out + M_pad) = make_uint2(pack_h2(t0 - f01.x, t1 - f01.y),
                                                                    pack_h2(t2 - f23.x, t3 - f23.y));
                float p0 = t0 * t0, p1 = t1 * t1, p2 = t2 * t2, p3 = t3 * t3;
                *reinterpret_cast<uint2*>(out + 2 * (size_t)M_pad) = make_uint2(pack_h2(p0, p1), pack_h2(p2, p3));
                for (int k = 3; k <= K; ++k) {
                    p0 *= t0; p1 *= t1; p2 *= t2; p3 *= t3;
                    *reinterpret_cast<uint2*>(out + (size_t)k * M_pad) = make_uint2(pack_b2(p0, p1), pack_b2(p2, p3));
                }
            }
        }
        if (logpsi_out == nullptr) return;
        drain();
        re = (r0 + r1) + (r2 + r3);
    }
    for (int j = lane; CPLX && j < M; j += 32) {
        {
            const float xf = th[j], yf = th[M_pad + j];
            if (theta_out) { theta_out[(s * M + j) * 2] = xf; theta_out[(s * M + j) * 2 + 1] = yf; }
            double x = xf, y = yf;
            if (x < 0.0) { x = -x; y = -y; }
            // w = exp(-2z);  log1p(w) = 0.5 log1p(wr (2 + wr) + wi^2) + i atan2(wi, 1 + wr)
            const double e = exp(-2.0 * x);
            double sn, cs;
            sincos(-2.0 * y, &sn, &cs);
            const double wr = e * cs, wi = e * sn;
            re += x + 0.5 * log1p(wr * (2.0 + wr) + wi * wi);
            im += y + atan2(wi, 1.0 + wr);
        }
    }
    re = warp_sum(re);
    if (CPLX) im = warp_sum(im);
    double are = 0.0, aim = 0.0;
    if (a != nullptr) {
        const int8_t* sg = sigma + s * N;
        for (int i = lane; i < N; i += 32) {
            const double si = (double)sg[i];
            if (!CPLX) are += si * (double)a[i];
            else { are += si * (double)a[2 * i]; aim += si * (double)a[2 * i + 1]; }
        }
        are = warp_sum(are);
        if (CPLX) aim = warp_sum(aim);
    }
    if (lane == 0) {
        re = re - (CPLX ? (double)M * 0.69314718055994530942 : 0.0) + are;
        im += aim;
        if (!CPLX) {
            if (out_f64) ((double*)logpsi_out)[s] = re; else ((float*)logpsi_out)[s] = (float)re;
        } else {
            if (out_f64) { ((double*)logpsi_out)[2 * s] = re; ((double*)logpsi_out)[2 * s + 1] = im; }
            else { ((float*)logpsi_out)[2 * s] = (float)re; ((float*)logpsi_out)[2 * s + 1] = (float)im; }
        }
    }
}

cudaError_t launch_logpsi(const int8_t* sigma, int64_t B, const Geometry& g, int dtype, const float* theta,
                          const void* a, void* logpsi_out, bool out_f64, void* theta_out, cudaStream_t st,
                          const unsigned* series_ctl, uint16_t* series_Ap) {
    if (B <= 0) return cudaSuccess;
    const int wpb = dtype == NK_C64 ? 8 : LOGPSI_WARPS_REAL;
    const unsigned grid = (unsigned)((B + wpb - 1) / wpb);
    if (dtype == NK_C64)
        logpsi_kernel<true><<<grid, wpb * 32, 0, st>>>(sigma, B, g.N, g.M, g.M_pad, g.M_eff, theta, (const float*)a,
                                                      logpsi_out, out_f64, (float*)theta_out, nullptr, nullptr);
    else
        logpsi_kernel<false><<<grid, wpb * 32, 0, st>>>(sigma, B, g.N, g.M, g.M_pad, g.M_eff, theta, (const float*)a,
                                                       logpsi_out, out_f64, (float*)theta_out, series_ctl,
                                                       series_Ap);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
