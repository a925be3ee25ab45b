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
// entries of a warp's compaction list (2 KB; the list is evaluated and emptied whenever the next 256 elements might not
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

// ---- real parameters: one pass of a warp over its sample's row of theta -----------------------------------------------
// A lane takes 8 consecutive hidden units per step (two 128-bit loads; 16-byte stores into each operand segment).
// |theta| < 1 (99.8 % of config 5, theta ~ N(0, 0.32)): ln cosh and tanh from their fp32 polynomials (lncosh.cuh), the
// eight terms of a lane added in fp32 (each < 0.44; one rounding of ~3e-8 per group against a conversion and an fp64
// add per element) and the groups in fp64.  Larger arguments need the stable form in fp64 (exp + log1p, ~30 DFMA each)
// and the exponential form of tanh: a warp that holds one takes ONE warp-uniform branch in which the large arguments are
// compacted into a per-warp list in shared memory (ballot + popc), evaluated densely afterwards by drain() — not a
// divergent slow path per element.  (Until round 2 the polynomial stopped at |theta| = 1/2, an eighth of config 5's
// elements went through the list and every element paid for its ballot: 92 lane instructions per hidden unit.  An fp32
// expf / log1pf slow path was measured in round 1 and rejected: ln psi error 2.9e-6 -> 3.6e-6.)
// K = number of series terms (0: no operand rows): per hidden unit t = tanh(theta) as fp16 hi + lo, t^2 as fp16 and
// t^3 .. t^K as bf16 in segments of M_pad (series_tc.cu) — theta is read once for both.
struct BigList {
    float* big; int n; unsigned lt; int lane; double acc;
    __device__ __forceinline__ void drain() {               // the stable form, fp64, for the compacted large arguments
        __syncwarp();
        for (int k = lane; k < n; k += 32) {
            const double t = fabs((double)big[k]);
            acc += t + log1p(exp(-2.0 * t)) - 0.69314718055994530942;
        }
        __syncwarp();
        n = 0;
    }
    // x: the argument; l, t: its polynomial ln cosh and tanh, replaced when |x| >= 1 (warp-collective)
    __device__ __forceinline__ void fix(float x, float& l, float& t) {
        const bool is_big = fabsf(x) >= 1.f;
        const unsigned m = __ballot_sync(0xffffffffu, is_big);
        if (is_big) { big[n + __popc(m & lt)] = x; l = 0.f; t = tanh_exp_f(x); }
        n += __popc(m);
    }
};

template <int K>
__device__ __forceinline__ double logpsi_row_real(const float* __restrict__ th, int M, int M_pad,
                                                  float* __restrict__ theta_out_row, uint16_t* __restrict__ Ap_row,
                                                  BigList& bl) {
    double r0 = 0.0, r1 = 0.0;
    const int lane = bl.lane;
#pragma unroll 1
    for (int j0 = 0; j0 < M_pad; j0 += 256) {              // warp-uniform trip count (M_pad is a multiple of 128)
        const int j = j0 + lane * 8;
        const bool valid = j < M_pad;
        float x[8], l[8], t[8];
        *reinterpret_cast<float4*>(x) = valid ? *reinterpret_cast<const float4*>(th + j) : make_float4(0.f, 0.f, 0.f, 0.f);
        *reinterpret_cast<float4*>(x + 4) = valid ? *reinterpret_cast<const float4*>(th + j + 4) : make_float4(0.f, 0.f, 0.f, 0.f);
        if (theta_out_row) {
#pragma unroll
            for (int e = 0; e < 8; ++e) if (j + e < M) theta_out_row[j + e] = x[e];
        }
        float ax = 0.f;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            ax = fmaxf(ax, fabsf(x[e]));                   // (a NaN is skipped here and goes through the polynomials)
            l[e] = ln_cosh_unit_f(x[e]);
            t[e] = tanh_unit_f(x[e]);
        }
        if (__any_sync(0xffffffffu, ax >= 1.f)) {          // warp-uniform, rare at the configs' parameter scale
            if (bl.n + 256 > LOGPSI_LIST) bl.drain();
#pragma unroll
            for (int e = 0; e < 8; ++e) bl.fix(x[e], l[e], t[e]);
        }
        const float q = ((l[0] + l[1]) + (l[2] + l[3])) + ((l[4] + l[5]) + (l[6] + l[7]));
        if ((j0 >> 8) & 1) r1 += (double)q; else r0 += (double)q;
        if (K > 0 && valid) {
            uint16_t* out = Ap_row + j;
            uint32_t hi[4], lo[4], pw[4];
            float p[8];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const __half2 h = __floats2half2_rn(t[2 * e], t[2 * e + 1]);
                const float2 f = __half22float2(h);
                hi[e] = *reinterpret_cast<const uint32_t*>(&h);
                lo[e] = pack_h2(t[2 * e] - f.x, t[2 * e + 1] - f.y);
                p[2 * e] = t[2 * e] * t[2 * e]; p[2 * e + 1] = t[2 * e + 1] * t[2 * e + 1];
                pw[e] = pack_h2(p[2 * e], p[2 * e + 1]);
            }
            *reinterpret_cast<uint4*>(out) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
            *reinterpret_cast<uint4*>(out + M_pad) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            *reinterpret_cast<uint4*>(out + 2 * (size_t)M_pad) = make_uint4(pw[0], pw[1], pw[2], pw[3]);
#pragma unroll
            for (int k = 3; k <= K; ++k) {
#pragma unroll
                for (int e = 0; e < 8; ++e) p[e] *= t[e];
                *reinterpret_cast<uint4*>(out + (size_t)k * M_pad) =
                    make_uint4(pack_b2(p[0], p[1]), pack_b2(p[2], p[3]), pack_b2(p[4], p[5]), pack_b2(p[6], p[7]));
            }
        }
    }
    return r0 + r1;
}

// series_ctl / series_Ap (real parameters only, may be NULL): when *series_ctl = K > 0 the same pass over theta also
// writes the sample-side operand rows of the tensor-core series form.
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
        __shared__ float big_list[LOGPSI_WARPS_REAL][LOGPSI_LIST];
        BigList bl{big_list[threadIdx.x >> 5], 0, (1u << lane) - 1u, lane, 0.0};
        float* to = theta_out ? theta_out + s * M : nullptr;
        uint16_t* ap = K > 0 ? series_Ap + (size_t)s * SERIES_SEGS * M_pad : nullptr;
        double r;
        switch (K) {                                       // the power loop and its segment offsets are compile-time
            case 0: r = logpsi_row_real<0>(th, M, M_pad, to, ap, bl); break;
            case 2: r = logpsi_row_real<2>(th, M, M_pad, to, ap, bl); break;
            case 3: r = logpsi_row_real<3>(th, M, M_pad, to, ap, bl); break;
            case 4: r = logpsi_row_real<4>(th, M, M_pad, to, ap, bl); break;
            case 5: r = logpsi_row_real<5>(th, M, M_pad, to, ap, bl); break;
            default: r = logpsi_row_real<SERIES_K_MAX>(th, M, M_pad, to, ap, bl); break;
        }
        if (logpsi_out == nullptr) return;
        bl.drain();
        re = r + bl.acc;
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
