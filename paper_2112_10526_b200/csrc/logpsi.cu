// Base log-amplitude  ln psi(s) = sum_i a_i s_i + sum_j ln cosh(theta_j)   (RBM: PAPER.md L575,
// ln cosh form Eq. (41)).  One warp per sample; theta comes from the fp32 contraction, every ln cosh term
// and both sums are evaluated in fp64 (at N = 1024 |ln psi| ~ 100, where one fp32 ulp is already 7.6e-6:
// DESIGN.md Q12), and ln 2 is applied once as M ln 2.
//   stable form (Q11): z <- z sign(Re z);  ln cosh z = z + log1p(exp(-2 z)) - ln 2
#include "nk_internal.h"

namespace nk {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <bool CPLX>
__global__ void __launch_bounds__(256)
logpsi_kernel(const int8_t* __restrict__ sigma, int64_t B, int N, int M, int M_pad, int M_eff,
              const float* __restrict__ theta, const float* __restrict__ a, void* __restrict__ logpsi_out,
              int out_f64, float* __restrict__ theta_out) {
    const int lane = threadIdx.x & 31;
    const int64_t s = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= B) return;
    const float* th = theta + s * M_eff;
    double re = 0.0, im = 0.0;
    for (int j = lane; j < M; j += 32) {
        if (!CPLX) {
            const float xf = th[j];
            if (theta_out) theta_out[s * M + j] = xf;
            const double t = fabs((double)xf);
            re += t + log1p(exp(-2.0 * t));
        } else {
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
        re = re - (double)M * 0.69314718055994530942 + are;
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
                          const void* a, void* logpsi_out, bool out_f64, void* theta_out, cudaStream_t st) {
    if (B <= 0) return cudaSuccess;
    const int wpb = 8;
    const unsigned grid = (unsigned)((B + wpb - 1) / wpb);
    if (dtype == NK_C64)
        logpsi_kernel<true><<<grid, wpb * 32, 0, st>>>(sigma, B, g.N, g.M, g.M_pad, g.M_eff, theta, (const float*)a,
                                                      logpsi_out, out_f64, (float*)theta_out);
    else
        logpsi_kernel<false><<<grid, wpb * 32, 0, st>>>(sigma, B, g.N, g.M, g.M_pad, g.M_eff, theta, (const float*)a,
                                                       logpsi_out, out_f64, (float*)theta_out);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
