// Quantum geometric tensor times a vector for the RBM, on the fly.
//   G_ij = E[O_i^* O_j] - E[O_i^*] E[O_j]                                   PAPER.md Eq. (23)
//   w = (1/N_s) J v;   dw = w - <w>;   v~ = J^dagger dw                      Eq. (75) L2219 (QGTOnTheFly)
// With the closed-form RBM log-derivatives O_a = s, O_b = tanh(theta), O_W = tanh(theta) s^T (Eq. (13)):
//   (J v)_s = s . v_a + sum_j T_sj (v_b[j] + (V_W s)_j),
// so the first step is a second theta-shaped contraction Y = s V_W^T + v_b (the tcgen05 kernel of theta_tc.cu with
// V_W in the place of W) followed by one dot product per sample (this file); the last step J^dagger dw is exactly the
// force-vector contraction of gradient.cu with w in the place of E_loc (api.cu wires the two together).
#include "nk_internal.h"

namespace nk {

// w[s] = sigma_s . v_a + sum_j tanh(theta_sj) * Y_sj     (one warp per sample; fp64 accumulation, fixed order)
template <bool CPLX>
__global__ void qgt_w_kernel(const int8_t* __restrict__ sigma, int64_t nb, int N, int M, int M_pad, int M_eff,
                             const float* __restrict__ theta, const float* __restrict__ Y,
                             const float* __restrict__ v_a, float* __restrict__ w_out) {
    const int lane = threadIdx.x & 31;
    const int64_t s = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= nb) return;
    const float* th = theta + s * M_eff;
    const float* y = Y + s * M_eff;
    double re = 0.0, im = 0.0;
    for (int j = lane; j < M; j += 32) {
        if (!CPLX) {
            re += (double)(tanhf(th[j]) * y[j]);
        } else {
            // tanh(x + i y) = [sign(x)(1 - e^2) + i 2 e sin 2y] / (1 + e^2 + 2 e cos 2y),  e = exp(-2|x|)
            const float x = th[j], yy = th[M_pad + j];
            const float e = expf(-2.f * fabsf(x));
            float sn, cs;
            sincosf(2.f * yy, &sn, &cs);
            const float den = 1.f / (1.f + e * e + 2.f * e * cs);
            const float tr = copysignf((1.f - e) * (1.f + e), x) * den, ti = 2.f * e * sn * den;
            const float yr = y[j], yi = y[M_pad + j];
            re += (double)(tr * yr - ti * yi);
            im += (double)(tr * yi + ti * yr);
        }
    }
    if (v_a != nullptr) {
        const int8_t* sg = sigma + s * N;
        for (int k = lane; k < N; k += 32) {
            const double sk = (double)sg[k];
            if (!CPLX) re += sk * (double)v_a[k];
            else { re += sk * (double)v_a[2 * k]; im += sk * (double)v_a[2 * k + 1]; }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        re += __shfl_xor_sync(0xffffffffu, re, o);
        if (CPLX) im += __shfl_xor_sync(0xffffffffu, im, o);
    }
    if (lane == 0) {
        if (!CPLX) w_out[s] = (float)re;
        else { w_out[2 * s] = (float)re; w_out[2 * s + 1] = (float)im; }
    }
}

// out[i] += shift * v[i] over n floats (v may be nullptr: nothing to add)
__global__ void qgt_shift_kernel(float* __restrict__ out, const float* __restrict__ v, float shift, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        out[i] = fmaf(shift, v[i], out[i]);
}

cudaError_t launch_qgt_w(const Geometry& g, int dtype, const int8_t* sigma, int64_t nb, const float* theta,
                         const float* Y, const void* v_a, void* w_out, cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((nb + 7) / 8);
    if (dtype == NK_C64)
        qgt_w_kernel<true><<<grid, 256, 0, st>>>(sigma, nb, g.N, g.M, g.M_pad, g.M_eff, theta, Y, (const float*)v_a,
                                                 (float*)w_out);
    else
        qgt_w_kernel<false><<<grid, 256, 0, st>>>(sigma, nb, g.N, g.M, g.M_pad, g.M_eff, theta, Y, (const float*)v_a,
                                                  (float*)w_out);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_qgt_shift(void* out, const void* v, double shift, int64_t n_floats, cudaStream_t st) {
    if (out == nullptr || v == nullptr || shift == 0.0 || n_floats <= 0) return cudaSuccess;
    int64_t blocks = (n_floats + 255) / 256;
    if (blocks > 2368) blocks = 2368;
    qgt_shift_kernel<<<(unsigned)blocks, 256, 0, st>>>((float*)out, (const float*)v, (float)shift, n_floats);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
