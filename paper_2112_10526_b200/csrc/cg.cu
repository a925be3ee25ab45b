// Conjugate gradients for the stochastic-reconfiguration system:
//   sum_j (G_ij + eps delta_ij) delta_j = f_i        PAPER.md Eq. (25) L886 with Eq. (30)/(31) L961-967;
// "a JAX-compatible linear solver (the default is jax.scipy.sparse.linalg.cg)" L969.  G + eps is Hermitian positive
// definite, so plain CG applies to real and complex (holomorphic) parameters alike, with the real part of the
// Hermitian inner product.  The matrix is never formed: every iteration is one nk_qgt_matvec (api.cu).  Vectors are
// packed [a | b | W] as floats (complex: interleaved), scalars live on the device in fp64; reductions have a fixed
// order (bit-reproducible).
#include "nk_internal.h"

namespace nk {

constexpr int CG_BLOCKS = 592, CG_THREADS = 256;

// part[block] = sum over the block's strided share of x_i y_i  (floats; for interleaved complex this is Re <x, y>)
__global__ void cg_dot_partial_kernel(const float* __restrict__ x, const float* __restrict__ y, int64_t n,
                                      double* __restrict__ part) {
    __shared__ double sh[CG_THREADS / 32];
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        acc += (double)x[i] * (double)y[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < CG_THREADS / 32; ++w) t += sh[w];
        part[blockIdx.x] = t;
    }
}
// one warp: lane l adds the partials l, l + 32, ... in order, then a butterfly over the lanes (a fixed order)
__global__ void cg_dot_final_kernel(const double* __restrict__ part, int n_part, double* __restrict__ out) {
    double t = 0.0;
    for (int i = threadIdx.x; i < n_part; i += 32) t += part[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (threadIdx.x == 0) *out = t;
}

// alpha = rr / pAp;  x += alpha p;  r -= alpha Ap       (alpha = 0 when pAp <= 0: converged or breakdown)
__global__ void cg_step_kernel(float* __restrict__ x, float* __restrict__ r, const float* __restrict__ p,
                               const float* __restrict__ Ap, int64_t n, const double* __restrict__ rr,
                               const double* __restrict__ pAp) {
    const double d = *pAp;
    const float alpha = d > 0.0 ? (float)(*rr / d) : 0.f;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        x[i] = fmaf(alpha, p[i], x[i]);
        r[i] = fmaf(-alpha, Ap[i], r[i]);
    }
}
// beta = rr_new / rr_old;  p = r + beta p
__global__ void cg_dir_kernel(float* __restrict__ p, const float* __restrict__ r, int64_t n,
                              const double* __restrict__ rr_new, const double* __restrict__ rr_old) {
    const double d = *rr_old;
    const float beta = d > 0.0 ? (float)(*rr_new / d) : 0.f;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        p[i] = fmaf(beta, p[i], r[i]);
}

static unsigned cg_grid(int64_t n) {
    const int64_t b = (n + CG_THREADS - 1) / CG_THREADS;
    return (unsigned)(b < CG_BLOCKS ? (b > 0 ? b : 1) : CG_BLOCKS);
}

int cg_partials() { return CG_BLOCKS; }

cudaError_t launch_cg_dot(const float* x, const float* y, int64_t n, double* part, double* out, cudaStream_t st) {
    const unsigned g = cg_grid(n);
    cg_dot_partial_kernel<<<g, CG_THREADS, 0, st>>>(x, y, n, part);
    cg_dot_final_kernel<<<1, 32, 0, st>>>(part, (int)g, out);
    count_launch(2);
    return cudaGetLastError();
}
cudaError_t launch_cg_step(float* x, float* r, const float* p, const float* Ap, int64_t n, const double* rr,
                           const double* pAp, cudaStream_t st) {
    cg_step_kernel<<<cg_grid(n), CG_THREADS, 0, st>>>(x, r, p, Ap, n, rr, pAp);
    count_launch();
    return cudaGetLastError();
}
cudaError_t launch_cg_dir(float* p, const float* r, int64_t n, const double* rr_new, const double* rr_old,
                          cudaStream_t st) {
    cg_dir_kernel<<<cg_grid(n), CG_THREADS, 0, st>>>(p, r, n, rr_new, rr_old);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
