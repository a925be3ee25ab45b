// Parameter packing, redone on every nk_local_energy / nk_rbm_logpsi call (W changes every VMC step):
//   Wg   [M_eff][N]   real planes of W with zero rows up to M_pad (complex: plane 0 = Re, plane 1 = Im)
//   bg   [M_eff]
//   Wt   [N][M_eff]   transpose of Wg (column k of W as a contiguous row)
//   Dtab [n_rows_pad][M_eff]   the rows the fused kernel streams:  theta_s' = theta_s + s * Dtab[r]
//        Heisenberg row r = bond (i,j):  2 KAPPA (W[:,i] - W[:,j])   (Im plane: 2 (..), radians)
//        Ising      row r = site k:      2 KAPPA  W[:,k]
//   rows [n_rows_pad]  RowInfo (sites, matrix element, visible-bias exponent)
// theta' = theta - 2 s_k W[:,k] for a flipped site k (BASELINE.json north_star (3)); an exchange of antiparallel
// spins i,j flips both: theta' = theta - 2 s_i (W[:,i] - W[:,j]).
#include "nk_internal.h"

namespace nk {

__global__ void pack_wg_kernel(const float* __restrict__ W, const float* __restrict__ b, int N, int M, int M_pad,
                               int M_eff, int cplx, float* __restrict__ Wg, float* __restrict__ bg) {
    const int me = blockIdx.y;
    const int plane = me / M_pad, m = me - plane * M_pad;
    const bool live = m < M;
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < N; k += gridDim.x * blockDim.x) {
        float v = 0.f;
        if (live) v = cplx ? W[((size_t)m * N + k) * 2 + plane] : W[(size_t)m * N + k];
        Wg[(size_t)me * N + k] = v;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        float v = 0.f;
        if (live && b != nullptr) v = cplx ? b[2 * m + plane] : b[m];
        bg[me] = v;
    }
}

// Wt[k][me] = Wg[me][k], 32x32 tiles through shared memory (both sides coalesced).
__global__ void transpose_kernel(const float* __restrict__ Wg, int M_eff, int N, float* __restrict__ Wt) {
    __shared__ float tile[32][33];
    const int k0 = blockIdx.x * 32, m0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int m = m0 + r, k = k0 + threadIdx.x;
        tile[r][threadIdx.x] = (m < M_eff && k < N) ? Wg[(size_t)m * N + k] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int k = k0 + r, m = m0 + threadIdx.x;
        if (k < N && m < M_eff) Wt[(size_t)k * M_eff + m] = tile[threadIdx.x][r];
    }
}

__global__ void dtab_kernel(const float* __restrict__ Wt, const int32_t* __restrict__ bonds, int kind, int n_rows,
                            int M_pad, int M_eff, float* __restrict__ Dtab) {
    const int r = blockIdx.y;
    int i = -1, j = -1;
    if (r < n_rows) {
        if (kind == NK_HEISENBERG) { i = bonds[2 * r]; j = bonds[2 * r + 1]; }
        else i = r;
    }
    for (int me = blockIdx.x * blockDim.x + threadIdx.x; me < M_eff; me += gridDim.x * blockDim.x) {
        float v = 0.f;
        if (i >= 0) {
            v = Wt[(size_t)i * M_eff + me];
            if (j >= 0) v -= Wt[(size_t)j * M_eff + me];
            v *= (me < M_pad) ? 2.f * KAPPA : 2.f;
        }
        Dtab[(size_t)r * M_eff + me] = v;
    }
}

__global__ void rowinfo_kernel(const int32_t* __restrict__ bonds, const int32_t* __restrict__ colors,
                               const float* __restrict__ Jf, float h, int kind, unsigned flags, int n_rows,
                               int n_rows_pad, const float* __restrict__ a, int cplx, RowInfo* __restrict__ rows) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rows_pad) return;
    RowInfo ri;
    ri.i = -1; ri.j = -1; ri.coef = 0.f; ri.jdiag = 0.f; ri.a2_re = 0.f; ri.a2_im = 0.f; ri.pad0 = 0; ri.pad1 = 0;
    if (r < n_rows) {
        float are = 0.f, aim = 0.f;
        if (kind == NK_HEISENBERG) {
            ri.i = bonds[2 * r]; ri.j = bonds[2 * r + 1];
            const float J = Jf[colors[r]];
            ri.jdiag = J;
            ri.coef = (flags & NK_FLAG_MARSHALL) ? -2.f * J : 2.f * J;
            if (a != nullptr) {
                if (cplx) { are = a[2 * ri.i] - a[2 * ri.j]; aim = a[2 * ri.i + 1] - a[2 * ri.j + 1]; }
                else are = a[ri.i] - a[ri.j];
            }
        } else {
            ri.i = r;
            ri.coef = -h;
            if (a != nullptr) {
                if (cplx) { are = a[2 * r]; aim = a[2 * r + 1]; }
                else are = a[r];
            }
        }
        ri.a2_re = 2.f * LOG2E * are;
        ri.a2_im = 2.f * aim;
    }
    rows[r] = ri;
}

cudaError_t launch_pack_gemm_only(const Geometry& g, int dtype, const void* W, const void* b, float* Wg, float* bg,
                                  cudaStream_t st) {
    dim3 grid((g.N + 255) / 256, g.M_eff);
    if (grid.x > 64) grid.x = 64;
    pack_wg_kernel<<<grid, 256, 0, st>>>((const float*)W, (const float*)b, g.N, g.M, g.M_pad, g.M_eff,
                                          dtype == NK_C64, Wg, bg);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_pack(const Operator* op, const Geometry& g, int dtype, const void* W, const void* a, const void* b,
                        float* Wg, float* bg, float* Wt, float* Dtab, RowInfo* rows, cudaStream_t st) {
    cudaError_t e = launch_pack_gemm_only(g, dtype, W, b, Wg, bg, st);
    if (e != cudaSuccess) return e;
    transpose_kernel<<<dim3((g.N + 31) / 32, (g.M_eff + 31) / 32), dim3(32, 8), 0, st>>>(Wg, g.M_eff, g.N, Wt);
    dim3 gd((g.M_eff + 255) / 256, g.n_rows_pad);
    dtab_kernel<<<gd, 256, 0, st>>>(Wt, op->d_bonds, op->kind, g.n_rows, g.M_pad, g.M_eff, Dtab);
    rowinfo_kernel<<<(g.n_rows_pad + 127) / 128, 128, 0, st>>>(op->d_bonds, op->d_colors, op->d_Jf, (float)op->h,
                                                               op->kind, op->flags, g.n_rows, g.n_rows_pad,
                                                               (const float*)a, dtype == NK_C64, rows);
    count_launch(3);
    return cudaGetLastError();
}

}  // namespace nk

namespace nk {

// Table for the Metropolis sampler (sampler.cu): Wg, bg, Wt as above and one row of Dtab per proposal —
// pairs_dev == nullptr: row k = 2 KAPPA W[:,k] (single flip of site k); else row c = 2 KAPPA (W[:,i_c] - W[:,j_c])
// for the exchange pair c = (i_c, j_c).  No row padding.
cudaError_t launch_pack_table(const Geometry& g, int dtype, const void* W, const void* b, const int32_t* pairs_dev,
                              int n_rows, float* Wg, float* bg, float* Wt, float* Dtab, cudaStream_t st) {
    cudaError_t e = launch_pack_gemm_only(g, dtype, W, b, Wg, bg, st);
    if (e != cudaSuccess) return e;
    transpose_kernel<<<dim3((g.N + 31) / 32, (g.M_eff + 31) / 32), dim3(32, 8), 0, st>>>(Wg, g.M_eff, g.N, Wt);
    dim3 gd((g.M_eff + 255) / 256, n_rows);
    dtab_kernel<<<gd, 256, 0, st>>>(Wt, pairs_dev, pairs_dev ? NK_HEISENBERG : NK_ISING, n_rows, g.M_pad, g.M_eff, Dtab);
    count_launch(2);
    return cudaGetLastError();
}

}  // namespace nk
