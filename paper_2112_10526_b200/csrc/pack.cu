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
#include "lncosh.cuh"
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
    ri.i = -1; ri.j = -1; ri.coef = 0.f; ri.jdiag = 0.f; ri.a2_re = 0.f; ri.a2_im = 0.f; ri.c2_re = 0.f; ri.c2_im = 0.f;
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

namespace nk {

// ---- product-form tables -------------------------------------------------------------
// cosh(theta + s d) / cosh(theta) = cosh(d) (1 + s tanh(theta) tanh(d)),  s = +-1,  so with tau = tanh(d)
//   psi'/psi = e^{s da} * prod_j cosh(d_j) * prod_j (1 + s t_j tau_j),   t = tanh(theta).
// Ttab [n_rows_pad][M_eff]: tau for row r and hidden unit j (complex: plane 0 = Re tau, plane 1 = Im tau),
// d = 2 (W[:,i] - W[:,j]) (exchange) or 2 W[:,k] (flip) — the same rows as Dtab, in natural units.
__global__ void ttab_kernel(const float* __restrict__ Wt, const int32_t* __restrict__ bonds, int kind, int n_rows,
                            int M_pad, int M_eff, int cplx, float* __restrict__ Ttab,
                            unsigned* __restrict__ taumax_bits) {
    const int r = blockIdx.y;
    unsigned tmax = 0;
    int i = -1, j = -1;
    if (r < n_rows) {
        if (kind == NK_HEISENBERG) { i = bonds[2 * r]; j = bonds[2 * r + 1]; }
        else i = r;
    }
    for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < M_pad; m += gridDim.x * blockDim.x) {
        float tr = 0.f, ti = 0.f;
        if (i >= 0) {
            float x = Wt[(size_t)i * M_eff + m], y = cplx ? Wt[(size_t)i * M_eff + M_pad + m] : 0.f;
            if (j >= 0) { x -= Wt[(size_t)j * M_eff + m]; if (cplx) y -= Wt[(size_t)j * M_eff + M_pad + m]; }
            x *= 2.f; y *= 2.f;
            if (!cplx) tr = tanhf(x);
            else {
                // tanh(x + i y) = [sign(x)(1 - e^2) + i 2 e sin 2y] / (1 + e^2 + 2 e cos 2y),  e = exp(-2|x|)
                const float e = expf(-2.f * fabsf(x));
                float sn, cs;
                sincosf(2.f * y, &sn, &cs);
                const float den = 1.f / (1.f + e * e + 2.f * e * cs);
                tr = copysignf((1.f - e) * (1.f + e), x) * den;
                ti = 2.f * e * sn * den;
            }
        }
        Ttab[(size_t)r * M_eff + m] = tr;
        if (cplx) Ttab[(size_t)r * M_eff + M_pad + m] = ti;
        tmax = max(tmax, __float_as_uint(fabsf(tr)));
    }
    if (taumax_bits != nullptr) {                            // max |tau| of the table (real parameters), float bits
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tmax = max(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
        if ((threadIdx.x & 31) == 0 && tmax) atomicMax(taumax_bits, tmax);
    }
}

// rows[r].c2_re / c2_im = sum_j ln cosh(d_j) (log2 units / radians), fp64 sum in a fixed order: one warp per row,
// lane-strided partial sums, butterfly.  ln cosh(x+iy) = |x| - ln 2 + (1/2) ln(1 + e^2 + 2 e cos 2y)
//                                                       + i atan2(sign(x)(1-e) sin y, (1+e) cos y),  e = exp(-2|x|).
__global__ void rowc_kernel(const float* __restrict__ Wt, int n_rows, int M_pad, int M_eff, int cplx,
                            RowInfo* __restrict__ rows) {
    const int r = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (r >= n_rows) return;
    const int i = rows[r].i, j = rows[r].j;
    double sre = 0.0, sim = 0.0;
    if (i >= 0) {
        for (int m = lane; m < M_pad; m += 32) {
            double x = (double)Wt[(size_t)i * M_eff + m], y = cplx ? (double)Wt[(size_t)i * M_eff + M_pad + m] : 0.0;
            if (j >= 0) {
                x -= (double)Wt[(size_t)j * M_eff + m];
                if (cplx) y -= (double)Wt[(size_t)j * M_eff + M_pad + m];
            }
            x *= 2.0; y *= 2.0;
            const double e = exp(-2.0 * fabs(x));
            if (!cplx) sre += fabs(x) + log1p(e) - 0.6931471805599453;
            else {
                double sn, cs;
                sincos(y, &sn, &cs);
                sre += fabs(x) - 0.6931471805599453 + 0.5 * log1p(e * e + 2.0 * e * (2.0 * cs * cs - 1.0));
                sim += atan2(copysign((1.0 - e) * sn, x * sn), (1.0 + e) * cs);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sre += __shfl_xor_sync(0xffffffffu, sre, o);
        sim += __shfl_xor_sync(0xffffffffu, sim, o);
    }
    if (lane == 0) {
        rows[r].c2_re = (float)(sre * 1.4426950408889634);
        rows[r].c2_im = (float)remainder(sim, 6.283185307179586);
    }
}

// Real parameters: the three per-row passes over d = 2 (W[:,i] - W[:,j]) in one — tau = tanh d into Ttab, the row
// constant sum_j ln cosh d_j (fp32 series below 1/2, the stable fp64 form above, fp64 sum in a fixed order) into
// rows[r].c2_re, max |tau| into *taumax_bits and, when series_ctl is given, the row sums of |tau|^3 .. |tau|^(K_MAX+1)
// that bound the remainder of the tensor-core series form (series_tc.cu) into its control block.  One block per row.
__global__ void __launch_bounds__(256)
rowtab_real_kernel(const float* __restrict__ Wt, const int32_t* __restrict__ bonds, int kind, int n_rows, int M_pad,
                   int M_eff, float* __restrict__ Ttab, RowInfo* __restrict__ rows, unsigned* __restrict__ taumax_bits,
                   unsigned* __restrict__ series_ctl) {
    const int r = blockIdx.x;
    int i = -1, j = -1;
    if (r < n_rows) {
        if (kind == NK_HEISENBERG) { i = bonds[2 * r]; j = bonds[2 * r + 1]; }
        else i = r;
    }
    float* out = Ttab + (size_t)r * M_eff;
    if (i < 0) {                                               // padded row of the table
        for (int m = threadIdx.x; m < M_pad; m += blockDim.x) out[m] = 0.f;
        return;
    }
    const float* wi = Wt + (size_t)i * M_eff;
    const float* wj = j >= 0 ? Wt + (size_t)j * M_eff : nullptr;
    double lc = 0.0;
    float pw[SERIES_K_MAX - 1];
#pragma unroll
    for (int k = 0; k < SERIES_K_MAX - 1; ++k) pw[k] = 0.f;
    unsigned tmax = 0;
    for (int m = threadIdx.x; m < M_pad; m += blockDim.x) {
        float x = wi[m];
        if (wj != nullptr) x -= wj[m];
        x *= 2.f;
        const float t = tanhf(x);
        out[m] = t;
        const float at = fabsf(t);
        tmax = max(tmax, __float_as_uint(at));
        float p = at * at;
#pragma unroll
        for (int k = 0; k < SERIES_K_MAX - 1; ++k) { p *= at; pw[k] += p; }
        if (fabsf(x) < 0.5f) lc += (double)ln_cosh_small_f(x);
        else {
            const double ax = fabs((double)x);
            lc += ax + log1p(exp(-2.0 * ax)) - 0.6931471805599453;
        }
    }
    __shared__ double red_d[8];
    __shared__ float red_f[8][SERIES_K_MAX - 1];
    __shared__ unsigned red_u[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lc += __shfl_xor_sync(0xffffffffu, lc, o);
        tmax = max(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
#pragma unroll
        for (int k = 0; k < SERIES_K_MAX - 1; ++k) pw[k] += __shfl_xor_sync(0xffffffffu, pw[k], o);
    }
    if (lane == 0) {
        red_d[warp] = lc; red_u[warp] = tmax;
#pragma unroll
        for (int k = 0; k < SERIES_K_MAX - 1; ++k) red_f[warp][k] = pw[k];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        unsigned u = 0;
        for (int w = 0; w < 8; ++w) { t += red_d[w]; u = max(u, red_u[w]); }
        rows[r].c2_re = (float)(t * 1.4426950408889634);
        rows[r].c2_im = 0.f;
        if (taumax_bits != nullptr && u) atomicMax(taumax_bits, u);
    }
    if (series_ctl != nullptr && threadIdx.x < SERIES_K_MAX - 1) {
        float t = 0.f;
        for (int w = 0; w < 8; ++w) t += red_f[w][threadIdx.x];
        if (t != t) t = __int_as_float(0x7f800000);           // a NaN in the table must not look like a small bound
        atomicMax(&series_ctl[4 + 3 + threadIdx.x], __float_as_uint(t));
    }
}

// Fills `tab` with Ttab and rows[].c2_*; call after launch_pack.  taumax_bits (optional): max |tau| as float bits.
// series_ctl (optional, real parameters): the zeroed control block of the series form, which receives the row sums of
// |tau|^p (see rowtab_real_kernel).
cudaError_t launch_pack_product(const Operator* op, const Geometry& g, int dtype, const float* Wt, float* tab,
                                RowInfo* rows, cudaStream_t st, unsigned* taumax_bits, unsigned* series_ctl) {
    const int cplx = dtype == NK_C64;
    if (taumax_bits != nullptr) {
        cudaError_t e = cudaMemsetAsync(taumax_bits, 0, sizeof(unsigned), st);
        if (e != cudaSuccess) return e;
    }
    if (!cplx) {
        rowtab_real_kernel<<<g.n_rows_pad, 256, 0, st>>>(Wt, op->d_bonds, op->kind, g.n_rows, g.M_pad, g.M_eff, tab, rows,
                                                         taumax_bits, series_ctl);
        count_launch();
        return cudaGetLastError();
    }
    dim3 gd((g.M_pad + 255) / 256, g.n_rows_pad);
    ttab_kernel<<<gd, 256, 0, st>>>(Wt, op->d_bonds, op->kind, g.n_rows, g.M_pad, g.M_eff, cplx, tab, taumax_bits);
    rowc_kernel<<<(g.n_rows_pad + 7) / 8, 256, 0, st>>>(Wt, g.n_rows, g.M_pad, g.M_eff, cplx, rows);
    count_launch(2);
    return cudaGetLastError();
}

}  // namespace nk
