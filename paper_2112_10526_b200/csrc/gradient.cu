// Force vector / energy gradient of the RBM.
//   O_i(s) = d ln psi(s) / d theta_i                      PAPER.md Eq. (13)
//   f~_i   = E[O_i^* (H~ - E[H~])]                        Eq. (14), Eq. (26)
//   grad   = 2 Re f~ (real parameters) | f~ (complex, holomorphic)   Eq. (15)/(16) L664-668, Eq. (27)/(28) L918-922
// RBM closed form: O_a = s, O_b = tanh(theta), O_W = tanh(theta) s^T, so with w_s = (E_loc(s) - mean) / B
//   g_a[k] = sum_s s_k w_s,  g_b[j] = sum_s conj(T_sj) w_s,  g_W[j][k] = sum_s conj(T_sj) w_s s_k   (x2, real part, for real parameters).
// g_W is a dense contraction over the samples -- tensor-core work: per chunk the values v_sj = conj(T_sj) w_s are split
// on three fixed-point bf16 grids (as W is in theta_tc.cu; sigma = +-1 is exact), written k-contiguous (k = sample),
// and contracted with sigma^T by the same tcgen05 kernel, accumulating [N][M_eff] in fp32 across chunks.
// g_a and g_b are fp64 column sums with a fixed order (bit-reproducible).

#include "lncosh.cuh"
#include "nk_internal.h"

namespace nk {

// w_s = (E_loc(s) - mean) / B in fp64 -> fp32 (complex: both parts)
__device__ __forceinline__ void sample_weight(const float* __restrict__ eloc, const double* __restrict__ stats,
                                              int64_t s, double inv_B, bool cplx, float& wr, float& wi) {
    if (cplx) {
        wr = (float)(((double)eloc[2 * s] - stats[0]) * inv_B);
        wi = (float)(((double)eloc[2 * s + 1] - stats[1]) * inv_B);
    } else {
        wr = (float)(((double)eloc[s] - stats[0]) * inv_B);
        wi = 0.f;
    }
}

// theta[s][.] -> v[s][.] in place (complex: plane 0 = Re v, plane 1 = Im v), and max |v| as float bits
template <bool CPLX>
__global__ void grad_tv_kernel(const float* theta_in, float* theta, int64_t nb, int M, int M_pad, int M_eff,
                               const float* __restrict__ eloc, const double* __restrict__ stats, double inv_B,
                               float real_scale, unsigned* __restrict__ absmax) {
    unsigned m = 0;
    for (int64_t s = blockIdx.y; s < nb; s += gridDim.y) {
    float wr, wi;
    sample_weight(eloc, stats, s, inv_B, CPLX, wr, wi);
    float* row = theta + s * M_eff;
    const float* rin = theta_in + s * M_eff;          // may alias row (in place) or be a cached theta
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < M_pad; j += gridDim.x * blockDim.x) {
        if (!CPLX) {
            const float v = (j < M) ? real_scale * tanhf(rin[j]) * wr : 0.f;
            row[j] = v;
            m = max(m, __float_as_uint(fabsf(v)));
        } else {
            float vr = 0.f, vi = 0.f;
            if (j < M) {
                // tanh(x + i y) = [sign(x)(1 - e^2) + i 2 e sin 2y] / (1 + e^2 + 2 e cos 2y),  e = exp(-2|x|)
                const float x = rin[j], y = rin[M_pad + j];
                const float e = expf(-2.f * fabsf(x));
                float sn, cs;
                sincosf(2.f * y, &sn, &cs);
                const float den = 1.f / (1.f + e * e + 2.f * e * cs);
                const float tr = copysignf((1.f - e) * (1.f + e), x) * den, ti = 2.f * e * sn * den;
                vr = tr * wr + ti * wi;                   // conj(T) * w
                vi = tr * wi - ti * wr;
            }
            row[j] = vr; row[M_pad + j] = vi;
            m = max(m, max(__float_as_uint(fabsf(vr)), __float_as_uint(fabsf(vi))));
        }
    }
    }
    // one atomic per block (all blocks hit the same address)
    __shared__ unsigned wmax[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = max(m, wmax[w]);
        if (m) atomicMax(absmax, m);
    }
}

// Column sums in fp64 with a fixed order (bit-reproducible): slabs of GRAD_SLAB samples are summed in parallel into
// part[slab][col], then one thread per column adds the slabs in order onto the running accumulator.
constexpr int GRAD_SLAB = 128;

// part[slab][me] = sum_{s in slab} v[s][me]
__global__ void grad_colsum_partial_kernel(const float* __restrict__ v, int64_t nb, int M_eff,
                                           double* __restrict__ part) {
    const int me = blockIdx.x * blockDim.x + threadIdx.x;
    if (me >= M_eff) return;
    const int64_t s0 = (int64_t)blockIdx.y * GRAD_SLAB;
    const int64_t s1 = (s0 + GRAD_SLAB < nb) ? s0 + GRAD_SLAB : nb;
    double acc = 0.0;
    for (int64_t s = s0; s < s1; ++s) acc += (double)v[s * M_eff + me];
    part[(size_t)blockIdx.y * M_eff + me] = acc;
}

// part[slab][plane * N + k] = sum_{s in slab} sigma[s][k] w_s[plane]   (x2 for real parameters); blockDim.x == GRAD_SLAB:
// thread t first forms the weight of sample s0 + t once for the whole block
__global__ void grad_a_partial_kernel(const int8_t* __restrict__ sigma, int64_t nb, int N,
                                      const float* __restrict__ eloc, const double* __restrict__ stats, double inv_B,
                                      int cplx, double real_scale, double* __restrict__ part,
                                      unsigned* __restrict__ wmax_bits) {
    __shared__ double wr_s[GRAD_SLAB], wi_s[GRAD_SLAB];
    const int64_t s0 = (int64_t)blockIdx.y * GRAD_SLAB;
    const int64_t s1 = (s0 + GRAD_SLAB < nb) ? s0 + GRAD_SLAB : nb;
    {
        float wr = 0.f, wi = 0.f;
        if (s0 + threadIdx.x < s1) sample_weight(eloc, stats, s0 + threadIdx.x, inv_B, cplx != 0, wr, wi);
        wr_s[threadIdx.x] = (cplx ? 1.0 : real_scale) * (double)wr;
        wi_s[threadIdx.x] = (double)wi;
        if (wmax_bits != nullptr && blockIdx.x == 0) {        // max_s |real_scale w_s| >= max |v_sj| since |tanh| <= 1
            unsigned m = __float_as_uint(fabsf((float)real_scale * wr));
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
            if ((threadIdx.x & 31) == 0 && m) atomicMax(wmax_bits, m);
        }
    }
    __syncthreads();
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    double ar = 0.0, ai = 0.0;
    const int n = (int)(s1 - s0);
    const int8_t* col = sigma + s0 * N + k;
    if (cplx) {
        for (int t = 0; t < n; ++t) {
            const double sg = (double)col[(size_t)t * N];
            ar += sg * wr_s[t];
            ai += sg * wi_s[t];
        }
    } else {
#pragma unroll 8
        for (int t = 0; t < n; ++t) ar += (double)col[(size_t)t * N] * wr_s[t];
    }
    part[(size_t)blockIdx.y * 2 * N + k] = ar;
    part[(size_t)blockIdx.y * 2 * N + N + k] = ai;
}

// acc[c] (+)= sum_slab part[slab][c] in a fixed order: block = 32 columns x blockDim.y <= 32 slab ranges; range r adds
// its contiguous share of the slabs in order, then the range sums are added in order
// scale_io (optional): [0] = max |v| bound as float bits (in) -> [2] = 2^(23 - ex), [3] = q = 2^(ex - 23) as floats (out)
__global__ void grad_slab_reduce_kernel(const double* __restrict__ part, int n_slabs, int n_cols,
                                        double* __restrict__ acc, int first, unsigned* scale_io) {
    if (scale_io != nullptr && blockIdx.x == 0 && threadIdx.x == 0 && threadIdx.y == 0) {
        const float vmax = __uint_as_float(scale_io[0]);
        int ex = -100;
        if (vmax > 0.f) {
            frexpf(vmax, &ex);
            if (ldexpf(vmax, 23 - ex) > 8355000.f) ++ex;      // keep the top digit inside [-128, 127]
            if (ex < -100) ex = -100;                         // keep 2^(23 - ex) finite
        }
        scale_io[2] = __float_as_uint(ldexpf(1.f, 23 - ex));
        scale_io[3] = __float_as_uint(ldexpf(1.f, ex - 23));
        if (scale_io[0] >= 0x7f800000u) {                     // a NaN / Inf local energy or mean: poison the block
            scale_io[2] = 0u;                                 // (zero digits, q = NaN: q D is NaN, Q14)
            scale_io[3] = 0x7fc00000u;
        }
    }
    __shared__ double sh[32][32];
    const int c = blockIdx.x * 32 + threadIdx.x;
    const int per = (n_slabs + (int)blockDim.y - 1) / (int)blockDim.y;
    const int sl0 = threadIdx.y * per, sl1 = min(n_slabs, sl0 + per);
    double a = 0.0;
    if (c < n_cols)
        for (int sl = sl0; sl < sl1; ++sl) a += part[(size_t)sl * n_cols + c];
    sh[threadIdx.y][threadIdx.x] = a;
    __syncthreads();
    if (threadIdx.y == 0 && c < n_cols) {
        double t = first ? 0.0 : acc[c];
        for (int r = 0; r < (int)blockDim.y; ++r) t += sh[r][threadIdx.x];
        acc[c] = t;
    }
}

// TwT[digit][me][s] (int8, k-contiguous, leading dimension ld bytes) from v[s][me]: rint(v / q) = d2 2^16 + d1 2^8 + d0
// with balanced base-256 digits and q a power of two tied to max|v| (the split of theta_tc.cu's split_w_i8_kernel);
// rows s in [nb, k_len) are zero; the scale q goes behind the three planes (byte offset 3 M_eff ld)
__global__ void grad_split_T_kernel(const float* __restrict__ v, int64_t nb, int k_len, int M_eff, int ld,
                                    const unsigned* __restrict__ absmax_bits, int8_t* __restrict__ TwT) {
    __shared__ float tile[32][33];
    const float vmax = __uint_as_float(*absmax_bits);
    int ex = -100;
    if (vmax > 0.f) {
        frexpf(vmax, &ex);
        if (ldexpf(vmax, 23 - ex) > 8355000.f) ++ex;      // keep the top digit inside [-128, 127]
    }
    const bool poison = *absmax_bits >= 0x7f800000u;      // NaN / Inf among the v: zero digits, q = NaN (Q14)
    const float sc = poison ? 0.f : ldexpf(1.f, 23 - ex);
    const int s0 = blockIdx.x * 32, m0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int64_t s = s0 + r;
        tile[r][threadIdx.x] = (s < nb) ? v[s * M_eff + m0 + threadIdx.x] : 0.f;
    }
    __syncthreads();
    const size_t plane = (size_t)M_eff * ld;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int me = m0 + r, s = s0 + threadIdx.x;
        if (s >= k_len) continue;
        const int I = poison ? 0 : (int)rintf(tile[threadIdx.x][r] * sc);
        const int d0 = ((I + 128) & 255) - 128;
        const int I1 = (I - d0) >> 8;
        const int d1 = ((I1 + 128) & 255) - 128;
        const size_t o = (size_t)me * ld + s;
        TwT[o] = (int8_t)((I1 - d1) >> 8);
        TwT[plane + o] = (int8_t)d1;
        TwT[2 * plane + o] = (int8_t)d0;
    }
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0 && threadIdx.y == 0)
        *reinterpret_cast<float*>(TwT + 3 * plane) = poison ? __int_as_float(0x7fc00000) : ldexpf(1.f, ex - 23);
}

// Real parameters, one pass: theta[s][.] -> v = real_scale tanh(theta) w_s -> the three int8 digit planes of
// grad_split_T_kernel (same layout, same digits) and the fp64 column sums of the slab, without storing v.  The scale
// is tied to max_s |real_scale w_s| >= max |v| (|tanh| <= 1; left by grad_a_partial_kernel), not to max |v| itself.
// Tile = GRAD_SLAB samples x 32 hidden units per block of 256 threads; blockIdx.x = slab * (M_eff / 32) + column group:
// blocks in flight together cover whole rows of theta (DRAM page locality).
__global__ void __launch_bounds__(256)
grad_tv_split_kernel(const float* __restrict__ theta, int64_t nb, int k_len, int M, int M_eff, int ld,
                     const float* __restrict__ eloc, const double* __restrict__ stats, double inv_B, float real_scale,
                     const unsigned* __restrict__ scale_io, int8_t* __restrict__ TwT, double* __restrict__ part) {
    __shared__ float w_s[GRAD_SLAB];                              // real_scale w_s / q: v / q = tanh(theta) * this
    __shared__ int dq[3][32][GRAD_SLAB / 4 + 1];                  // [digit][column][4 samples per word], stride 33 words
    __shared__ int cs[8][32];
    const float sc = __uint_as_float(scale_io[2]), q = __uint_as_float(scale_io[3]);
    const int n_cg = M_eff >> 5;
    const int slab = blockIdx.x / n_cg;
    const int64_t s0 = (int64_t)slab * GRAD_SLAB;
    const int m0 = (blockIdx.x - slab * n_cg) * 32;
    const int n_rows = (int)min((int64_t)GRAD_SLAB, nb - s0);
    if (threadIdx.x < GRAD_SLAB) {
        float wr = 0.f, wi;
        if ((int)threadIdx.x < n_rows) sample_weight(eloc, stats, s0 + threadIdx.x, inv_B, false, wr, wi);
        w_s[threadIdx.x] = real_scale * wr * sc;                  // two exact scalings (1 or 2, a power of two)
    }
    __syncthreads();
    const int c = threadIdx.x & 31, r = threadIdx.x >> 5;
    const float* col = theta + s0 * M_eff + m0 + c;
    const int lim = (m0 + c < M) ? n_rows : 0;
    const bool whole = n_rows == GRAD_SLAB && m0 + 32 <= M;       // block-uniform: no predicates on the loads
    const float* ptr = col + (unsigned)(4 * r * M_eff);
    int acc = 0;                                                  // sum of the slab's integers: |I| <= 2^23, 128 of them
#pragma unroll
    for (int p = 0; p < GRAD_SLAB / 32; ++p) {
        const int sl = 4 * (r + 8 * p);                           // this thread: samples sl .. sl + 3 of column c
        float th[4];
        if (whole) {
#pragma unroll
            for (int i = 0; i < 4; ++i) th[i] = ptr[i * M_eff];
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) th[i] = (sl + i < lim) ? ptr[i * M_eff] : 0.f;
        }
        ptr += 32 * M_eff;
        // rint(v / q) = d2 2^16 + d1 2^8 + d0 with balanced digits: the low bytes of I, (I + 128) >> 8 and of that again
        // |theta| < 1 almost everywhere at the configs' parameter scale: the polynomial alone, unless a lane of the warp
        // holds a larger argument (a NaN passes the max and propagates through the polynomial)
        float tv[4];
        const float amax = fmaxf(fmaxf(fabsf(th[0]), fabsf(th[1])), fmaxf(fabsf(th[2]), fabsf(th[3])));
        if (__any_sync(0xffffffffu, amax >= 1.f)) {
#pragma unroll
            for (int i = 0; i < 4; ++i) tv[i] = tanh_f32(th[i]);
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) tv[i] = tanh_unit_f(th[i]);
        }
        unsigned w0 = 0, w1 = 0, w2 = 0;
#define NK_DIGITS(i, sel)                                                         \
        {                                                                         \
            const int I = __float2int_rn(tv[i] * w_s[sl + i]);                    \
            const int I1 = (I + 128) >> 8;                                        \
            const int I2 = (I1 + 128) >> 8;                                       \
            acc += I;                                                             \
            w0 = __byte_perm(w0, (unsigned)I, sel);                               \
            w1 = __byte_perm(w1, (unsigned)I1, sel);                              \
            w2 = __byte_perm(w2, (unsigned)I2, sel);                              \
        }
        NK_DIGITS(0, 0x3214) NK_DIGITS(1, 0x3240) NK_DIGITS(2, 0x3410) NK_DIGITS(3, 0x4210)
#undef NK_DIGITS
        dq[0][c][r + 8 * p] = (int)w2;
        dq[1][c][r + 8 * p] = (int)w1;
        dq[2][c][r + 8 * p] = (int)w0;
    }
    cs[r][c] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        int t = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) t += cs[k][threadIdx.x];
        part[(size_t)slab * M_eff + m0 + threadIdx.x] = (double)t * (double)q;
    }
    const size_t plane = (size_t)M_eff * ld;
    int8_t* out = TwT + (size_t)m0 * ld + s0 + 4 * c;             // k_len is a multiple of GRAD_SLAB: whole rows of the tile
#pragma unroll
    for (int row = r; row < 96; row += 8) {
        const int d = row >> 5, j = row & 31;
        *reinterpret_cast<int*>(out + d * plane + (size_t)j * ld) = dq[d][j][c];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) *reinterpret_cast<float*>(TwT + 3 * plane) = q;
}

// sigT[k][s] = sigma[s][k] (int8), zero for s in [nb, k_len).  Tile = 128 samples x 128 sites per block of 256 threads:
// a thread takes 4 sites x 4 samples (one 32-bit word from each of 4 rows), transposes the 4 x 4 bytes in registers
// (byte permutes) and leaves 4 words, one per site, in a shared tile [site][sample word ^ site word] (XOR swizzle: both
// the writes and the row reads are bank-conflict-free); rows of 128 samples go out as one 128-B line per warp.
// Needs N % 4 == 0 and 4-B aligned rows for the word loads; other shapes take the byte path.
__global__ void __launch_bounds__(256)
grad_sigma_T_kernel(const int8_t* __restrict__ sigma, int64_t nb, int k_len, int N, int ld, int8_t* __restrict__ sigT) {
    __shared__ unsigned tile[128][32];
    const int64_t s0 = (int64_t)blockIdx.x * 128;
    const int k0 = blockIdx.y * 128;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool words = (N & 3) == 0 && ((uintptr_t)sigma & 3) == 0;
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const int a = warp + 8 * p;                               // samples s0 + 4a .. 4a + 3, sites k0 + 4 lane .. + 3
        unsigned r[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int64_t s = s0 + 4 * a + i;
            const int k = k0 + 4 * lane;
            r[i] = 0;
            if (s < nb) {
                if (words && k + 3 < N) r[i] = *reinterpret_cast<const unsigned*>(sigma + s * N + k);
                else
                    for (int b = 0; b < 4; ++b)
                        if (k + b < N) r[i] |= (unsigned)(uint8_t)sigma[s * N + k + b] << (8 * b);
            }
        }
        // 4 x 4 byte transpose: t[b] = bytes b of r[0..3]
        const unsigned x0 = __byte_perm(r[0], r[1], 0x5140), x1 = __byte_perm(r[0], r[1], 0x7362);
        const unsigned y0 = __byte_perm(r[2], r[3], 0x5140), y1 = __byte_perm(r[2], r[3], 0x7362);
        tile[4 * lane + 0][a ^ lane] = __byte_perm(x0, y0, 0x5410);
        tile[4 * lane + 1][a ^ lane] = __byte_perm(x0, y0, 0x7632);
        tile[4 * lane + 2][a ^ lane] = __byte_perm(x1, y1, 0x5410);
        tile[4 * lane + 3][a ^ lane] = __byte_perm(x1, y1, 0x7632);
    }
    __syncthreads();
    const int n_words = (int)min((int64_t)128, (int64_t)k_len - s0) >> 2;     // k_len is a multiple of 128: 32
    for (int row = warp; row < 128; row += 8) {
        const int k = k0 + row;
        if (k < N && lane < n_words)
            *reinterpret_cast<unsigned*>(sigT + (size_t)k * ld + s0 + 4 * lane) = tile[row][lane ^ (row >> 2)];
    }
}

// g_W[j][k] = Gacc[k][j] (complex: (Gacc[k][j], Gacc[k][M_pad + j]) interleaved); 32x32 tiles through shared memory
__global__ void grad_finalize_W_kernel(const float* __restrict__ Gacc, int N, int M, int M_pad, int M_eff, int cplx,
                                       float* __restrict__ gW) {
    __shared__ float tr[32][33], ti[32][33];
    const int j0 = blockIdx.x * 32, k0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int k = k0 + r, j = j0 + threadIdx.x;
        const bool ok = k < N && j < M;
        tr[r][threadIdx.x] = ok ? Gacc[(size_t)k * M_eff + j] : 0.f;
        ti[r][threadIdx.x] = (ok && cplx) ? Gacc[(size_t)k * M_eff + M_pad + j] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int j = j0 + r, k = k0 + threadIdx.x;
        if (j < M && k < N) {
            if (cplx) {
                gW[((size_t)j * N + k) * 2] = tr[threadIdx.x][r];
                gW[((size_t)j * N + k) * 2 + 1] = ti[threadIdx.x][r];
            } else gW[(size_t)j * N + k] = tr[threadIdx.x][r];
        }
    }
}

__global__ void grad_finalize_ab_kernel(const double* __restrict__ ga_acc, const double* __restrict__ gb_acc, int N,
                                        int M, int M_pad, int cplx, float* __restrict__ ga, float* __restrict__ gb) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (ga != nullptr && i < N) {
        if (cplx) { ga[2 * i] = (float)ga_acc[i]; ga[2 * i + 1] = (float)ga_acc[N + i]; }
        else ga[i] = (float)ga_acc[i];
    }
    if (gb != nullptr && i < M) {
        if (cplx) { gb[2 * i] = (float)gb_acc[i]; gb[2 * i + 1] = (float)gb_acc[M_pad + i]; }
        else gb[i] = (float)gb_acc[i];
    }
}

int grad_slab() { return GRAD_SLAB; }

// phase: 0 = the whole chunk on `st`; 1 = only the part that does not read theta (sample weights into grad_a, the
// power-of-two scale of the split, the transposed spins); 2 = the rest.  nk_energy_gradient runs phase 1 on a second
// stream beside the theta contraction of the same chunk (71 us of small kernels at config 5) and phase 2 after both.
cudaError_t launch_gradient_chunk(const Geometry& g, int dtype, const int8_t* sigma, int64_t nb, int64_t B_total,
                                  const void* eloc, const double* stats, const GradWs& w, int first_chunk,
                                  float real_scale, cudaStream_t st, const float* theta_in, const void* sigT_ready,
                                  int phase) {
    if (nb <= 0) return cudaSuccess;
    const bool cplx = dtype == NK_C64;
    const double inv_B = 1.0 / (double)B_total;
    const int k_len = (int)((nb + 127) / 128 * 128);
    const int n_slabs = (int)((nb + GRAD_SLAB - 1) / GRAD_SLAB);
    const dim3 red_block(32, n_slabs >= 128 ? 32 : 8);
    cudaError_t e;
    if (phase != 2) {
        e = cudaMemsetAsync(w.absmax, 0, sizeof(unsigned), st);
        if (e != cudaSuccess) return e;
        // (grad_a's partial sums go to the upper part of `part`'s allocation when the phases run side by side: see carve_grad)
        grad_a_partial_kernel<<<dim3((g.N + 127) / 128, n_slabs), 128, 0, st>>>(
            sigma, nb, g.N, (const float*)eloc, stats, inv_B, cplx, (double)real_scale, w.part_a,
            cplx ? nullptr : w.absmax);
        grad_slab_reduce_kernel<<<(2 * g.N + 31) / 32, red_block, 0, st>>>(w.part_a, n_slabs, 2 * g.N, w.ga_acc,
                                                                       first_chunk, cplx ? nullptr : w.absmax);
        count_launch(2);
        if (sigT_ready == nullptr) {
            grad_sigma_T_kernel<<<dim3(k_len / 128, (g.N + 127) / 128), 256, 0, st>>>(sigma, nb, k_len, g.N, w.ld,
                                                                                         (int8_t*)w.sigT);
            count_launch();
        }
        e = cudaGetLastError();
        if (e != cudaSuccess || phase == 1) return e;
    }
    const float* th_in = theta_in ? theta_in : w.theta;
    if (!cplx) {
        // k_len / GRAD_SLAB == n_slabs (both round nb up to 128)
        grad_tv_split_kernel<<<(unsigned)n_slabs * (unsigned)(g.M_eff / 32), 256, 0, st>>>(
            th_in, nb, k_len, g.M, g.M_eff, w.ld, (const float*)eloc, stats, inv_B, real_scale, w.absmax,
            (int8_t*)w.TwT, w.part);
        count_launch(2);
    } else {
        dim3 gtv((g.M_pad + 255) / 256, (unsigned)(nb < 1184 ? nb : 1184));
        grad_tv_kernel<true><<<gtv, 256, 0, st>>>(th_in, w.theta, nb, g.M, g.M_pad, g.M_eff, (const float*)eloc, stats,
                                                  inv_B, real_scale, w.absmax);
        grad_colsum_partial_kernel<<<dim3((g.M_eff + 127) / 128, n_slabs), 128, 0, st>>>(w.theta, nb, g.M_eff, w.part);
        grad_split_T_kernel<<<dim3(k_len / 32, g.M_eff / 32), dim3(32, 8), 0, st>>>(
            w.theta, nb, k_len, g.M_eff, w.ld, w.absmax, (int8_t*)w.TwT);
        count_launch(4);
    }
    grad_slab_reduce_kernel<<<(g.M_eff + 31) / 32, red_block, 0, st>>>(w.part, n_slabs, g.M_eff, w.gb_acc, first_chunk,
                                                                   nullptr);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return launch_tc_gemm_pieces(sigT_ready ? sigT_ready : (const void*)w.sigT, g.N, w.TwT, g.M_eff, w.ld, k_len, w.Gacc,
                                 first_chunk ? 0 : 1, st);
}

// sigT[k][s] = sigma[s][k] (int8, zero padded to a multiple of 128 samples) for one chunk (what launch_gradient_chunk builds itself unless given sigT_ready)
cudaError_t launch_sigma_T(const int8_t* sigma, int64_t nb, int N, int ld, void* sigT, cudaStream_t st) {
    const int k_len = (int)((nb + 127) / 128 * 128);
    grad_sigma_T_kernel<<<dim3(k_len / 128, (N + 127) / 128), 256, 0, st>>>(sigma, nb, k_len, N, ld, (int8_t*)sigT);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_gradient_finalize(const Geometry& g, int dtype, const GradWs& w, void* grad_a, void* grad_b,
                                     void* grad_W, cudaStream_t st) {
    const int cplx = dtype == NK_C64;
    grad_finalize_W_kernel<<<dim3((g.M + 31) / 32, (g.N + 31) / 32), dim3(32, 8), 0, st>>>(
        w.Gacc, g.N, g.M, g.M_pad, g.M_eff, cplx, (float*)grad_W);
    const int n = g.N > g.M ? g.N : g.M;
    grad_finalize_ab_kernel<<<(n + 127) / 128, 128, 0, st>>>(w.ga_acc, w.gb_acc, g.N, g.M, g.M_pad, cplx,
                                                            (float*)grad_a, (float*)grad_b);
    count_launch(2);
    return cudaGetLastError();
}

}  // namespace nk
