// Fused incremental local-energy kernel (SURVEY.md §8 a1 + a4): for every sample, enumerate the connected
// configurations from the device bond table (never materialising sigma'), update theta by one row of the
// bond-difference table, and accumulate  E_loc(s) = H_ss + sum_s' H_ss' psi(s')/psi(s)   (Eq. (12)).
//
// Mapping: one warp owns one sample; lane l holds hidden units {128 v + 4 l + c : v < V, c < 4} of theta in
// registers.  A CTA = FW = 16 warps (4 per SM sub-partition, so the four MUFU pipes carry equal load; 16 x 32 x
// 128 registers = the whole register file).  Each CTA owns a contiguous range of samples and works through it in
// rounds of 16 (the last round may be partial).  Tiles of the table Dtab flow through a shared-memory ring filled
// by 1-D bulk async copies (TMA engine) that complete on mbarriers; there is no producer warp: the LAST warp to
// finish a stage (a shared-memory arrival counter) re-arms that stage's barrier and issues the next copy.  Every
// warp walks the same tiles, tests its own sample's bonds (spins bit-packed in shared memory, one ballot per
// tile), and for each active row does, per hidden unit,
//      theta_s' = theta_s + s D                      (theta_s = 2 log2(e) theta, s = -sigma_i)
//      e'  = 2^(-|theta_s'|) = exp(-2|theta'|)       (1 MUFU)
//      P  *= (1 + e')                                (FMA)
//      acc += |theta_s'| - |theta_s|                 (per-term difference: no cancellation of O(100) sums)
// which is the stable form ln cosh x = |x| + ln(1 + e^{-2|x|}) - ln 2 with the logarithm hoisted out of the sum
// over hidden units (sum_j ln(1+e_j) = ln prod_j (1+e_j)) and cancelled against the final exp:
//      psi'/psi = 2^(acc/2 + s a2) * prod_j (1+e'_j) / prod_j (1+e_j).
// Complex parameters: cosh(x+iy) = (e^{|x|}/2) [(1+e) cos u + i (1-e) sin u], u = sign(x) y, and the product runs
// over complex factors.
#include <type_traits>

#include "nk_internal.h"
#include "ptx_helpers.cuh"

namespace nk {

constexpr int FW = 16;                       // warps (samples in flight) per CTA
constexpr int FTHREADS = FW * 32;

struct FusedParams {
    const int8_t* sigma;
    int64_t B;
    int N, n_words;                          // n_words = ceil(N / 32): bit-packed spins per sample
    const float* theta;
    int M_pad, M_eff;
    const float* Dtab;
    const RowInfo* rows;
    int n_rows, tile_rows, n_tiles, stages;
    const int32_t* bonds;
    const int32_t* colors;
    const float* Jf;
    int n_bonds, kind;
    float* eloc;
    int64_t per_cta;                         // samples per CTA (contiguous range)
};

__device__ __forceinline__ float warp_sum_f(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_prod_f(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v *= __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- per-row inner loops ---------------------------------------------------------------------------------
template <int V>
struct RealState {
    float4 th[V];      // theta_s
    float qinv;        // 1 / prod_{j in lane} (1 + e_j)

    __device__ __forceinline__ void load(const float* __restrict__ row, int lane, int /*M_pad*/) {
        float p0 = 1.f, p1 = 1.f, p2 = 1.f, p3 = 1.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            float4 t = *reinterpret_cast<const float4*>(row + (v * 32 + lane) * 4);
            t.x *= KAPPA; t.y *= KAPPA; t.z *= KAPPA; t.w *= KAPPA;
            th[v] = t;
            p0 = fmaf(p0, ex2_approx(-fabsf(t.x)), p0);
            p1 = fmaf(p1, ex2_approx(-fabsf(t.y)), p1);
            p2 = fmaf(p2, ex2_approx(-fabsf(t.z)), p2);
            p3 = fmaf(p3, ex2_approx(-fabsf(t.w)), p3);
        }
        qinv = 1.f / ((p0 * p1) * (p2 * p3));
    }
    // this lane's share of psi'/psi for one row: r = prod_{j in lane} (1+e'_j)/(1+e_j), acc = sum_j (|x'_j| - |x_j|)
    __device__ __forceinline__ void partial(const float* __restrict__ drow, int lane, float s, float& r,
                                            float& acc) const {
        float p0 = 1.f, p1 = 1.f, p2 = 1.f, p3 = 1.f, acc0 = 0.f, acc1 = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 d = *reinterpret_cast<const float4*>(drow + (v * 32 + lane) * 4);
            const float4 t = th[v];
            const float x0 = fmaf(s, d.x, t.x), x1 = fmaf(s, d.y, t.y);
            const float x2 = fmaf(s, d.z, t.z), x3 = fmaf(s, d.w, t.w);
            p0 = fmaf(p0, ex2_approx(-fabsf(x0)), p0);
            p1 = fmaf(p1, ex2_approx(-fabsf(x1)), p1);
            p2 = fmaf(p2, ex2_approx(-fabsf(x2)), p2);
            p3 = fmaf(p3, ex2_approx(-fabsf(x3)), p3);
            acc0 += fabsf(x0) - fabsf(t.x);
            acc1 += fabsf(x1) - fabsf(t.y);
            acc0 += fabsf(x2) - fabsf(t.z);
            acc1 += fabsf(x3) - fabsf(t.w);
        }
        r = ((p0 * p1) * (p2 * p3)) * qinv;
        acc = acc0 + acc1;
    }
};

// One pending row of a sample: lane partials plus the row's scalars.  Rows are reduced across the warp two at a
// time: after the first exchange (lane ^ 16) the lower half-warp owns row A and the upper half row B, so the
// five butterfly levels cost 10 shuffles per PAIR of rows instead of 10 per row, and the two rows' serial
// reduction latencies overlap.
struct RowPartR {
    float r, acc, ex, coef;     // ex = s * a2 (visible-bias exponent, log2 units)
};
__device__ __forceinline__ float finish_pair(const RowPartR& A, const RowPartR& B, int lane) {
    const bool up = (lane & 16) != 0;
    float rk = up ? B.r : A.r, ak = up ? B.acc : A.acc;
    const float rs = up ? A.r : B.r, as = up ? A.acc : B.acc;
    rk *= __shfl_xor_sync(0xffffffffu, rs, 16);
    ak += __shfl_xor_sync(0xffffffffu, as, 16);
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) {
        rk *= __shfl_xor_sync(0xffffffffu, rk, o);
        ak += __shfl_xor_sync(0xffffffffu, ak, o);
    }
    const float ex = up ? B.ex : A.ex, c = up ? B.coef : A.coef;
    return c * (rk * ex2_approx(fmaf(0.5f, ak, ex)));   // lower half: row A's term, upper half: row B's
}
__device__ __forceinline__ float finish_single(const RowPartR& A) {
    const float r = warp_prod_f(A.r), acc = warp_sum_f(A.acc);
    return A.coef * (r * ex2_approx(fmaf(0.5f, acc, A.ex)));
}

template <int V>
struct CplxState {
    float4 tx[V], ty[V];   // Re theta_s (scaled), Im theta (radians)
    float qr, qi;          // 1 / prod_{j in lane} f_j

    static __device__ __forceinline__ void factor(float x, float y, float& p, float& q) {
        const float e = ex2_approx(-fabsf(x));
        float sn, cs;
        __sincosf(y, &sn, &cs);
        p = fmaf(e, cs, cs);                      // (1+e) cos y
        q = fmaf(-e, sn, sn);                     // (1-e) sin y
        q = __int_as_float(__float_as_int(q) ^ (__float_as_int(x) & 0x80000000));   // times sign(x)
    }
    static __device__ __forceinline__ void cmul(float& ar, float& ai, float br, float bi) {
        const float r = fmaf(ar, br, -ai * bi), i = fmaf(ar, bi, ai * br);
        ar = r; ai = i;
    }
    __device__ __forceinline__ void load(const float* __restrict__ row, int lane, int M_pad) {
        float ar = 1.f, ai = 0.f, br = 1.f, bi = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            float4 x = *reinterpret_cast<const float4*>(row + (v * 32 + lane) * 4);
            const float4 y = *reinterpret_cast<const float4*>(row + M_pad + (v * 32 + lane) * 4);
            x.x *= KAPPA; x.y *= KAPPA; x.z *= KAPPA; x.w *= KAPPA;
            tx[v] = x; ty[v] = y;
            float p, q;
            factor(x.x, y.x, p, q); cmul(ar, ai, p, q);
            factor(x.y, y.y, p, q); cmul(br, bi, p, q);
            factor(x.z, y.z, p, q); cmul(ar, ai, p, q);
            factor(x.w, y.w, p, q); cmul(br, bi, p, q);
        }
        cmul(ar, ai, br, bi);
        const float inv = 1.f / fmaf(ar, ar, ai * ai);
        qr = ar * inv; qi = -ai * inv;
    }
    // this lane's share: (ar + i ai) = prod_{j in lane} f'_j / f_j, acc = sum_j (|x'_j| - |x_j|)
    __device__ __forceinline__ void partial(const float* __restrict__ drow, int lane, int M_pad, float s, float& ar,
                                            float& ai, float& acc) const {
        float br = 1.f, bi = 0.f;
        ar = 1.f; ai = 0.f; acc = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 dx = *reinterpret_cast<const float4*>(drow + (v * 32 + lane) * 4);
            const float4 dy = *reinterpret_cast<const float4*>(drow + M_pad + (v * 32 + lane) * 4);
            const float4 x = tx[v], y = ty[v];
            float p, q;
            const float x0 = fmaf(s, dx.x, x.x), x1 = fmaf(s, dx.y, x.y);
            const float x2 = fmaf(s, dx.z, x.z), x3 = fmaf(s, dx.w, x.w);
            factor(x0, fmaf(s, dy.x, y.x), p, q); cmul(ar, ai, p, q);
            factor(x1, fmaf(s, dy.y, y.y), p, q); cmul(br, bi, p, q);
            factor(x2, fmaf(s, dy.z, y.z), p, q); cmul(ar, ai, p, q);
            factor(x3, fmaf(s, dy.w, y.w), p, q); cmul(br, bi, p, q);
            acc += (fabsf(x0) - fabsf(x.x)) + (fabsf(x1) - fabsf(x.y));
            acc += (fabsf(x2) - fabsf(x.z)) + (fabsf(x3) - fabsf(x.w));
        }
        cmul(ar, ai, br, bi);
        cmul(ar, ai, qr, qi);
    }
    static __device__ __forceinline__ void cmul_pub(float& ar, float& ai, float br, float bi) { cmul(ar, ai, br, bi); }
};

struct RowPartC {
    float ar, ai, acc, ex_re, ex_im, coef;   // ex_re = s a2_re (log2 units), ex_im = s a2_im (radians)
};
__device__ __forceinline__ void cmul_f(float& ar, float& ai, float br, float bi) {
    const float r = fmaf(ar, br, -ai * bi), i = fmaf(ar, bi, ai * br);
    ar = r; ai = i;
}
__device__ __forceinline__ void finish_c(float ar, float ai, float acc, float ex_re, float ex_im, float c,
                                         float& out_re, float& out_im) {
    const float mag = c * ex2_approx(fmaf(0.5f, acc, ex_re));
    float sn, cs;
    __sincosf(ex_im, &sn, &cs);
    cmul_f(ar, ai, mag * cs, mag * sn);
    out_re = ar; out_im = ai;
}
__device__ __forceinline__ void finish_pair_c(const RowPartC& A, const RowPartC& B, int lane, float& out_re,
                                              float& out_im) {
    const bool up = (lane & 16) != 0;
    float kr = up ? B.ar : A.ar, ki = up ? B.ai : A.ai, ka = up ? B.acc : A.acc;
    const float sr = up ? A.ar : B.ar, si = up ? A.ai : B.ai, sa = up ? A.acc : B.acc;
    cmul_f(kr, ki, __shfl_xor_sync(0xffffffffu, sr, 16), __shfl_xor_sync(0xffffffffu, si, 16));
    ka += __shfl_xor_sync(0xffffffffu, sa, 16);
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) {
        const float orr = __shfl_xor_sync(0xffffffffu, kr, o), oi = __shfl_xor_sync(0xffffffffu, ki, o);
        cmul_f(kr, ki, orr, oi);
        ka += __shfl_xor_sync(0xffffffffu, ka, o);
    }
    finish_c(kr, ki, ka, up ? B.ex_re : A.ex_re, up ? B.ex_im : A.ex_im, up ? B.coef : A.coef, out_re, out_im);
}
__device__ __forceinline__ void finish_single_c(const RowPartC& A, float& out_re, float& out_im) {
    float ar = A.ar, ai = A.ai, acc = A.acc;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float orr = __shfl_xor_sync(0xffffffffu, ar, o), oi = __shfl_xor_sync(0xffffffffu, ai, o);
        cmul_f(ar, ai, orr, oi);
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
    }
    finish_c(ar, ai, acc, A.ex_re, A.ex_im, A.coef, out_re, out_im);
}

// ---- kernel ----------------------------------------------------------------------------------------------
template <int V, bool CPLX>
constexpr int min_blocks() { return ((CPLX ? 8 : 4) * V <= 16) ? 2 : 1; }

__device__ __forceinline__ void issue_tile(const FusedParams& p, uint32_t ring_u32, uint32_t full0, int stage,
                                           int tile, uint32_t stage_bytes) {
    mbar_arrive_expect_tx(full0 + 8 * stage, stage_bytes);
    bulk_g2s(ring_u32 + stage * stage_bytes, p.Dtab + (size_t)tile * p.tile_rows * p.M_eff, stage_bytes,
             full0 + 8 * stage);
}

template <int V, bool CPLX>
__global__ void __launch_bounds__(FTHREADS, (min_blocks<V, CPLX>())) fused_eloc_kernel(const FusedParams p) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t stage_bytes = (uint32_t)p.tile_rows * p.M_eff * 4u;
    float* ring = reinterpret_cast<float*>(smem);
    uint32_t* bits_all = reinterpret_cast<uint32_t*>(smem + (size_t)p.stages * stage_bytes);
    uint64_t* bars = reinterpret_cast<uint64_t*>(bits_all + (size_t)FW * p.n_words);   // full[stages]
    int* done_cnt = reinterpret_cast<int*>(bars + p.stages);                           // arrivals per stage
    const uint32_t full0 = smem_u32(bars), ring_u32 = smem_u32(ring);

    // this CTA's contiguous sample range, processed in rounds of FW samples
    const int64_t first = (int64_t)blockIdx.x * p.per_cta;
    const int64_t last = (first + p.per_cta < p.B) ? first + p.per_cta : p.B;
    const int64_t n_rounds = (last > first) ? (last - first + FW - 1) / FW : 0;
    const int64_t total_tiles = n_rounds * p.n_tiles;

    if (threadIdx.x == 0) {
        for (int s = 0; s < p.stages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            done_cnt[s] = 0;
        }
        mbar_fence_init();
        for (int s = 0; s < p.stages && s < total_tiles; ++s)          // prime the ring
            issue_tile(p, ring_u32, full0, s, s % p.n_tiles, stage_bytes);
    }
    __syncthreads();

    // ===== consumers =====
    uint32_t* bits = bits_all + warp * p.n_words;     // bit i set <=> sigma_i = -1
    auto spin_bit = [&](int i) -> int { return (int)((bits[i >> 5] >> (i & 31)) & 1u); };
    int stage = 0;
    uint32_t parity = 0;
    int64_t g = 0;                                    // running tile counter of this CTA
    typename std::conditional<CPLX, CplxState<V>, RealState<V>>::type st;

    for (int64_t rnd = 0; rnd < n_rounds; ++rnd) {
        const int64_t sample = first + rnd * FW + warp;
        const bool valid = sample < last;
        const int64_t srow = valid ? sample : first;  // idle warps of a partial round shadow a valid row
        __syncwarp();
        {
            const int8_t* sp = p.sigma + srow * p.N;
            for (int wi = lane; wi < p.n_words; wi += 32) {
                uint32_t w = 0;
                const int base = wi * 32;
                const int cnt = (p.N - base < 32) ? (p.N - base) : 32;
                for (int t = 0; t < cnt; ++t) w |= (uint32_t)(sp[base + t] < 0) << t;
                bits[wi] = w;
            }
        }
        st.load(p.theta + srow * p.M_eff, lane, p.M_pad);
        __syncwarp();

        // e_u*: terms identical on all lanes (single rows); e_h*: half-warp-specific terms (paired rows)
        float diag = 0.f, e_ure = 0.f, e_uim = 0.f, e_hre = 0.f, e_him = 0.f;
        bool pending = false;                         // warp-uniform: one row waits for a partner
        typename std::conditional<CPLX, RowPartC, RowPartR>::type pend;
        if (p.kind == NK_ISING) {
            for (int b = lane; b < p.n_bonds; b += 32) {
                const int i = p.bonds[2 * b], j = p.bonds[2 * b + 1];
                const float J = p.Jf[p.colors[b]];
                diag += (spin_bit(i) != spin_bit(j)) ? -J : J;
            }
        }
        for (int t = 0; t < p.n_tiles; ++t) {
            // enumerate this tile's rows for this sample: lane r <-> row t*tile_rows + r
            bool active = false;
            float sgn = 0.f, coef = 0.f, a2re = 0.f, a2im = 0.f;
            if (lane < p.tile_rows) {
                const RowInfo ri = p.rows[t * p.tile_rows + lane];
                if (ri.i >= 0) {
                    const int bi = spin_bit(ri.i);
                    const int bj = (ri.j >= 0) ? spin_bit(ri.j) : (bi ^ 1);
                    active = valid && (bi != bj);
                    diag += (bi != bj) ? -ri.jdiag : ri.jdiag;
                    sgn = bi ? 1.f : -1.f;            // s = -sigma_i
                    coef = ri.coef; a2re = ri.a2_re; a2im = ri.a2_im;
                }
            }
            unsigned mask = __ballot_sync(0xffffffffu, active);
            mbar_wait(full0 + 8 * stage, parity);
            const float* tile = ring + (size_t)stage * (stage_bytes / 4);
            while (mask) {
                const int r = __ffs(mask) - 1;
                mask &= mask - 1;
                const float s = __shfl_sync(0xffffffffu, sgn, r);
                const float c = __shfl_sync(0xffffffffu, coef, r);
                const float ar = __shfl_sync(0xffffffffu, a2re, r);
                const float* drow = tile + (size_t)r * p.M_eff;
                if constexpr (!CPLX) {
                    RowPartR cur;
                    st.partial(drow, lane, s, cur.r, cur.acc);
                    cur.ex = s * ar; cur.coef = c;
                    if (pending) { e_hre += finish_pair(pend, cur, lane); pending = false; }
                    else { pend = cur; pending = true; }
                } else {
                    const float ai = __shfl_sync(0xffffffffu, a2im, r);
                    RowPartC cur;
                    st.partial(drow, lane, p.M_pad, s, cur.ar, cur.ai, cur.acc);
                    cur.ex_re = s * ar; cur.ex_im = s * ai; cur.coef = c;
                    if (pending) {
                        float rr, rim;
                        finish_pair_c(pend, cur, lane, rr, rim);
                        e_hre += rr; e_him += rim; pending = false;
                    } else { pend = cur; pending = true; }
                }
            }
            __syncwarp();
            if (lane == 0) {
                // release the stage; the last of the FW warps refills it with tile g + stages
                __threadfence_block();
                if (atomicAdd(&done_cnt[stage], 1) == FW - 1) {
                    done_cnt[stage] = 0;
                    const int64_t g2 = g + p.stages;
                    if (g2 < total_tiles) {
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        issue_tile(p, ring_u32, full0, stage, (int)(g2 % p.n_tiles), stage_bytes);
                    }
                }
            }
            ++g;
            if (++stage == p.stages) { stage = 0; parity ^= 1; }
        }
        if (pending) {
            if constexpr (!CPLX) e_ure = finish_single(pend);
            else finish_single_c(pend, e_ure, e_uim);
        }
        e_hre += __shfl_xor_sync(0xffffffffu, e_hre, 16);          // row-A half + row-B half
        if constexpr (CPLX) e_him += __shfl_xor_sync(0xffffffffu, e_him, 16);
        diag = warp_sum_f(diag);
        if (valid && lane == 0) {
            if constexpr (!CPLX) p.eloc[sample] = diag + (e_ure + e_hre);
            else { p.eloc[2 * sample] = diag + (e_ure + e_hre); p.eloc[2 * sample + 1] = e_uim + e_him; }
        }
    }
}

// ---- dispatch ----------------------------------------------------------------------------------------------
using KernelFn = void (*)(const FusedParams);

template <int V>
static KernelFn pick_real(int v) {
    if (v == V) return fused_eloc_kernel<V, false>;
    if constexpr (V < MAX_V_REAL) return pick_real<V + 1>(v);
    return nullptr;
}
template <int V>
static KernelFn pick_cplx(int v) {
    if (v == V) return fused_eloc_kernel<V, true>;
    if constexpr (V < MAX_V_CPLX) return pick_cplx<V + 1>(v);
    return nullptr;
}

static int g_num_sms = 0;
static bool g_attr_done = false;

cudaError_t fused_eloc_init() {
    if (g_attr_done) return cudaSuccess;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    for (int v = 1; v <= MAX_V_REAL; ++v) {
        e = cudaFuncSetAttribute((const void*)pick_real<1>(v), cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
    }
    for (int v = 1; v <= MAX_V_CPLX; ++v) {
        e = cudaFuncSetAttribute((const void*)pick_cplx<1>(v), cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
    }
    g_attr_done = true;
    return cudaSuccess;
}

int fused_ctas_per_sm(int M_pad, bool cplx) {
    const int V = M_pad / MPAD_ALIGN;
    return ((cplx ? 8 : 4) * V <= 16) ? 2 : 1;
}
int fused_consumer_warps() { return FW; }

cudaError_t launch_fused_eloc(const Operator* op, const Geometry& g, int dtype, const int8_t* sigma, int64_t B,
                              const float* theta, const float* Dtab, const RowInfo* rows, void* eloc_out,
                              cudaStream_t st) {
    if (B <= 0) return cudaSuccess;
    cudaError_t e = fused_eloc_init();
    if (e != cudaSuccess) return e;
    const bool cplx = dtype == NK_C64;
    const int V = g.M_pad / MPAD_ALIGN;
    KernelFn fn = cplx ? pick_cplx<1>(V) : pick_real<1>(V);
    if (fn == nullptr) return cudaErrorInvalidValue;
    FusedParams p;
    p.sigma = sigma; p.B = B; p.N = g.N; p.n_words = g.n_words;
    p.theta = theta; p.M_pad = g.M_pad; p.M_eff = g.M_eff;
    p.Dtab = Dtab; p.rows = rows; p.n_rows = g.n_rows; p.tile_rows = g.tile_rows; p.n_tiles = g.n_tiles;
    p.stages = g.stages;
    p.bonds = op->d_bonds; p.colors = op->d_colors; p.Jf = op->d_Jf; p.n_bonds = op->n_bonds; p.kind = op->kind;
    p.eloc = (float*)eloc_out;
    // one CTA per SM slot, each with an equal contiguous share of the samples (rounds of FW inside the CTA);
    // small batches use fewer CTAs so that every round is full
    const int64_t max_ctas = (int64_t)g_num_sms * g.ctas_per_sm;
    const int64_t n_groups = (B + FW - 1) / FW;
    const int64_t grid = n_groups < max_ctas ? n_groups : max_ctas;
    p.per_cta = (B + grid - 1) / grid;
    fn<<<(unsigned)grid, FTHREADS, g.smem_bytes, st>>>(p);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
