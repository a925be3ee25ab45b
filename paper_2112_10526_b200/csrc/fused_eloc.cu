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
#include <mutex>
#include <type_traits>

#include "nk_internal.h"
#include "ptx_helpers.cuh"
#include "rbm_lane_state.cuh"

namespace nk {

// warps (samples in flight) per CTA: lane_state_warps(V, CPLX) — 16, or 8 for the wide variants (M_pad > 2048 real,
// > 1024 complex: theta alone takes up to 128 registers per lane)

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
    // automatic choice of the form (api.cu): both kernels are launched, each returns at once unless the table's
    // max |tanh delta| (float bits at *gate) is on its side of NK_FORM_TAU_MAX.  gate_mode 0: always run,
    // 1: run iff max <= NK_FORM_TAU_MAX (product form), 2: run iff max > NK_FORM_TAU_MAX (log-cosh form)
    const unsigned* gate;
    int gate_mode;
    const unsigned* series_ctl;              // automatic choice: both SIMT kernels stand down when the tensor-core
                                             // series form runs (series_tc.cu: *series_ctl = K > 0)
};

// ---- kernel ----------------------------------------------------------------------------------------------
template <int V, bool CPLX>
constexpr int min_blocks() { return ((CPLX ? 8 : 4) * V <= 16) ? 2 : 1; }

// per-lane state of the sample: log-cosh form (theta_s, 1 MUFU per pair) or product form (tanh theta, no MUFU)
template <int V, bool CPLX, bool PROD>
using LaneState = typename std::conditional<
    PROD, typename std::conditional<CPLX, ProdCplxState<V>, ProdRealState<V>>::type,
    typename std::conditional<CPLX, CplxState<V>, RealState<V>>::type>::type;

__device__ __forceinline__ void issue_tile(const FusedParams& p, uint32_t ring_u32, uint32_t full0, int stage,
                                           int tile, uint32_t stage_bytes) {
    mbar_arrive_expect_tx(full0 + 8 * stage, stage_bytes);
    bulk_g2s(ring_u32 + stage * stage_bytes, p.Dtab + (size_t)tile * p.tile_rows * p.M_eff, stage_bytes,
             full0 + 8 * stage);
}

template <int V, bool CPLX, bool PROD>
__global__ void __launch_bounds__(lane_state_warps(V, CPLX) * 32, (min_blocks<V, CPLX>())) fused_eloc_kernel(const FusedParams p) {
    constexpr int FW = lane_state_warps(V, CPLX);
    extern __shared__ __align__(128) uint8_t smem[];
    if (p.gate_mode != 0) {                                  // grid-uniform: every thread takes the same branch
        const bool product_ok = __uint_as_float(*p.gate) <= NK_FORM_TAU_MAX;
        if ((p.gate_mode == 1) != product_ok) return;
        if (p.series_ctl != nullptr && *p.series_ctl != 0u) return;
    }
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
    LaneState<V, CPLX, PROD> st;

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
        // real product form: the row pair whose reduction is deferred by one step (products per lane, factors uniform;
        // the neutral start contributes 0)
        float d_a = 1.f, d_b = 1.f, d_fa = 0.f, d_fb = 0.f;
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
            float sgn = 0.f, coef = 0.f, a2re = 0.f, a2im = 0.f, c2re = 0.f, c2im = 0.f;
            if (lane < p.tile_rows) {
                const RowInfo ri = p.rows[t * p.tile_rows + lane];
                if (ri.i >= 0) {
                    const int bi = spin_bit(ri.i);
                    const int bj = (ri.j >= 0) ? spin_bit(ri.j) : (bi ^ 1);
                    active = valid && (bi != bj);
                    diag += (bi != bj) ? -ri.jdiag : ri.jdiag;
                    sgn = bi ? 1.f : -1.f;            // s = -sigma_i
                    coef = ri.coef; a2re = ri.a2_re; a2im = ri.a2_im;
                    if constexpr (PROD) { c2re = ri.c2_re; c2im = ri.c2_im; }
                }
            }
            unsigned mask = __ballot_sync(0xffffffffu, active);
            // real product form: lane r keeps its row's factor c_r 2^(s a2 + c2) and adds the row's term itself, so
            // the row scalars are never broadcast; the sign of s travels in a ballot
            unsigned negm = 0;
            float ce = 0.f;
            if constexpr (PROD && !CPLX) {
                negm = __ballot_sync(0xffffffffu, sgn < 0.f);
                ce = coef * ex2_approx(fmaf(sgn, a2re, c2re));
            }
            mbar_wait(full0 + 8 * stage, parity);
            const float* tile = ring + (size_t)stage * (stage_bytes / 4);
            while (mask) {
                const int r = __ffs(mask) - 1;
                mask &= mask - 1;
                if constexpr (PROD && !CPLX) {
                    // rows are reduced in pairs, one step late: the butterfly of the pair completed before runs inside
                    // the next row's loads (partial_s_retire).  f: the row's factor, broadcast from its lane now, while
                    // the lanes still hold this tile's factors
                    const float* trow = tile + (size_t)r * p.M_eff;
                    const bool neg = ((negm >> r) & 1u) != 0;
                    const float f = __shfl_sync(0xffffffffu, ce, r);
                    if (pending || mask != 0u) {
                        float rk;
                        const float pr = neg ? st.template partial_s_retire<true>(trow, lane, d_a, d_b, rk)
                                             : st.template partial_s_retire<false>(trow, lane, d_a, d_b, rk);
                        e_hre = fmaf((lane & 16) ? d_fb : d_fa, rk, e_hre);
                        if (pending) { d_a = pend.r; d_fa = pend.coef; pending = false; }
                        else {
                            d_a = pr; d_fa = f;
                            const int r2 = __ffs(mask) - 1;
                            mask &= mask - 1;
                            const float* trow2 = tile + (size_t)r2 * p.M_eff;
                            const float f2 = __shfl_sync(0xffffffffu, ce, r2);
                            const float pr2 = ((negm >> r2) & 1u) ? st.template partial_s<true>(trow2, lane)
                                                                  : st.template partial_s<false>(trow2, lane);
                            d_b = pr2; d_fb = f2;
                            continue;
                        }
                        d_b = pr; d_fb = f;
                    } else {                              // last row of the tile, no partner yet
                        pend.r = neg ? st.template partial_s<true>(trow, lane) : st.template partial_s<false>(trow, lane);
                        pend.coef = f;
                        pending = true;
                    }
                    continue;
                }
                const float s = __shfl_sync(0xffffffffu, sgn, r);
                const float c = __shfl_sync(0xffffffffu, coef, r);
                const float ar = __shfl_sync(0xffffffffu, a2re, r);
                const float* drow = tile + (size_t)r * p.M_eff;
                float cre = 0.f;                      // product form: log2 of prod_j |cosh d_j| of this row
                if constexpr (PROD) cre = __shfl_sync(0xffffffffu, c2re, r);
                if constexpr (!CPLX) {
                    RowPartR cur;
                    st.partial(drow, lane, s, cur.r, cur.acc);
                    cur.ex = fmaf(s, ar, cre); cur.coef = c;
                    if (pending) {
                        e_hre += PROD ? finish_pair_prod(pend, cur, lane) : finish_pair(pend, cur, lane);
                        pending = false;
                    } else { pend = cur; pending = true; }
                } else {
                    const float ai = __shfl_sync(0xffffffffu, a2im, r);
                    float cim = 0.f;
                    if constexpr (PROD) cim = __shfl_sync(0xffffffffu, c2im, r);
                    RowPartC cur;
                    st.partial(drow, lane, p.M_pad, s, cur.ar, cur.ai, cur.acc);
                    cur.ex_re = fmaf(s, ar, cre); cur.ex_im = fmaf(s, ai, cim); cur.coef = c;
                    if (pending) {
                        float rr, rim;
                        if constexpr (PROD) finish_pair_prod_c(pend, cur, lane, rr, rim);
                        else finish_pair_c(pend, cur, lane, rr, rim);
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
            if constexpr (PROD && !CPLX) e_ure = pend.coef * warp_prod_f(pend.r);
            else if constexpr (!CPLX) e_ure = finish_single(pend);
            else if constexpr (PROD) finish_single_prod_c(pend, e_ure, e_uim);
            else finish_single_c(pend, e_ure, e_uim);
        }
        if constexpr (PROD && !CPLX) {                             // the pair still deferred
            const bool up = (lane & 16) != 0;
            float k = up ? d_b : d_a;
            k *= __shfl_xor_sync(0xffffffffu, up ? d_a : d_b, 16);
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) k *= __shfl_xor_sync(0xffffffffu, k, o);
            e_hre = fmaf(up ? d_fb : d_fa, k, e_hre);
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

template <int V, bool PROD = false>
static KernelFn pick_real(int v) {
    if (v == V) return fused_eloc_kernel<V, false, PROD>;
    if constexpr (V < MAX_V_REAL) return pick_real<V + 1, PROD>(v);
    return nullptr;
}
template <int V, bool PROD = false>
static KernelFn pick_cplx(int v) {
    if (v == V) return fused_eloc_kernel<V, true, PROD>;
    if constexpr (V < MAX_V_CPLX) return pick_cplx<V + 1, PROD>(v);
    return nullptr;
}

// per-device one-time set-up (the shared-memory attribute and the SM count belong to the current device)
static std::mutex g_fused_mutex;
static int g_sms_of[NK_MAX_DEVICES];
static bool g_attr_done_of[NK_MAX_DEVICES];
#define g_num_sms (g_sms_of[current_device()])

cudaError_t fused_eloc_init() {
    std::lock_guard<std::mutex> lock(g_fused_mutex);
    if (g_attr_done_of[current_device()]) return cudaSuccess;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&g_sms_of[current_device()], cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    for (int v = 1; v <= MAX_V_REAL; ++v)
        for (const void* fn : {(const void*)pick_real<1>(v), (const void*)pick_real<1, true>(v)}) {
            e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
            if (e != cudaSuccess) return e;
        }
    for (int v = 1; v <= MAX_V_CPLX; ++v)
        for (const void* fn : {(const void*)pick_cplx<1>(v), (const void*)pick_cplx<1, true>(v)}) {
            e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
            if (e != cudaSuccess) return e;
        }
    g_attr_done_of[current_device()] = true;
    return cudaSuccess;
}

int fused_ctas_per_sm(int M_pad, bool cplx) {
    const int V = M_pad / MPAD_ALIGN;
    return ((cplx ? 8 : 4) * V <= 16) ? 2 : 1;
}
int fused_consumer_warps(int M_pad, bool cplx) { return lane_state_warps(M_pad / MPAD_ALIGN, cplx); }

cudaError_t launch_fused_eloc(const Operator* op, const Geometry& g, int dtype, const int8_t* sigma, int64_t B,
                              const float* theta, const float* Dtab, const RowInfo* rows, void* eloc_out,
                              bool product_form, cudaStream_t st, const unsigned* gate, int gate_mode,
                              const unsigned* series_ctl) {
    if (B <= 0) return cudaSuccess;
    cudaError_t e = fused_eloc_init();
    if (e != cudaSuccess) return e;
    const bool cplx = dtype == NK_C64;
    const int V = g.M_pad / MPAD_ALIGN;
    KernelFn fn = product_form ? (cplx ? pick_cplx<1, true>(V) : pick_real<1, true>(V))
                               : (cplx ? pick_cplx<1>(V) : pick_real<1>(V));
    if (fn == nullptr) return cudaErrorInvalidValue;
    FusedParams p;
    p.sigma = sigma; p.B = B; p.N = g.N; p.n_words = g.n_words;
    p.theta = theta; p.M_pad = g.M_pad; p.M_eff = g.M_eff;
    p.Dtab = Dtab; p.rows = rows; p.n_rows = g.n_rows; p.tile_rows = g.tile_rows; p.n_tiles = g.n_tiles;
    p.stages = g.stages;
    p.bonds = op->d_bonds; p.colors = op->d_colors; p.Jf = op->d_Jf; p.n_bonds = op->n_bonds; p.kind = op->kind;
    p.eloc = (float*)eloc_out;
    p.gate = gate; p.gate_mode = gate_mode; p.series_ctl = series_ctl;
    // one CTA per SM slot, each with an equal contiguous share of the samples (rounds of FW inside the CTA);
    // small batches use fewer CTAs so that every round is full
    const int FW = lane_state_warps(V, cplx);
    const int64_t max_ctas = (int64_t)g_num_sms * g.ctas_per_sm;
    const int64_t n_groups = (B + FW - 1) / FW;
    const int64_t grid = n_groups < max_ctas ? n_groups : max_ctas;
    p.per_cta = (B + grid - 1) / grid;
    fn<<<(unsigned)grid, FW * 32, g.smem_bytes, st>>>(p);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
