// Local energies with the amplitude ratios evaluated on the tensor cores (Eq. (12); the cost the paper
// names at L691 / L1630: one model evaluation per connected configuration).
//
// Product form: psi'/psi = e^{s da} prod_j cosh(d_j) prod_j (1 + s t_j tau_j), t = tanh(theta) per
// sample, tau = tanh(d) per table row, s = +-1.  Taking the logarithm of the last product and expanding,
//     ln prod_j (1 + s t_sj tau_bj) = sum_{k>=1} ((-1)^{k+1} / k) s^k  sum_j t_sj^k tau_bj^k ,
// turns the [samples] x [rows] block of log-ratios into a SHORT SERIES OF GEMMs over the hidden units, one per power k:
//     odd [s][b] = sum_{k odd}  (1/k)  (T^k (tau^k)^T)[s][b]        (multiplied by s in the epilogue)
//     even[s][b] = sum_{k even} (-1/k) (T^k (tau^k)^T)[s][b]
//     ln(psi'/psi)[s][b] = c_b + s (da_b + odd) + even .
// |t| <= 1, so the remainder after K terms is at most sum_j |tau_bj|^(K+1) / ((K+1)(1 - tau_max)) — a number that
// depends on the parameters only.  series_select_kernel takes the smallest K <= K_MAX that brings it under
// SERIES_TOL for every row (config 5: K = 5, bound 5.6e-6) or switches the path off (K = 0: the SIMT kernels of
// fused_eloc.cu run instead); everything downstream reads K from device memory, so the call never synchronises.
//
// Precision plan (fp32 accumulation in tensor memory; measured against the float64 oracle in tests/test_gpu_series.py):
//   k = 1   carries ~0.4 in the exponent and needs ~17 bits: both operands are split into fp16 hi + lo pieces and
//           three MMA passes hi*hi + lo*hi + hi*lo run (the dropped lo*lo is 2^-24 relative);
//   k = 2   one fp16 pass (11 bits: 1.3e-6 rms at config 5);   k >= 3: one bf16 pass each (range down to 1e-38).
//   tau is scaled by a power of two so that tau_max lands in [1/2, 1) and by log2(e) (the epilogue works in log2 units);
//   the scale is undone exactly in the epilogue.
// So a sample row / table row is a vector of (K + 1) M_pad 16-bit numbers [hi | lo | k=2 | ... | k=K] and the whole
// series is ONE GEMM with K + 2 passes per block of hidden units into two fp32 accumulators (odd, even).
//
// Kernel (series_gemm_kernel): persistent, one CTA per SM, 128 (samples) x 256 (table rows) tiles, tcgen05.mma
// kind::f16 M = 128, N = 256, K = 16 issued by one thread; accumulators odd / even fill the 512 TMEM columns.  The two
// operands flow through separate shared-memory rings (4 x 16 KB and 4 x 32 KB, 128B-swizzled TMA boxes of 64 hidden
// units), each with its own producer warp.  Eight epilogue warps (two per TMEM lane
// quarter, half of the 256 columns each) read both accumulators, form the exponent, take 2^x, multiply by the matrix element, mask by the
// sample's spins (antiparallel bond / sign of s from bit-packed transposed spins) and sum over the tile's rows —
// [samples] x [rows] never leaves the SM.  Partial sums per half column tile go to `part`, summed in a fixed order by
// series_finish_kernel (bit-reproducible, independent of chunk_size).
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <mutex>

#include "nk_internal.h"
#include "ptx_helpers.cuh"
#include "tc_helpers.cuh"

namespace nk {

namespace ser {
constexpr int BM = 128, BN = 256, BK = 64;                // BK 16-bit elements = one 128-B swizzle row
constexpr int A_TILE = BM * BK * 2;                       // 16 KB
constexpr int NA = 4;                                     // ring depths (3 + 3 measured: GEMM 181 -> 207 us per chunk)
constexpr int EPI_HALVES = 2;                             // epilogue warps per TMEM lane quarter: each drains BN / 2 columns
constexpr int EPI_WARPS = 4 * EPI_HALVES, EPI_COLS = BN / EPI_HALVES;
constexpr int THREADS = 96 + 32 * EPI_WARPS;              // warps: A producer, MMA, B producer, 8 x epilogue
constexpr int TAB_BYTES = BN * 16, MSK_BYTES = EPI_COLS * 8;   // (coef, jdiag, a2, c2) per column, shared by the epilogue
                                                          // warps; (act, neg) spin masks per column of each epilogue warp
// CG = CTAs per tile: 1 (a CTA owns a 128 x 256 tile) or 2 (a CTA PAIR owns 256 x 256 through tcgen05 cta_group::2: each
// CTA holds its 128 samples' A tiles and HALF of every B tile, so the table-row operand crosses L2 -> shared memory and
// shared memory -> tensor core once per 256 samples instead of once per 128)
template <int CG> struct Cfg {
    static constexpr int B_TILE = (BN / CG) * BK * 2;     // 32 KB, or 16 KB per CTA of a pair
    static constexpr int NB = CG == 2 ? 6 : 4;
    static constexpr int SMEM_BYTES = NA * A_TILE + NB * B_TILE + TAB_BYTES + EPI_WARPS * MSK_BYTES + 256 /*barriers*/ + 1024 /*alignment*/;
};
constexpr uint32_t TMEM_COLS = 512;                       // odd at column 0, even at column 256
// instruction descriptors of kind::f16 (the cute::UMMA::InstrDescriptor bit layout): D = F32 (c_format 1 at bit 4),
// A / B format at bits 7 / 10 (0 = F16, 1 = BF16), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
template <int CG> struct Idesc {
    static constexpr uint32_t F16 = (1u << 4) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)((BM * CG) >> 4) << 24);
    static constexpr uint32_t BF16 = F16 | (1u << 7) | (1u << 10);
};
}  // namespace ser

// ---- control block (device): ctl[0] = K (0: path off), ctl[1] = 2^e as float bits (undoes the power-of-two scale of
// tau), ctl[2] = log2(e) 2^-e as float bits (the scale applied to tau), ctl[4 + p] = max over rows of sum_j |tau|^p ----
constexpr int SER_CTL_WORDS = 16;

// (the row sums ctl[4 + p] are formed by rowtab_real_kernel, pack.cu, in its pass over the table)

// force: 0 = automatic (K = 0 when no K <= K_MAX meets SERIES_TOL or tau_max > SERIES_TAU_MAX); 1 = the caller forced
// the path (NK_FORM_SERIES): K_MAX terms are used when the bound cannot be met
__global__ void series_select_kernel(unsigned* __restrict__ ctl, const unsigned* __restrict__ taumax_bits, int force) {
    const float tau = __uint_as_float(*taumax_bits);
    int K = 0;
    if (tau <= SERIES_TAU_MAX) {
        for (int k = 2; k <= SERIES_K_MAX; ++k) {
            const float bound = __uint_as_float(ctl[4 + k + 1]) / ((float)(k + 1) * (1.f - tau));
            if (bound <= SERIES_TOL) { K = k; break; }
        }
    }
    if (force && K == 0) K = SERIES_K_MAX;
    int ex = 0;
    if (tau > 0.f && tau < 1.f) frexpf(tau, &ex);         // tau = f 2^ex, f in [1/2, 1): tau 2^-ex lands in [1/2, 1)
    ctl[0] = (unsigned)K;
    ctl[1] = __float_as_uint(ldexpf(1.f, ex));
    ctl[2] = __float_as_uint(LOG2E * ldexpf(1.f, -ex));
}

__device__ __forceinline__ uint16_t f2h(float x) { return __half_as_ushort(__float2half_rn(x)); }
__device__ __forceinline__ float h2f(uint16_t h) { return __half2float(__ushort_as_half(h)); }
__device__ __forceinline__ uint16_t f2b(float x) { return __bfloat16_as_ushort(__float2bfloat16_rn(x)); }

// Bp[r][seg][j]: seg 0 / 1 = fp16 hi / lo of x = log2(e) 2^-e tau; seg k >= 2 = (-1)^(k+1) log2(e) 2^-e tau^k / k
// (fp16 for k = 2, bf16 above).  One block per table row.
__global__ void __launch_bounds__(256)
series_bpow_kernel(const float* __restrict__ Ttab, int M_pad, int M_eff, const unsigned* __restrict__ ctl,
                   uint16_t* __restrict__ Bp) {
    const int K = (int)ctl[0];
    if (K == 0) return;
    const float sc = __uint_as_float(ctl[2]);
    const float* row = Ttab + (size_t)blockIdx.x * M_eff;
    uint16_t* out = Bp + (size_t)blockIdx.x * SERIES_SEGS * M_pad;
    for (int j = threadIdx.x; j < M_pad; j += blockDim.x) {
        const float tau = row[j];
        const float x = sc * tau;
        const uint16_t hi = f2h(x);
        out[j] = hi;
        out[M_pad + j] = f2h(x - h2f(hi));
        float p = x;                                       // sc tau^k
        for (int k = 2; k <= K; ++k) {
            p *= tau;
            const float v = ((k & 1) ? p : -p) / (float)k;
            out[(size_t)k * M_pad + j] = k == 2 ? f2h(v) : f2b(v);
        }
    }
}

// The sample-side operand Ap[s][seg][j] (seg 0 / 1 = fp16 hi / lo of t = tanh(theta); seg 2 = fp16 t^2; seg k >= 3 =
// bf16 t^k) is written by logpsi_kernel (logpsi.cu) in its pass over theta.

// sigT[i][w]: bit l of word w <=> sigma[32 w + l][i] = -1 (samples beyond nb: 0).  One warp = 32 samples x 16 sites:
// lane l loads 16 spins of sample 32 w + l (one 16-B load when the rows allow it), 16 ballots transpose them.
__global__ void __launch_bounds__(256)
series_bits_kernel(const int8_t* __restrict__ sigma, int64_t nb, int N, int w32, int n_groups,
                   const unsigned* __restrict__ ctl, uint32_t* __restrict__ sigT) {
    if (ctl[0] == 0) return;
    const int lane = threadIdx.x & 31;
    const int n16 = (N + 15) / 16;
    const int64_t gw = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (gw >= (int64_t)n_groups * n16) return;
    const int grp = (int)(gw / n16), i0 = (int)(gw - (int64_t)grp * n16) * 16;
    const int64_t s = (int64_t)grp * 32 + lane;
    uint32_t v[4] = {0x01010101u, 0x01010101u, 0x01010101u, 0x01010101u};      // +1: bit clear
    if (s < nb) {
        const int8_t* src = sigma + s * N + i0;
        if ((N & 15) == 0 && (((uintptr_t)sigma) & 15) == 0) {
            const uint4 q = *reinterpret_cast<const uint4*>(src);
            v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
        } else {
            for (int k = 0; k < 16 && i0 + k < N; ++k)
                v[k >> 2] = (v[k >> 2] & ~(0xffu << (8 * (k & 3)))) | ((uint32_t)(uint8_t)src[k] << (8 * (k & 3)));
        }
    }
    uint32_t mine = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const uint32_t w = __ballot_sync(0xffffffffu, (v[k >> 2] >> (8 * (k & 3) + 7)) & 1u);
        if (lane == k) mine = w;
    }
    if (lane < 16 && i0 + lane < N) sigT[(size_t)(i0 + lane) * w32 + grp] = mine;
}

// ---- the GEMM with the fused local-energy epilogue ---------------------------------------------------------------
struct SeriesParams {
    const unsigned* ctl;
    const RowInfo* rows;
    const uint32_t* sigT;
    int w32;                      // words per site of sigT
    int64_t nb;                   // samples of this chunk
    int n_rows, M_pad;
    int n_mt, n_nt;               // tiles along samples / table rows
    float* part;                  // [n_nt * EPI_HALVES][part_stride]
    int64_t part_stride;
};

__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                         uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}

// ---- cta_group::2 forms (the CTA pair of one TPC; rank 0 = the leader, which alone issues the MMAs) -----------------
__device__ __forceinline__ void umma_f16_cg2(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                             uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
template <int CG>
__global__ void __launch_bounds__(ser::THREADS, 1)
series_gemm_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
                   const SeriesParams p) {
    using namespace ser;
    constexpr int NB = Cfg<CG>::NB, B_TILE = Cfg<CG>::B_TILE;
    constexpr uint32_t IDESC_F16 = Idesc<CG>::F16, IDESC_BF16 = Idesc<CG>::BF16;
    const uint32_t rank = CG == 2 ? cluster_ctarank() : 0u;            // rank 0 leads the pair
    const int K = (int)p.ctl[0];
    if (K == 0) return;                                    // grid-uniform: the path is off for these parameters
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_al = smem_raw + (smem_base - smem_u32(smem_raw));
    const uint32_t a_ring = smem_base, b_ring = smem_base + NA * A_TILE;
    const uint32_t epi_off = NA * A_TILE + NB * B_TILE;
    const uint32_t bars = smem_base + epi_off + TAB_BYTES + EPI_WARPS * MSK_BYTES;
    const uint32_t a_full = bars, a_empty = bars + 8 * NA, b_full = bars + 16 * NA, b_empty = b_full + 8 * NB;
    const uint32_t t_full = b_empty + 8 * NB, t_empty = t_full + 8, tmem_slot = t_empty + 8;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_al + (tmem_slot - smem_base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_jb = p.M_pad / BK;
    const int n_tiles = ((p.n_mt + CG - 1) / CG) * p.n_nt;              // tiles of CG x 128 samples x 256 table rows
    const int unit = blockIdx.x / CG, n_units = gridDim.x / CG;         // the CTA (pair) as a tile worker
    // `full` barriers count the bytes of BOTH CTAs of a pair and live in the leader; `empty` / accumulator-ready barriers
    // are local, signalled in both CTAs by the leader's multicast commits; the accumulators of both CTAs are handed back
    // on the leader's t_empty
    const uint32_t a_full_l = CG == 2 ? map_to_rank(a_full, 0) : a_full;
    const uint32_t b_full_l = CG == 2 ? map_to_rank(b_full, 0) : b_full;
    const uint32_t t_empty_l = CG == 2 ? map_to_rank(t_empty, 0) : t_empty;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NA; ++s) { mbar_init(a_full + 8 * s, 1); mbar_init(a_empty + 8 * s, 1); }
        for (int s = 0; s < NB; ++s) { mbar_init(b_full + 8 * s, 1); mbar_init(b_empty + 8 * s, 1); }
        mbar_init(t_full, 1);
        mbar_init(t_empty, 32 * EPI_WARPS * CG);
        mbar_fence_init();
    }
    if (warp == 1) {                                       // the same warp in both CTAs of a pair
        if (CG == 2) {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(TMEM_COLS)
                         : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(TMEM_COLS)
                         : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (CG == 2) cluster_sync_all();                       // the peer's barriers exist before anything signals them
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot_ptr;

    // Order of the passes inside a tile.  The tensor core adds every product to the fp32 accumulator on the accumulator's
    // own grid (measured: a bias of 2048 half-ulps when 2048 same-sign products meet a large running sum, and products
    // below the grid are lost), so SMALL terms go first, while the sums are small:
    //   sweep 1 over the blocks of hidden units:  k = K .. 3 (bf16), then the two fp16 lo passes t_lo tau_hi, t_hi tau_lo
    //   sweep 2:                                  k = 2, then the dominant t_hi tau_hi
    // (the first version ran all passes of a block together: E_loc came out 7e-6 high — the k = 4 and lo terms were
    // being added to full-size sums.)  t_hi and tau_hi are therefore loaded in both sweeps: K + 2 tiles of each operand
    // per block for K + 2 passes.  A ring slot is handed back by the tcgen05.commit of the last pass that reads it.
    if (warp == 0) {
        // ===== A producer =====
        if (lane == 0) {
            uint32_t it = 0;
            auto load = [&](int seg, int jb, int m0) {
                const uint32_t slot = it % NA, par = ((it / NA) & 1u) ^ 1u;
                mbar_wait(a_empty + 8 * slot, par);
                if (rank == 0) mbar_arrive_expect_tx(a_full + 8 * slot, CG * A_TILE);
                if (CG == 2) tma_load_2d_cg2(a_ring + slot * A_TILE, &map_a, seg * p.M_pad + jb * BK, m0, a_full_l + 8 * slot);
                else tma_load_2d(a_ring + slot * A_TILE, &map_a, seg * p.M_pad + jb * BK, m0, a_full + 8 * slot);
                ++it;
            };
            for (int tile = unit; tile < n_tiles; tile += n_units) {
                const int m0 = ((tile / p.n_nt) * CG + (int)rank) * BM;
                for (int jb = 0; jb < n_jb; ++jb) {
                    for (int k = K; k >= 3; --k) load(k, jb, m0);
                    load(1, jb, m0);                       // t_lo
                    load(0, jb, m0);                       // t_hi
                }
                for (int jb = 0; jb < n_jb; ++jb) { load(2, jb, m0); load(0, jb, m0); }
            }
        }
    } else if (warp == 2) {
        // ===== B producer =====
        if (lane == 0) {
            uint32_t it = 0;
            auto load = [&](int seg, int jb, int n0) {
                const uint32_t slot = it % NB, par = ((it / NB) & 1u) ^ 1u;
                mbar_wait(b_empty + 8 * slot, par);
                if (rank == 0) mbar_arrive_expect_tx(b_full + 8 * slot, CG * B_TILE);
                if (CG == 2) tma_load_2d_cg2(b_ring + slot * B_TILE, &map_b, seg * p.M_pad + jb * BK, n0, b_full_l + 8 * slot);
                else tma_load_2d(b_ring + slot * B_TILE, &map_b, seg * p.M_pad + jb * BK, n0, b_full + 8 * slot);
                ++it;
            };
            for (int tile = unit; tile < n_tiles; tile += n_units) {
                const int n0 = (tile % p.n_nt) * BN + (int)rank * (BN / CG);      // this CTA's half of the table rows
                for (int jb = 0; jb < n_jb; ++jb) {
                    for (int k = K; k >= 3; --k) load(k, jb, n0);
                    load(0, jb, n0);                       // tau_hi
                    load(1, jb, n0);                       // tau_lo
                }
                for (int jb = 0; jb < n_jb; ++jb) { load(2, jb, n0); load(0, jb, n0); }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one thread of the leader CTA) =====
        if (lane == 0 && rank == 0) {
            uint32_t ia = 0, ib = 0, n_done = 0;
            const uint32_t acc_odd = tmem_base, acc_even = tmem_base + BN;
            bool fresh_odd = true, fresh_even = true;
            auto a_wait = [&](uint32_t i) { mbar_wait(a_full + 8 * (i % NA), (i / NA) & 1u); };
            auto b_wait = [&](uint32_t i) { mbar_wait(b_full + 8 * (i % NB), (i / NB) & 1u); };
            auto pass = [&](uint32_t sa, uint32_t sb, bool odd, uint32_t idesc) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t a_addr = a_ring + (sa % NA) * A_TILE, b_addr = b_ring + (sb % NB) * B_TILE;
                bool& fresh = odd ? fresh_odd : fresh_even;
#pragma unroll
                for (int k = 0; k < BK / 16; ++k) {        // 16 elements = 32 B inside the 128-B swizzle row
                    if (CG == 2)
                        umma_f16_cg2(odd ? acc_odd : acc_even, make_sdesc(a_addr + k * 32), make_sdesc(b_addr + k * 32),
                                     idesc, (fresh && k == 0) ? 0u : 1u);
                    else
                        umma_f16(odd ? acc_odd : acc_even, make_sdesc(a_addr + k * 32), make_sdesc(b_addr + k * 32), idesc,
                                 (fresh && k == 0) ? 0u : 1u);
                }
                fresh = false;
            };
            auto commit = [&](uint32_t bar) { if (CG == 2) umma_commit_cg2(bar); else umma_commit(bar); };
            auto a_free = [&](uint32_t i) { commit(a_empty + 8 * (i % NA)); };
            auto b_free = [&](uint32_t i) { commit(b_empty + 8 * (i % NB)); };
            for (int tile = unit; tile < n_tiles; tile += n_units, ++n_done) {
                mbar_wait(t_empty, (n_done & 1u) ^ 1u);    // the epilogue has drained the accumulators (free at first)
                fresh_odd = fresh_even = true;
                for (int jb = 0; jb < n_jb; ++jb) {        // sweep 1: the small terms
                    for (int k = K; k >= 3; --k, ++ia, ++ib) {
                        a_wait(ia); b_wait(ib);
                        pass(ia, ib, (k & 1) != 0, IDESC_BF16);
                        a_free(ia); b_free(ib);
                    }
                    const uint32_t a_lo = ia, a_hi = ia + 1, b_hi = ib, b_lo = ib + 1;
                    a_wait(a_lo); b_wait(b_hi);
                    pass(a_lo, b_hi, true, IDESC_F16);
                    a_free(a_lo); b_free(b_hi);
                    a_wait(a_hi); b_wait(b_lo);
                    pass(a_hi, b_lo, true, IDESC_F16);
                    a_free(a_hi); b_free(b_lo);
                    ia += 2; ib += 2;
                }
                for (int jb = 0; jb < n_jb; ++jb) {        // sweep 2: k = 2 and the dominant hi x hi
                    a_wait(ia); b_wait(ib);
                    pass(ia, ib, false, IDESC_F16);
                    a_free(ia); b_free(ib);
                    a_wait(ia + 1); b_wait(ib + 1);
                    pass(ia + 1, ib + 1, true, IDESC_F16);
                    a_free(ia + 1); b_free(ib + 1);
                    ia += 2; ib += 2;
                }
                commit(t_full);
            }
        }
    } else {
        // ===== epilogue: warps 3..10; TMEM lane quarter q = warp % 4, column half h (two warps drain a quarter's 256
        // columns side by side: the tensor pipe idles from the last MMA of a tile until the accumulators are handed back,
        // so the drain time is what the tile pays for having one accumulator set) =====
        const int q = warp & 3;
        const int we = warp - 3, h = we >> 2;              // 0..7; this warp's columns are [h EPI_COLS, (h + 1) EPI_COLS)
        float4* tab = reinterpret_cast<float4*>(smem_al + epi_off);
        uint2* msk = reinterpret_cast<uint2*>(smem_al + epi_off + TAB_BYTES + we * MSK_BYTES);
        const float inv = __uint_as_float(p.ctl[1]);
        uint32_t n_done = 0;
        for (int tile = unit; tile < n_tiles; tile += n_units, ++n_done) {
            const int nt = tile % p.n_nt, mt = (tile / p.n_nt) * CG + (int)rank;     // this CTA's 128 samples
            const int n0 = nt * BN;
            // per column: matrix element, diagonal coupling and exponents (the warp stages the records of the 32 columns
            // q of its half for everyone) and the two spin masks of this warp's 32 samples
            asm volatile("bar.sync 1, %0;" ::"n"(32 * EPI_WARPS) : "memory");   // all are done with the previous tile's records
            for (int cc = lane; cc < EPI_COLS; cc += 32) {
                const int c = h * EPI_COLS + cc;
                uint2 m = make_uint2(0u, 0u);
                float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
                if (n0 + c < p.n_rows) {
                    const RowInfo ri = p.rows[n0 + c];
                    if (ri.i >= 0) {
                        t = make_float4(ri.coef, ri.jdiag, ri.a2_re, ri.c2_re);
                        if ((int64_t)mt * BM + q * 32 < p.nb) {   // a pair's second tile may lie beyond the samples
                            const uint32_t wi = p.sigT[(size_t)ri.i * p.w32 + mt * 4 + q];
                            const uint32_t wj = ri.j >= 0 ? p.sigT[(size_t)ri.j * p.w32 + mt * 4 + q] : ~wi;
                            m = make_uint2(wi ^ wj, wi);   // antiparallel <=> active; sigma_i = -1 <=> s = +1
                        }
                    }
                }
                if (((cc >> 5) & 3) == q) tab[c] = t;
                msk[cc] = m;
            }
            asm volatile("bar.sync 1, %0;" ::"n"(32 * EPI_WARPS) : "memory");
            const int64_t row = (int64_t)mt * BM + q * 32 + lane;
            float E = 0.f;
            mbar_wait(t_full, n_done & 1u);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll 1
            for (int c0 = 0; c0 < EPI_COLS; c0 += 32) {
                float od[32], ev[32];
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + h * EPI_COLS + c0;
                tmem_ld32(taddr, od);
                tmem_ld32(taddr + BN, ev);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (c0 + 32 == EPI_COLS) {                 // both accumulators are in registers: hand them back
                    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                    if (CG == 2) mbar_arrive_cluster(t_empty_l); else mbar_arrive(t_empty);
                }
#pragma unroll
                for (int jj = 0; jj < 32; ++jj) {
                    const float4 t = tab[h * EPI_COLS + c0 + jj];
                    const uint2 m = msk[c0 + jj];
                    const float u = fmaf(inv, od[jj], t.z);                 // da + odd        (log2 units)
                    const float v = fmaf(inv, ev[jj], t.w);                 // c + even
                    const float e2 = ((m.y >> lane) & 1u) ? v + u : v - u;  // c + s (da + odd) + even
                    const float term = fmaf(t.x, ex2_approx(e2), -t.y);     // mel psi'/psi - J   (antiparallel bond)
                    E += ((m.x >> lane) & 1u) ? term : t.y;                 // parallel bond: + J, no connected state
                }
            }
            if (row < p.nb) p.part[(size_t)(nt * EPI_HALVES + h) * p.part_stride + row] = E;
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (CG == 2) cluster_sync_all();                       // no peer still signals this CTA's barriers or reads its operands
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (CG == 2)
            asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
        else
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
    }
}

// eloc[s] = sum over column tiles of part (fixed order) + the diagonal of the Ising bonds (the Heisenberg diagonal is
// already inside part: every bond is a table row).  One warp per sample.
__global__ void __launch_bounds__(256)
series_finish_kernel(const float* __restrict__ part, int n_nt, int64_t part_stride, const int8_t* __restrict__ sigma,
                     int64_t nb, int N, int kind, const int32_t* __restrict__ bonds, const int32_t* __restrict__ colors,
                     const float* __restrict__ Jf, int n_bonds, const unsigned* __restrict__ ctl,
                     float* __restrict__ eloc) {
    if (ctl[0] == 0) return;
    const int lane = threadIdx.x & 31;
    const int64_t s = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= nb) return;
    float diag = 0.f;
    if (kind == NK_ISING) {
        const int8_t* sg = sigma + s * N;
        for (int b = lane; b < n_bonds; b += 32) {
            const float J = Jf[colors[b]];
            diag += (sg[bonds[2 * b]] != sg[bonds[2 * b + 1]]) ? -J : J;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) diag += __shfl_xor_sync(0xffffffffu, diag, o);
    }
    if (lane == 0) {
        float e = 0.f;
        for (int t = 0; t < n_nt; ++t) e += part[(size_t)t * part_stride + s];
        eloc[s] = diag + e;
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------
static std::mutex g_ser_mutex;
static bool g_ser_ready[NK_MAX_DEVICES];
static int g_ser_sms[NK_MAX_DEVICES];
static int g_ser_pairs[NK_MAX_DEVICES];                    // co-resident CTA pairs (0: the device refuses 2-CTA clusters)

static cudaError_t series_init() {
    std::lock_guard<std::mutex> lock(g_ser_mutex);
    const int d = current_device();
    if (g_ser_ready[d]) return cudaSuccess;
    if (tensor_map_encoder() == nullptr) return cudaErrorNotSupported;
    cudaError_t e = cudaFuncSetAttribute((const void*)series_gemm_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         ser::Cfg<1>::SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute((const void*)series_gemm_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 ser::Cfg<2>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0;
    e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    g_ser_sms[d] = sms > 0 ? sms : 148;
    {   // how many CTA pairs the device co-schedules
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(2, 1, 1); cfg.blockDim = dim3(ser::THREADS, 1, 1); cfg.dynamicSmemBytes = ser::Cfg<2>::SMEM_BYTES;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, (const void*)series_gemm_kernel<2>, &cfg) != cudaSuccess) n = 0;
        (void)cudaGetLastError();
        g_ser_pairs[d] = n;
    }
    g_ser_ready[d] = true;
    return cudaSuccess;
}

// 2-D tensor map over a [rows][cols] operand of 16-bit elements, box = box_rows x 64 elements (128 B), 128B swizzle;
// rows beyond `rows` read as zeros
static bool encode_u16(CUtensorMap* map, const void* base, uint64_t rows, uint64_t cols, int box_rows) {
    const cuuint64_t dims[2] = {cols, rows};
    const cuuint64_t strides[1] = {cols * 2};
    const cuuint32_t box[2] = {(cuuint32_t)ser::BK, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return tensor_map_encoder()(map, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, const_cast<void*>(base), dims, strides, box,
                                estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool series_possible(const Geometry& g, int dtype) {
    // real parameters; large enough that 128 x 256 tiles over >= 4 blocks of 64 hidden units make sense
    return dtype == NK_F32 && g.n_rows >= SERIES_MIN_ROWS && g.M_pad >= SERIES_MIN_MPAD;
}

// How many chunks one tensor-core launch covers.  A launch runs ceil(tiles / units) waves of tiles over `units` CTA pairs
// (or CTAs), so a chunk whose tile count is not a multiple of `units` leaves the last wave partly idle (config 5: 128
// pair tiles on 74 pairs = 1.73 waves, 13 % idle).  The sample-side operand rows of `group` consecutive chunks are
// therefore kept (two such buffers when there is more than one group: the preparation of group G + 1 runs beside the
// launch of group G) and contracted together: the smallest group <= 8 within 3 % of the best wave efficiency, capped at
// 1 GiB of operand rows per buffer.  Depends on sizes only, never on the parameters or the samples.
static int series_group(const Geometry& g, int64_t chunk, int64_t B, int n_nt) {
    if (chunk >= B) return 1;
    int units = 74, cg = 2;
    if (series_init() == cudaSuccess) {
        const int d = current_device();
        if (g_ser_pairs[d] > 0) units = g_ser_pairs[d];
        else { units = g_ser_sms[d]; cg = 1; }
    }
    const size_t row_bytes = (size_t)SERIES_SEGS * g.M_pad * 2;
    double best = 0.0, eff[9];
    int gmax = 1;
    for (int k = 1; k <= 8; ++k) {
        if ((int64_t)k * chunk > B && k > 1 && (int64_t)(k - 1) * chunk >= B) break;
        if ((size_t)k * chunk * row_bytes > ((size_t)1 << 30) && k > 1) break;
        const int64_t rows = (int64_t)k * chunk < B ? (int64_t)k * chunk : B;
        const int64_t tiles = (rows + 128 * cg - 1) / (128 * cg) * n_nt;
        eff[k] = (double)tiles / (double)((tiles + units - 1) / units * units);
        if (eff[k] > best) best = eff[k];
        gmax = k;
    }
    for (int k = 1; k <= gmax; ++k)
        if (eff[k] >= 0.97 * best) return k;
    return 1;
}

SeriesWs carve_series(uint8_t* base, size_t* off, const Geometry& g, int64_t chunk, int64_t B) {
    auto take = [&](size_t bytes) -> void* {
        void* r = base ? base + *off : nullptr;
        *off += align256(bytes);
        return r;
    };
    SeriesWs w;
    w.n_nt = (g.n_rows + ser::BN - 1) / ser::BN;
    w.group = series_group(g, chunk, B, w.n_nt);
    w.group_rows = (int64_t)w.group * chunk < B ? (int64_t)w.group * chunk : B;
    w.n_sets = w.group_rows < B ? 2 : 1;
    w.w32 = (int)((w.group_rows + 127) / 128 * 4);
    w.part_stride = (B + 127) / 128 * 128 + 128;       // whole batch (64 B per sample at config 5): one finishing pass
    w.ctl = (unsigned*)take(SER_CTL_WORDS * sizeof(unsigned));
    w.Bp = (uint16_t*)take((size_t)g.n_rows * SERIES_SEGS * g.M_pad * 2);
    for (int k = 0; k < 2; ++k) {                      // per-group buffers
        if (k < w.n_sets) {
            w.Ap[k] = (uint16_t*)take((size_t)w.group_rows * SERIES_SEGS * g.M_pad * 2);
            w.sigT[k] = (uint32_t*)take((size_t)g.N * w.w32 * 4);
        } else { w.Ap[k] = w.Ap[0]; w.sigT[k] = w.sigT[0]; }
    }
    w.part = (float*)take((size_t)w.n_nt * ser::EPI_HALVES * w.part_stride * 4);
    return w;
}

// per call, after launch_pack_product (Ttab, tau_max): choose K and write the table-row operand
// before launch_pack_product: zero the control block that its row pass fills
cudaError_t launch_series_ctl_reset(const SeriesWs& w, cudaStream_t st) {
    return cudaMemsetAsync(w.ctl, 0, SER_CTL_WORDS * sizeof(unsigned), st);
}

cudaError_t launch_series_pack(const Geometry& g, const float* Ttab, const unsigned* taumax_bits, const SeriesWs& w,
                               bool force, cudaStream_t st) {
    cudaError_t e = series_init();
    if (e != cudaSuccess) return e;
    series_select_kernel<<<1, 1, 0, st>>>(w.ctl, taumax_bits, force ? 1 : 0);
    series_bpow_kernel<<<g.n_rows, 256, 0, st>>>(Ttab, g.M_pad, g.M_eff, w.ctl, w.Bp);
    count_launch(2);
    return cudaGetLastError();
}

// per group of chunks (nb samples), buffer set `set`: the transposed spin bits (preparation; may run on another stream
// than the GEMM)
cudaError_t launch_series_prep(const Geometry& g, const int8_t* sigma, int64_t nb, const SeriesWs& w, int set,
                               cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    ProfScope sc(PH_SERIES_PREP, st);
    const int n_groups = (int)((nb + ser::BM - 1) / ser::BM) * 4;
    const int64_t warps = (int64_t)n_groups * ((g.N + 15) / 16);
    series_bits_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, st>>>(sigma, nb, g.N, w.w32, n_groups, w.ctl, w.sigT[set]);
    count_launch();
    return cudaGetLastError();
}

// per group of chunks (samples s0 .. s0 + nb of the batch): partial local energies per column tile into w.part, from the operand
// rows launch_logpsi left in w.Ap[set] and the bits of launch_series_prep (returns at once when ctl says the path is off)
cudaError_t launch_series_gemm(const Geometry& g, int64_t s0, int64_t nb, const RowInfo* rows, const SeriesWs& w, int set,
                               cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    cudaError_t e = series_init();
    if (e != cudaSuccess) return e;
    const int sms = g_ser_sms[current_device()], pairs = g_ser_pairs[current_device()];
    const int n_mt = (int)((nb + ser::BM - 1) / ser::BM);
    const bool pair = pairs > 0 && n_mt >= 2;              // CTA pairs (cta_group::2) whenever there are two sample tiles
    CUtensorMap map_a, map_b;
    const uint64_t cols = (uint64_t)SERIES_SEGS * g.M_pad;
    if (!encode_u16(&map_a, w.Ap[set], (uint64_t)nb, cols, ser::BM)) return cudaErrorInvalidValue;
    if (!encode_u16(&map_b, w.Bp, (uint64_t)g.n_rows, cols, pair ? ser::BN / 2 : ser::BN)) return cudaErrorInvalidValue;
    SeriesParams p;
    p.ctl = w.ctl; p.rows = rows; p.sigT = w.sigT[set]; p.w32 = w.w32; p.nb = nb; p.n_rows = g.n_rows; p.M_pad = g.M_pad;
    p.n_mt = n_mt; p.n_nt = w.n_nt; p.part = w.part + s0; p.part_stride = w.part_stride;
    ProfScope sc(PH_SERIES_GEMM, st);
    if (pair) {
        const int n_tiles = ((n_mt + 1) / 2) * w.n_nt;
        const int units = n_tiles < pairs ? n_tiles : pairs;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(2 * units), 1, 1);
        cfg.blockDim = dim3(ser::THREADS, 1, 1);
        cfg.dynamicSmemBytes = ser::Cfg<2>::SMEM_BYTES;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, series_gemm_kernel<2>, map_a, map_b, p);
        if (e != cudaSuccess) return e;
    } else {
        const int n_tiles = n_mt * w.n_nt;
        series_gemm_kernel<1><<<n_tiles < sms ? n_tiles : sms, ser::THREADS, ser::Cfg<1>::SMEM_BYTES, st>>>(map_a, map_b, p);
    }
    count_launch();
    return cudaGetLastError();
}

// once per call, after the last chunk: E_loc of the whole batch from the partial sums
cudaError_t launch_series_finish(const Operator* op, const Geometry& g, const int8_t* sigma, int64_t B, const SeriesWs& w,
                                 float* eloc_out, cudaStream_t st) {
    if (B <= 0) return cudaSuccess;
    series_finish_kernel<<<(unsigned)((B + 7) / 8), 256, 0, st>>>(w.part, w.n_nt * ser::EPI_HALVES, w.part_stride, sigma, B, g.N, op->kind,
                                                                 op->d_bonds, op->d_colors, op->d_Jf, op->n_bonds,
                                                                 w.ctl, eloc_out);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
