// Base activations theta = sigma W^T + b on the 5th-generation tensor cores (BASELINE.json
// north_star (2): "the one place tensor cores are justified").
//
// One kernel, two uses, both with int8 operands on tcgen05 kind::i8 (twice the bf16 MMA rate, half the operand bytes)
// and int32 accumulators:
//  * theta: sigma = +-1 IS the A operand (used in place when its rows are a multiple of 128 long).  W (fp32) becomes
//    three int8 digit planes of a fixed-point number, rint(W / q) = d2 2^16 + d1 2^8 + d0, q a power of two tied to
//    max|W| (split_w_i8_kernel); every product and every int32 partial sum is exact, each plane has its own TMEM
//    accumulator, and only the epilogue rounds: theta = q (D2 2^16 + D1 2^8 + D0) + b in fp32.
//  * the contraction over samples of the force vector / QGT (launch_tc_gemm_pieces): A = the transposed spins, the
//    digit planes are those of v = conj(tanh theta) w_s, split the same way per chunk by gradient.cu.
//  History: a bf16 kind::f16 version with three 9-bit fixed-point pieces (27 bits) ran at half the rate with twice
//  the operand bytes; per-ELEMENT bf16 splitting had been measured to bias the result by ~0.25 ulp through the adder's
//  truncation — with integer accumulators there is no adder rounding at all.
//
// Kernel: persistent, one CTA per SM walking over 128 (rows) x 64 (columns) tiles (column tiles fastest: neighbouring
// CTAs share their A rows in L2).  Warp 0 = TMA producer (cp.async.bulk.tensor, 128B swizzle, 4-stage ring: per stage
// the A tile and the three digit tiles of a k block of 128 int8 per row, 40 KB); warp 1 = TMEM allocator and
// single-thread tcgen05.mma issuer: the three digit tiles lie back to back in the stage, so ONE MMA with M = 128,
// N = 192, K = 32 per k step contracts all three planes and reads the A tile from shared memory once (three N = 64
// MMAs, one per plane, read it three times and were measured shared-memory-bandwidth-bound: 547 against 390 us);
// the accumulator columns [0, 64), [64, 128), [128, 192) are D_hi, D_mid, D_lo.  Warps 2-5 = epilogue (tcgen05.ld
// 32x32b, scale / bias, fp32 stores).  The accumulators are double-buffered in TMEM (2 x 192 of the 512 columns), so
// the epilogue of tile i runs under the MMAs of tile i + 1 and the producer runs ahead across tile boundaries; one
// TMEM allocation and one barrier set-up per CTA instead of per tile.  Thread-block clusters of CM x CN CTAs share
// operand tiles by TMA multicast (default 2 x 1: the two CTAs of a tile column load half of every digit tile each).
// (The first version, one CTA per 128 x 128 tile with three 128-column accumulators, the prologue, the MMAs and the
// epilogue in series, took 437 us for the same product.)
#include <cuda.h>

#include <mutex>

#include "nk_internal.h"
#include "ptx_helpers.cuh"
#include "tc_helpers.cuh"

namespace nk {

namespace tc {
constexpr int BM = 128, BN = 64, BKB = 128, STAGES = 4, UMMA_KB = 32;   // BKB: bytes = int8 elements per k-block row
constexpr int A_BYTES = BM * BKB;                         // 16 KB: 128 rows x 128 B
constexpr int P_BYTES = BN * BKB;                         //  8 KB: one digit plane, 64 rows x 128 B
constexpr int STAGE_BYTES = A_BYTES + 3 * P_BYTES;        // sigma + hi + mid + lo
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * 128 * 128 /*output staging*/ + 1024 /*alignment*/ + 256 /*barriers*/;
constexpr int THREADS = 192;
constexpr uint32_t TMEM_COLS = 512;                       // two accumulator sets: D_hi, D_mid, D_lo at +0, +64, +128
constexpr uint32_t ACC_STRIDE = 256;                      // of column 0 and of column 256
// instruction descriptor of kind::i8 (cute::UMMA::InstrDescriptor bit layout): D = S32 (c_format 2), A = B = signed
// 8 bit (format 1), K-major both, N >> 3, M >> 4
constexpr uint32_t IDESC_I8 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)((3 * BN) >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}  // namespace tc

// ---- int8 operands of the theta contraction (tcgen05 kind::i8: twice the bf16 MMA rate, half the operand bytes) ----
// Wq[piece][me][k] (int8, K_pad columns, zero padded): rint(W[me][k] / q_me) = I = d2 2^16 + d1 2^8 + d0 with balanced
// base-256 digits d in [-128, 127].  The scale is PER HIDDEN UNIT (row me of W = output column of theta): q_me is a
// POWER OF TWO, 2^(ex-23) with 2^ex > max_k |W[me][k]| (one step coarser if the row maximum / q would pass 8355000:
// three digits hold |I| <= 8355711), so W / q and q I are exact scalings and every row keeps 23 bits of ITS OWN
// largest entry — with one scale for the whole matrix small rows lost bits (ln psi error 5.4e-6 of the 1e-5 bound at
// config 5).  A scale that is not a power of two was measured to bias every theta by the same 1e-7 relative error,
// which adds up coherently in ln psi.  Pieces stored hi, mid, lo.  The products with sigma = +-1 and their int32 sums
// over k are exact; the residual |W - q I| <= q / 2 <= 2^-23 max_k |W[me][k]|.  The scales q_me follow the three
// planes as M_eff floats (byte offset 3 M_eff K_pad).  A row holding a NaN or an Inf gets q = NaN and zero digits:
// the epilogue's q D + b is then NaN for that hidden unit — non-finite parameters propagate (Q14).
// One block per row: the row maximum first (float bits of |w| order like unsigned integers, NaN above Inf), then the digits.
__global__ void __launch_bounds__(256)
split_w_i8_kernel(const float* __restrict__ Wg, int M_eff, int N, int K_pad, int8_t* __restrict__ Wq) {
    const int me = blockIdx.x;
    const float* row = Wg + (size_t)me * N;
    unsigned m = 0;
    for (int k = threadIdx.x; k < N; k += blockDim.x) m = max(m, __float_as_uint(fabsf(row[k])));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    __shared__ unsigned red[8];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    m = red[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) m = max(m, red[w]);
    const float wmax = __uint_as_float(m);
    int ex = -100;
    float sc, q;
    if (m >= 0x7f800000u) { sc = 0.f; q = __int_as_float(0x7fc00000); }          // NaN / Inf in the row: poison it
    else {
        if (wmax > 0.f) frexpf(wmax, &ex);                // wmax = f 2^ex, f in [0.5, 1)
        if (ldexpf(wmax, 23 - ex) > 8355000.f) ++ex;      // f > 0.996: the top digit would overflow
        if (ex < -100) ex = -100;                         // keep 2^(23 - ex) finite
        sc = ldexpf(1.f, 23 - ex);
        q = ldexpf(1.f, ex - 23);
    }
    const size_t plane = (size_t)M_eff * K_pad;
    for (int k = threadIdx.x; k < K_pad; k += blockDim.x) {
        const float w = (k < N) ? row[k] : 0.f;
        const int I = (m >= 0x7f800000u) ? 0 : (int)rintf(w * sc);
        const int d0 = ((I + 128) & 255) - 128;
        const int I1 = (I - d0) >> 8;
        const int d1 = ((I1 + 128) & 255) - 128;
        const int d2 = (I1 - d1) >> 8;                    // |I| <= 8355000 < 8355711: fits [-128, 127]
        const size_t o = (size_t)me * K_pad + k;
        Wq[o] = (int8_t)d2;
        Wq[plane + o] = (int8_t)d1;
        Wq[2 * plane + o] = (int8_t)d0;
    }
    if (threadIdx.x == 0) reinterpret_cast<float*>(Wq + 3 * plane)[me] = q;
}

// A[s][k] = sigma[s][k] zero padded to K_pad (only needed when N is not a multiple of 128: TMA wants 16-B strides)
__global__ void sigma_pad_i8_kernel(const int8_t* __restrict__ sigma, int64_t B, int N, int K_pad,
                                    int8_t* __restrict__ A) {
    const int64_t total = B * K_pad;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t s = idx / K_pad;
        const int k = (int)(idx - s * K_pad);
        A[idx] = k < N ? sigma[s * N + k] : (int8_t)0;
    }
}

// ---- epilogue of one 128 x 64 output tile (shared by the three kernels below) -----------------------------------------
// out (+)= q (D2 2^16 + D1 2^8 + D0) + bias.  The four epilogue warps (TMEM lane quarter q each) read the three int32
// accumulators, combine them in fp32, write the tile into a 128B-swizzled staging buffer (two boxes of 128 rows x 32
// floats: a thread owns a row, so its eight 16-B chunks per box go to chunk ^ (row & 7) — conflict-free quarter-warps)
// and ONE thread hands it to the TMA engine: a bulk tensor store, or a bulk tensor reduce-add when the product
// accumulates over chunks.  (Until round 2 every thread stored its own row with 16-B STG 8 KB apart: the epilogue, not
// the MMAs, bounded theta-shaped products — 9 k cycles per tile against 3 k of MMAs.)  Rows beyond the operand are
// clipped by the tensor map.  `arrive` hands the accumulator set back to the MMA issuer.
constexpr int TC_STAGE_OUT = 2 * 128 * 128;                // 32 KB staging tile
template <typename Arrive>
__device__ __forceinline__ void tc_epilogue_tile(uint32_t tmem_acc, int q, int lane, bool elected, uint32_t stage_u32,
                                                 uint8_t* stage_ptr, const CUtensorMap* map_out, int row0, int n0,
                                                 const float* __restrict__ bg, const float* __restrict__ scale,
                                                 int scale_per_col, float qs0, int accumulate, Arrive arrive) {
    using namespace tc;
    const int r = q * 32 + lane;
#pragma unroll 1
    for (int c0 = 0; c0 < BN; c0 += 32) {
        // bias and scale of these 32 columns first: their latency runs under the TMEM loads
        float4 bb[8], qs[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            bb[j] = bg != nullptr ? __ldg(reinterpret_cast<const float4*>(bg + n0 + c0) + j) : make_float4(0.f, 0.f, 0.f, 0.f);
            qs[j] = scale_per_col ? __ldg(reinterpret_cast<const float4*>(scale + n0 + c0) + j)
                                  : make_float4(qs0, qs0, qs0, qs0);
        }
        float hi[32], mid[32], lo[32];
        const uint32_t taddr = tmem_acc + ((uint32_t)(q * 32) << 16) + c0;
        tmem_ld32(taddr, hi);
        tmem_ld32(taddr + BN, mid);
        tmem_ld32(taddr + 2 * BN, lo);
        // the two halves of the staging tile alternate: the store of this half issued for the previous tile has finished
        // READING it (at most one newer store — the other half's — may still be in flight)
        if (elected) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
        asm volatile("bar.sync 1, 128;" ::: "memory");
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (c0 + 32 == BN) {                               // everything is in registers: hand the set back to the MMAs
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            arrive();
        }
        const int bx = c0 >> 5;
        uint8_t* box = stage_ptr + bx * (128 * 128) + r * 128;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            float4 o;
            auto comb = [&](int jj) -> float {             // exact ints below 2^24 each
                const float h = (float)__float_as_int(hi[jj]), m = (float)__float_as_int(mid[jj]),
                            l = (float)__float_as_int(lo[jj]);
                return fmaf(h, 65536.f, fmaf(m, 256.f, l));
            };
            o.x = fmaf(qs[j].x, comb(4 * j), bb[j].x); o.y = fmaf(qs[j].y, comb(4 * j + 1), bb[j].y);
            o.z = fmaf(qs[j].z, comb(4 * j + 2), bb[j].z); o.w = fmaf(qs[j].w, comb(4 * j + 3), bb[j].w);
            *reinterpret_cast<float4*>(box + ((j ^ (r & 7)) << 4)) = o;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy writes -> visible to the TMA engine
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (elected) {
            if (accumulate)
                asm volatile("cp.reduce.async.bulk.tensor.2d.global.shared::cta.add.tile.bulk_group [%0, {%1, %2}], [%3];"
                             ::"l"(map_out), "r"(n0 + c0), "r"(row0), "r"(stage_u32 + bx * (128 * 128))
                             : "memory");
            else
                asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];"
                             ::"l"(map_out), "r"(n0 + c0), "r"(row0), "r"(stage_u32 + bx * (128 * 128))
                             : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
}
// before the CTA exits: the last store has read the staging buffer
__device__ __forceinline__ void tc_epilogue_drain(bool elected) {
    if (elected) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// ---- the GEMM ---------------------------------------------------------------------------------------------
// int8 operands (128 elements per 128-B swizzle row, so K_pad / 128 k blocks), int32 accumulators,
// out (+)= q (D2 2^16 + D1 2^8 + D0) + bias with the scale q read from `scale`.
// A cluster of CM x CN CTAs (rank = rm CN + rn) works on CM x CN neighbouring tiles: the CN CTAs of a tile row share
// their A tile (each loads 1 / CN of its rows and multicasts it), the CM CTAs of a tile column share the three digit
// tiles (each loads 1 / CM of the rows of every plane).  A stage of a CTA is therefore written by CM + CN - 1 CTAs
// (itself included), and the MMA commit that frees the stage arrives on the `empty` barrier of every one of them.
template <int CM, int CN>
__global__ void __launch_bounds__(tc::THREADS, 1)
theta_tc_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_w,
                const __grid_constant__ CUtensorMap map_out, int64_t B,
                int M_eff, int K_pad, const float* __restrict__ bg, float* __restrict__ theta, int accumulate,
                const float* __restrict__ scale, int scale_per_col, int n_sup_n, int n_sup) {
    using namespace tc;
    constexpr int CS = CM * CN;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;            // SWIZZLE_128B needs 1024 B
    const uint32_t bars = smem_base + STAGES * STAGE_BYTES + TC_STAGE_OUT;       // ring | output staging tile | barriers
    const uint32_t full0 = bars, empty0 = bars + 8 * STAGES;                     // smem ring
    const uint32_t tfull0 = bars + 16 * STAGES, tempty0 = tfull0 + 16;          // the two accumulator sets
    const uint32_t tmem_slot = tempty0 + 16;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_kb = K_pad / BKB;
    const int rank = CS > 1 ? (int)cluster_ctarank() : 0;
    const int rm = rank / CN, rn = rank - rm * CN;
    const int cluster_id = blockIdx.x / CS, n_clusters = gridDim.x / CS;
    uint16_t mask_a = 0, mask_w = 0;
#pragma unroll
    for (int j = 0; j < CN; ++j) mask_a |= (uint16_t)(1u << (rm * CN + j));
#pragma unroll
    for (int i = 0; i < CM; ++i) mask_w |= (uint16_t)(1u << (i * CN + rn));

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, CM + CN - 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(tfull0 + 8 * a, 1); mbar_init(tempty0 + 8 * a, 128); }
        mbar_fence_init();
    }
    if (warp == 1) {   // TMEM allocation by one full warp; the base address lands in shared memory
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (CS > 1) cluster_sync_all();                       // every CTA's barriers exist before anything is multicast
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===== TMA producer: runs ahead of the MMAs across tile boundaries =====
        if (lane == 0) {
            int stage = 0; uint32_t parity = 1;
            for (int sup = cluster_id; sup < n_sup; sup += n_clusters) {
                const int sm = sup / n_sup_n;
                const int m0 = (sm * CM + rm) * BM, n0 = ((sup - sm * n_sup_n) * CN + rn) * BN;
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(empty0 + 8 * stage, parity);
                    mbar_arrive_expect_tx(full0 + 8 * stage, STAGE_BYTES);
                    const uint32_t dst = smem_base + stage * STAGE_BYTES;
                    if (CN > 1)
                        tma_load_2d_mc(dst + rn * (A_BYTES / CN), &map_a, kb * BKB, m0 + rn * (BM / CN),
                                       full0 + 8 * stage, mask_a);
                    else
                        tma_load_2d(dst, &map_a, kb * BKB, m0, full0 + 8 * stage);
#pragma unroll
                    for (int pc = 0; pc < 3; ++pc) {
                        if (CM > 1)
                            tma_load_2d_mc(dst + A_BYTES + pc * P_BYTES + rm * (P_BYTES / CM), &map_w, kb * BKB,
                                           pc * M_eff + n0 + rm * (BN / CM), full0 + 8 * stage, mask_w);
                        else
                            tma_load_2d(dst + A_BYTES + pc * P_BYTES, &map_w, kb * BKB, pc * M_eff + n0,
                                        full0 + 8 * stage);
                    }
                    if (++stage == STAGES) { stage = 0; parity ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one thread) =====
        if (lane == 0) {
            int stage = 0; uint32_t parity = 0;
            int it = 0;
            for (int sup = cluster_id; sup < n_sup; sup += n_clusters, ++it) {
                const int set = it & 1;
                mbar_wait(tempty0 + 8 * set, ((it >> 1) & 1) ^ 1);      // the epilogue has drained this set (free at first)
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t acc = tmem_base + set * ACC_STRIDE;
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(full0 + 8 * stage, parity);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t a_addr = smem_base + stage * STAGE_BYTES;
#pragma unroll
                    for (int k = 0; k < BKB / UMMA_KB; ++k) {
                        const uint32_t koff = k * UMMA_KB;                      // bytes inside the 128 B swizzle row
                        const uint64_t ad = make_sdesc(a_addr + koff);
                        const uint32_t first = (kb | k) ? 1u : 0u;
                        // 32 B = 32 int8 = one K = 32 MMA; the three digit tiles lie back to back in the stage, so ONE
                        // MMA with N = 3 BN takes them as a single B operand and reads the A tile once instead of thrice
                        umma_i8(acc, ad, make_sdesc(a_addr + A_BYTES + koff), IDESC_I8, first);
                    }
                    // frees the stage, here and in the CTAs that multicast into it, once these MMAs have read it
                    if (CS > 1) umma_commit_mc(empty0 + 8 * stage, (uint16_t)(mask_a | mask_w));
                    else umma_commit(empty0 + 8 * stage);
                    if (++stage == STAGES) { stage = 0; parity ^= 1; }
                }
                umma_commit(tfull0 + 8 * set);            // this tile's accumulators are complete
            }
        }
    } else {
        // ===== epilogue: warps 2..5, TMEM lane quarter = warp % 4 =====
        const int q = warp & 3;
        const float qs0 = *scale;                         // one scale, or (scale_per_col) one per output column
        const bool elected = warp == 2 && lane == 0;
        const uint32_t stage_u32 = smem_base + STAGES * STAGE_BYTES;
        uint8_t* stage_ptr = smem_raw + (stage_u32 - smem_u32(smem_raw));
        int it = 0;
        for (int sup = cluster_id; sup < n_sup; sup += n_clusters, ++it) {
            const int set = it & 1;
            const int sm = sup / n_sup_n;
            const int n0 = ((sup - sm * n_sup_n) * CN + rn) * BN;
            mbar_wait(tfull0 + 8 * set, (it >> 1) & 1);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            tc_epilogue_tile(tmem_base + set * ACC_STRIDE, q, lane, elected, stage_u32, stage_ptr, &map_out,
                             (sm * CM + rm) * BM, n0, bg, scale, scale_per_col, qs0, accumulate,
                             [&]() { mbar_arrive(tempty0 + 8 * set); });
        }
        tc_epilogue_drain(elected);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (CS > 1) cluster_sync_all();                       // no peer still multicasts into, or arrives on, this CTA
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
    }
}

// ---- the same contraction by CTA PAIRS (tcgen05 cta_group::2) ------------------------------------------------------
// A pair of CTAs of one TPC owns 256 rows x 64 output columns: each CTA holds its 128 rows' A tile and HALF of the B
// operand — rows [96 r, 96 r + 96) of the 192 digit rows (hi | mid | lo) x 64 columns, three TMA boxes of 32 rows — so
// a stage is 28 KB instead of 40 and the digit planes cross L2 -> shared memory -> tensor core once per 256 rows.  What
// bounded the single-CTA kernel was shared-memory bandwidth (40 KB of MMA reads + 40 KB of TMA writes = 625 cycles per k
// block against 384 MMA cycles); here it is 28 + 28 KB.  The leader (rank 0) issues M = 256, N = 192,
// K = 32 MMAs; both CTAs' loads count on the leader's `full` barrier, multicast commits free the stage and publish the
// accumulators in both, and both CTAs' epilogue warps hand the accumulator set back on the leader's `tempty`.
namespace tc2 {
constexpr int STAGES = 6;
constexpr int B_HALF = 96 * tc::BKB;                       // 12 KB
constexpr int STAGE_BYTES = tc::A_BYTES + B_HALF;          // 28 KB
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * 128 * 128 + 1024 + 256;
constexpr uint32_t IDESC_I8 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)((3 * tc::BN) >> 3) << 17) | ((uint32_t)((2 * tc::BM) >> 4) << 24);
}  // namespace tc2

__device__ __forceinline__ void umma_i8_cg2(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                            uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::i8 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}

__global__ void __launch_bounds__(tc::THREADS, 1)
theta_tc2_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_w,
                 const __grid_constant__ CUtensorMap map_out, int64_t B,
                 int M_eff, int K_pad, const float* __restrict__ bg, float* __restrict__ theta, int accumulate,
                 const float* __restrict__ scale, int scale_per_col, int n_tn, int n_tiles) {
    using namespace tc;
    constexpr int STAGES2 = tc2::STAGES, STAGE2 = tc2::STAGE_BYTES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bars = smem_base + STAGES2 * STAGE2 + TC_STAGE_OUT;
    const uint32_t full0 = bars, empty0 = bars + 8 * STAGES2;
    const uint32_t tfull0 = bars + 16 * STAGES2, tempty0 = tfull0 + 16;
    const uint32_t tmem_slot = tempty0 + 16;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_kb = K_pad / BKB;
    const uint32_t rank = cluster_ctarank();
    const int unit = blockIdx.x / 2, n_units = gridDim.x / 2;
    const uint32_t full_l = map_to_rank(full0, 0), tempty_l = map_to_rank(tempty0, 0);

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES2; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(tfull0 + 8 * a, 1); mbar_init(tempty0 + 8 * a, 256); }
        mbar_fence_init();
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    cluster_sync_all();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===== TMA producer (each CTA: its A rows and its half of the digit rows) =====
        if (lane == 0) {
            int stage = 0; uint32_t parity = 1;
            for (int t = unit; t < n_tiles; t += n_units) {
                const int tm = t / n_tn;
                const int m0 = (tm * 2 + (int)rank) * BM, n0 = (t - tm * n_tn) * BN;
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(empty0 + 8 * stage, parity);
                    if (rank == 0) mbar_arrive_expect_tx(full0 + 8 * stage, 2 * STAGE2);
                    const uint32_t dst = smem_base + stage * STAGE2;
                    tma_load_2d_cg2(dst, &map_a, kb * BKB, m0, full_l + 8 * stage);
#pragma unroll
                    for (int bx = 0; bx < 3; ++bx) {       // digit row v = 96 rank + 32 bx .. + 31 of (hi | mid | lo) x 64
                        const int v = 96 * (int)rank + 32 * bx;
                        tma_load_2d_cg2(dst + A_BYTES + bx * 32 * BKB, &map_w, kb * BKB, (v >> 6) * M_eff + n0 + (v & 63),
                                        full_l + 8 * stage);
                    }
                    if (++stage == STAGES2) { stage = 0; parity ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one thread of the leader) =====
        if (lane == 0 && rank == 0) {
            int stage = 0; uint32_t parity = 0;
            int it = 0;
            for (int t = unit; t < n_tiles; t += n_units, ++it) {
                const int set = it & 1;
                mbar_wait(tempty0 + 8 * set, ((it >> 1) & 1) ^ 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t acc = tmem_base + set * ACC_STRIDE;
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(full0 + 8 * stage, parity);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t a_addr = smem_base + stage * STAGE2;
#pragma unroll
                    for (int k = 0; k < BKB / UMMA_KB; ++k) {
                        const uint32_t koff = k * UMMA_KB;
                        umma_i8_cg2(acc, make_sdesc(a_addr + koff), make_sdesc(a_addr + A_BYTES + koff), tc2::IDESC_I8,
                                    (kb | k) ? 1u : 0u);
                    }
                    umma_commit_cg2(empty0 + 8 * stage);
                    if (++stage == STAGES2) { stage = 0; parity ^= 1; }
                }
                umma_commit_cg2(tfull0 + 8 * set);
            }
        }
    } else {
        // ===== epilogue: warps 2..5 of each CTA, its own 128 rows =====
        const int q = warp & 3;
        const float qs0 = *scale;
        const bool elected = warp == 2 && lane == 0;
        const uint32_t stage_u32 = smem_base + STAGES2 * STAGE2;
        uint8_t* stage_ptr = smem_raw + (stage_u32 - smem_u32(smem_raw));
        int it = 0;
        for (int t = unit; t < n_tiles; t += n_units, ++it) {
            const int set = it & 1;
            const int tm = t / n_tn;
            const int n0 = (t - tm * n_tn) * BN;
            mbar_wait(tfull0 + 8 * set, (it >> 1) & 1);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            tc_epilogue_tile(tmem_base + set * ACC_STRIDE, q, lane, elected, stage_u32, stage_ptr, &map_out,
                             (tm * 2 + (int)rank) * BM, n0, bg, scale, scale_per_col, qs0, accumulate,
                             [&]() { mbar_arrive_cluster(tempty_l + 8 * set); });
        }
        tc_epilogue_drain(elected);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    cluster_sync_all();
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
    }
}

// ---- theta-shaped products (k extent <= 1024 bytes): CTA pairs with the A operand RESIDENT in shared memory ----------
// theta = sigma W^T has a short k extent (N <= 1024 spins = 8 k blocks) and many output columns, so the streaming kernels
// above read every spin tile once per 64-column tile — 32 times at M = 2048 — and are bound by L2 -> shared-memory
// traffic (ncu: L2 63 %, tensor pipe 46 % on the 65536 x 2048 x 1024 launch).  Here a CTA pair loads the spins of its
// 256 rows ONCE (n_kb x 16 KB per CTA, kept for all the column tiles of its work range) and streams only its half of the
// digit rows (12 KB per k block): per k block a CTA writes 12 KB and the MMAs read 28 KB = 312 shared-memory cycles
// against 384 MMA cycles, and the pair pulls 24 KB instead of 56 KB through L2.  Work = (row-pair tile, column tile)
// items, column tiles fastest; pair u takes a contiguous range of them (the spins are reloaded when the row tile changes).
namespace tc3 {
constexpr int MAX_KB = 8;                                  // resident k blocks: K_pad <= 1024
constexpr int STAGES = 4;
constexpr int B_HALF = 96 * tc::BKB;                       // 12 KB
constexpr int SMEM_BYTES = MAX_KB * tc::A_BYTES + STAGES * B_HALF + 2 * 128 * 128 + 1024 + 256;
}  // namespace tc3

__global__ void __launch_bounds__(tc::THREADS, 1)
theta_tc3_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_w,
                 const __grid_constant__ CUtensorMap map_out, int64_t B,
                 int M_eff, int K_pad, const float* __restrict__ bg, float* __restrict__ theta, int accumulate,
                 const float* __restrict__ scale, int scale_per_col, int n_tn, int n_items, int per_unit) {
    using namespace tc;
    constexpr int STG = tc3::STAGES, BH = tc3::B_HALF;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t b_ring = smem_base + tc3::MAX_KB * A_BYTES;
    const uint32_t bars = b_ring + STG * BH + TC_STAGE_OUT;
    const uint32_t full0 = bars, empty0 = bars + 8 * STG;
    const uint32_t tfull0 = bars + 16 * STG, tempty0 = tfull0 + 16;
    const uint32_t afull = tempty0 + 16, aempty = afull + 8;
    const uint32_t tmem_slot = aempty + 8;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_kb = K_pad / BKB;
    const uint32_t rank = cluster_ctarank();
    const int unit = blockIdx.x / 2;
    const int item_lo = unit * per_unit, item_hi = min(n_items, item_lo + per_unit);
    const uint32_t full_l = map_to_rank(full0, 0), tempty_l = map_to_rank(tempty0, 0), afull_l = map_to_rank(afull, 0);

    if (threadIdx.x == 0) {
        for (int s = 0; s < STG; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(tfull0 + 8 * a, 1); mbar_init(tempty0 + 8 * a, 256); }
        mbar_init(afull, 1);
        mbar_init(aempty, 1);
        mbar_fence_init();
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    cluster_sync_all();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            int stage = 0; uint32_t parity = 1, a_parity = 1;
            int cur_tm = -1;
            for (int it = item_lo; it < item_hi; ++it) {
                const int tm = it / n_tn;
                const int n0 = (it - tm * n_tn) * BN;
                if (tm != cur_tm) {                        // the spins of this pair's 256 rows, once per row tile
                    cur_tm = tm;
                    mbar_wait(aempty, a_parity);
                    a_parity ^= 1;
                    if (rank == 0) mbar_arrive_expect_tx(afull, 2 * n_kb * A_BYTES);
                    const int m0 = (tm * 2 + (int)rank) * BM;
                    for (int kb = 0; kb < n_kb; ++kb)
                        tma_load_2d_cg2(smem_base + kb * A_BYTES, &map_a, kb * BKB, m0, afull_l);
                }
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(empty0 + 8 * stage, parity);
                    if (rank == 0) mbar_arrive_expect_tx(full0 + 8 * stage, 2 * BH);
                    const uint32_t dst = b_ring + stage * BH;
#pragma unroll
                    for (int bx = 0; bx < 3; ++bx) {       // digit row v = 96 rank + 32 bx .. + 31 of (hi | mid | lo) x 64
                        const int v = 96 * (int)rank + 32 * bx;
                        tma_load_2d_cg2(dst + bx * 32 * BKB, &map_w, kb * BKB, (v >> 6) * M_eff + n0 + (v & 63),
                                        full_l + 8 * stage);
                    }
                    if (++stage == STG) { stage = 0; parity ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one thread of the leader) =====
        if (lane == 0 && rank == 0) {
            int stage = 0; uint32_t parity = 0, a_parity = 0;
            int cur_tm = -1, n = 0;
            for (int it = item_lo; it < item_hi; ++it, ++n) {
                const int tm = it / n_tn;
                if (tm != cur_tm) {
                    cur_tm = tm;
                    mbar_wait(afull, a_parity);
                    a_parity ^= 1;
                }
                const int set = n & 1;
                mbar_wait(tempty0 + 8 * set, ((n >> 1) & 1) ^ 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t acc = tmem_base + set * ACC_STRIDE;
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(full0 + 8 * stage, parity);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t a_addr = smem_base + kb * A_BYTES, b_addr = b_ring + stage * BH;
#pragma unroll
                    for (int k = 0; k < BKB / UMMA_KB; ++k) {
                        const uint32_t koff = k * UMMA_KB;
                        umma_i8_cg2(acc, make_sdesc(a_addr + koff), make_sdesc(b_addr + koff), tc2::IDESC_I8,
                                    (kb | k) ? 1u : 0u);
                    }
                    umma_commit_cg2(empty0 + 8 * stage);
                    if (++stage == STG) { stage = 0; parity ^= 1; }
                }
                umma_commit_cg2(tfull0 + 8 * set);
                if (it + 1 == item_hi || (it + 1) / n_tn != tm) umma_commit_cg2(aempty);   // the spins may be replaced
            }
        }
    } else {
        // ===== epilogue: warps 2..5 of each CTA, its own 128 rows =====
        const int q = warp & 3;
        const float qs0 = *scale;
        const bool elected = warp == 2 && lane == 0;
        const uint32_t stage_u32 = b_ring + STG * BH;
        uint8_t* stage_ptr = smem_raw + (stage_u32 - smem_u32(smem_raw));
        int n = 0;
        for (int it = item_lo; it < item_hi; ++it, ++n) {
            const int set = n & 1;
            const int tm = it / n_tn;
            const int n0 = (it - tm * n_tn) * BN;
            mbar_wait(tfull0 + 8 * set, (n >> 1) & 1);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            tc_epilogue_tile(tmem_base + set * ACC_STRIDE, q, lane, elected, stage_u32, stage_ptr, &map_out,
                             (tm * 2 + (int)rank) * BM, n0, bg, scale, scale_per_col, qs0, accumulate,
                             [&]() { mbar_arrive_cluster(tempty_l + 8 * set); });
        }
        tc_epilogue_drain(elected);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    cluster_sync_all();
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
    }
}

// ---- host side ---------------------------------------------------------------------------------------------
static bool encode_2d(CUtensorMap* map, const void* base, uint64_t rows, uint64_t cols, int box_rows);
// One-time set-up is per DEVICE (function attributes, SM and cluster counts belong to the current device) and guarded
// by a mutex: a process may drive several GPUs, and first calls may come from several host threads.
namespace {
struct TcDevice { bool ready = false; int num_sms = 148, cm = 1, cn = 1, max_clusters = 148, pairs = 0; };
std::mutex g_tc_mutex;
TcDevice g_tc_dev[NK_MAX_DEVICES];
EncodeTiledFn g_encode = nullptr;
}  // namespace
#define g_num_sms (tc_dev().num_sms)
#define g_cm (tc_dev().cm)
#define g_cn (tc_dev().cn)
#define g_max_clusters (tc_dev().max_clusters)
static TcDevice& tc_dev() { return g_tc_dev[current_device()]; }

EncodeTiledFn tensor_map_encoder() {
    std::lock_guard<std::mutex> lock(g_tc_mutex);
    if (g_encode == nullptr) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            g_encode = (EncodeTiledFn)fn;
    }
    return g_encode;
}

template <int CM, int CN>
static cudaError_t tc_prepare(int* max_clusters) {
    const void* fn = (const void*)theta_tc_kernel<CM, CN>;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(CM * CN, 1, 1);
    cfg.blockDim = dim3(tc::THREADS, 1, 1);
    cfg.dynamicSmemBytes = tc::SMEM_BYTES;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CM * CN; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaOccupancyMaxActiveClusters(max_clusters, fn, &cfg);
}

template <int CM, int CN>
static cudaError_t tc_launch(const CUtensorMap& map_a, const CUtensorMap& map_w, const CUtensorMap& map_out,
                             int64_t rows, int cols, int k_len,
                             const float* bg, float* out, int accumulate, const float* scale, int scale_per_col,
                             cudaStream_t st) {
    const int n_sup_n = cols / (tc::BN * CN);
    const int64_t n_sup = (rows + (int64_t)tc::BM * CM - 1) / ((int64_t)tc::BM * CM) * n_sup_n;
    if (n_sup > 0x7fffffff) return cudaErrorInvalidValue;
    const int n_clusters = (int)(n_sup < g_max_clusters ? n_sup : g_max_clusters);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(n_clusters * CM * CN), 1, 1);
    cfg.blockDim = dim3(tc::THREADS, 1, 1);
    cfg.dynamicSmemBytes = tc::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CM * CN; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, theta_tc_kernel<CM, CN>, map_a, map_w, map_out, rows, cols, k_len, bg, out, accumulate, scale,
                              scale_per_col, n_sup_n, (int)n_sup);
}

cudaError_t theta_tc_init() {
    if (tensor_map_encoder() == nullptr) return cudaErrorNotSupported;
    std::lock_guard<std::mutex> lock(g_tc_mutex);
    if (tc_dev().ready) return cudaSuccess;
    cudaError_t e;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
        sms > 0)
        g_num_sms = sms;
    // cluster shape: 2 x 1 (measured best at 65536 x 2048 x 1024: 374 us against 390 for 1 x 1, 394 for 2 x 2, 403 for
    // 4 x 1 and 4 x 2) unless the device cannot co-schedule such clusters; NK_TC_CLUSTER ("1x1", "2x1", "2x2", "4x1",
    // "4x2") overrides it in -DNK_DEBUG builds only
    int want_m = 2, want_n = 1;
#ifdef NK_DEBUG
    if (const char* v = getenv("NK_TC_CLUSTER")) {
        if (v[0] >= '1' && v[0] <= '4' && v[1] == 'x' && v[2] >= '1' && v[2] <= '2') { want_m = v[0] - '0'; want_n = v[2] - '0'; }
    }
#endif
    int n = 0;
    g_cm = g_cn = 1;
    if (want_m == 4 && want_n == 2 && tc_prepare<4, 2>(&n) == cudaSuccess && n > 0) { g_cm = 4; g_cn = 2; }
    else if (want_m == 4 && want_n == 1 && tc_prepare<4, 1>(&n) == cudaSuccess && n > 0) { g_cm = 4; g_cn = 1; }
    else if (want_m == 2 && want_n == 2 && tc_prepare<2, 2>(&n) == cudaSuccess && n > 0) { g_cm = 2; g_cn = 2; }
    else if (want_m == 2 && want_n == 1 && tc_prepare<2, 1>(&n) == cudaSuccess && n > 0) { g_cm = 2; g_cn = 1; }
    (void)cudaGetLastError();                              // a refused cluster shape is not an error of the call
    if (g_cm * g_cn == 1) {
        e = tc_prepare<1, 1>(&n);
        if (e != cudaSuccess) return e;
        if (n <= 0) n = g_num_sms;
    }
    g_max_clusters = n;
    {   // CTA pairs for the cta_group::2 kernel
        int np = 0;
        if (cudaFuncSetAttribute((const void*)theta_tc2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 tc2::SMEM_BYTES) == cudaSuccess &&
            cudaFuncSetAttribute((const void*)theta_tc3_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 tc3::SMEM_BYTES) == cudaSuccess) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(2, 1, 1); cfg.blockDim = dim3(tc::THREADS, 1, 1); cfg.dynamicSmemBytes = tc2::SMEM_BYTES;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
            cfg.attrs = attr; cfg.numAttrs = 1;
            if (cudaOccupancyMaxActiveClusters(&np, (const void*)theta_tc2_kernel, &cfg) != cudaSuccess) np = 0;
        }
        (void)cudaGetLastError();
        tc_dev().pairs = np;
    }
    tc_dev().ready = true;
    return cudaSuccess;
}

static cudaError_t tc_gemm(const void* A, int64_t rows, const void* P, int cols, int ld, int k_len, const float* bg,
                           float* out, int accumulate, int scale_per_col, cudaStream_t st) {
    cudaError_t e = theta_tc_init();
    if (e != cudaSuccess) return e;
    CUtensorMap map_a, map_p, map_out;
    {   // fp32 output [rows][cols], box = 128 rows x 32 floats (128 B), 128B swizzle: the epilogue's staging layout
        const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
        const cuuint64_t strides[1] = {(cuuint64_t)cols * 4};
        const cuuint32_t box[2] = {32, 128};
        const cuuint32_t estr[2] = {1, 1};
        if (g_encode(&map_out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, out, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return cudaErrorInvalidValue;
    }
    // CTA pairs (cta_group::2) whenever there are two row tiles: the resident-A kernel for short k extents (theta-shaped
    // products), the streaming one for long ones (the contractions over samples); the single-CTA cluster kernel otherwise
    const bool resident = k_len <= tc3::MAX_KB * tc::BKB;
    if (tc_dev().pairs > 0 && rows > tc::BM && (resident || k_len >= 4096)) {
        if (!encode_2d(&map_a, A, (uint64_t)rows, (uint64_t)ld, tc::BM)) return cudaErrorInvalidValue;
        if (!encode_2d(&map_p, P, (uint64_t)3 * cols, (uint64_t)ld, 32)) return cudaErrorInvalidValue;
        const float* scale2 = reinterpret_cast<const float*>((const int8_t*)P + (size_t)3 * cols * ld);
        const int n_tn = cols / tc::BN;
        const int64_t n_tiles = (rows + 2 * tc::BM - 1) / (2 * tc::BM) * n_tn;
        if (n_tiles > 0x7fffffff) return cudaErrorInvalidValue;
        const int units = (int)(n_tiles < tc_dev().pairs ? n_tiles : tc_dev().pairs);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(2 * units), 1, 1);
        cfg.blockDim = dim3(tc::THREADS, 1, 1);
        cfg.dynamicSmemBytes = resident ? tc3::SMEM_BYTES : tc2::SMEM_BYTES;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        if (resident) {
            const int per_unit = (int)((n_tiles + units - 1) / units);
            e = cudaLaunchKernelEx(&cfg, theta_tc3_kernel, map_a, map_p, map_out, rows, cols, k_len, bg, out, accumulate, scale2,
                                   scale_per_col, n_tn, (int)n_tiles, per_unit);
        } else {
            e = cudaLaunchKernelEx(&cfg, theta_tc2_kernel, map_a, map_p, map_out, rows, cols, k_len, bg, out, accumulate, scale2,
                                   scale_per_col, n_tn, (int)n_tiles);
        }
        count_launch();
        return e != cudaSuccess ? e : cudaGetLastError();
    }
    if (!encode_2d(&map_a, A, (uint64_t)rows, (uint64_t)ld, tc::BM / g_cn)) return cudaErrorInvalidValue;
    if (!encode_2d(&map_p, P, (uint64_t)3 * cols, (uint64_t)ld, tc::BN / g_cm)) return cudaErrorInvalidValue;
    const float* scale = reinterpret_cast<const float*>((const int8_t*)P + (size_t)3 * cols * ld);
    if (g_cm == 4 && g_cn == 2) e = tc_launch<4, 2>(map_a, map_p, map_out, rows, cols, k_len, bg, out, accumulate, scale, scale_per_col, st);
    else if (g_cm == 4) e = tc_launch<4, 1>(map_a, map_p, map_out, rows, cols, k_len, bg, out, accumulate, scale, scale_per_col, st);
    else if (g_cm == 2 && g_cn == 2) e = tc_launch<2, 2>(map_a, map_p, map_out, rows, cols, k_len, bg, out, accumulate, scale, scale_per_col, st);
    else if (g_cm == 2) e = tc_launch<2, 1>(map_a, map_p, map_out, rows, cols, k_len, bg, out, accumulate, scale, scale_per_col, st);
    else e = tc_launch<1, 1>(map_a, map_p, map_out, rows, cols, k_len, bg, out, accumulate, scale, scale_per_col, st);
    count_launch();
    return e != cudaSuccess ? e : cudaGetLastError();
}

// 2-D tensor map over a k-contiguous int8 [rows][cols] operand, box = box_rows rows x 128 B, 128B swizzle
static bool encode_2d(CUtensorMap* map, const void* base, uint64_t rows, uint64_t cols, int box_rows) {
    const cuuint64_t dims[2] = {cols, rows};
    const cuuint64_t strides[1] = {cols};
    const cuuint32_t box[2] = {(cuuint32_t)tc::BKB, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return g_encode(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2,
                    const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// W -> three int8 planes + one scale per row (K_pad a multiple of 128); the buffer must hold 3 M_eff K_pad + 4 M_eff bytes
cudaError_t launch_split_w(const float* Wg, int M_eff, int N, int K_pad, void* Ws, cudaStream_t st) {
    split_w_i8_kernel<<<M_eff, 256, 0, st>>>(Wg, M_eff, N, K_pad, (int8_t*)Ws);
    count_launch();
    return cudaGetLastError();
}

// the spins as the A operand: sigma itself when its rows are already K_pad long, else a zero-padded int8 copy in A
cudaError_t launch_sigma_operand(const int8_t* sigma, int64_t B, int N, int K_pad, void* A, cudaStream_t st) {
    if (B <= 0) return cudaSuccess;
    const int64_t total = B * K_pad;
    int64_t blocks = (total + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    sigma_pad_i8_kernel<<<(unsigned)blocks, 256, 0, st>>>(sigma, B, N, K_pad, (int8_t*)A);
    count_launch();
    return cudaGetLastError();
}

// theta[s][m] = bg[m] + sum_k A[s][k] W[m][k] with A an int8 [B][K_pad] operand (see launch_sigma_operand) and Ws the
// planes of launch_split_w
cudaError_t launch_theta_tc_pre(const void* A, int64_t B, int M_eff, int K_pad, const void* Ws, const float* bg,
                                float* theta, cudaStream_t st) {
    if (B <= 0) return cudaSuccess;
    return tc_gemm(A, B, Ws, M_eff, K_pad, K_pad, bg, theta, 0, 1, st);
}

cudaError_t launch_theta_tc(const int8_t* sigma, int64_t B, int N, int M_eff, int K_pad, const void* Ws, void* A,
                            const float* bg, float* theta, cudaStream_t st) {
    if (B <= 0) return cudaSuccess;
    if (N == K_pad && ((uintptr_t)sigma & 15) == 0)                      // rows already padded and 16-B aligned
        return launch_theta_tc_pre(sigma, B, M_eff, K_pad, Ws, bg, theta, st);
    cudaError_t e = launch_sigma_operand(sigma, B, N, K_pad, A, st);
    if (e != cudaSuccess) return e;
    return launch_theta_tc_pre(A, B, M_eff, K_pad, Ws, bg, theta, st);
}

// Generic entry used by the gradient / QGT contraction over samples: out[r][c] (+)= q sum_k A[r][k] I[c][k] with A an
// int8 [rows][ld] operand (the transposed spins) and P the three int8 digit planes [3][cols][ld] + scale q of
// I = rint(v / q) (grad_split_T_kernel); k < k_len (a multiple of 128), cols a multiple of 128.
cudaError_t launch_tc_gemm_pieces(const void* A, int64_t rows, const void* P, int cols, int ld, int k_len, float* out,
                                  int accumulate, cudaStream_t st) {
    if (rows <= 0) return cudaSuccess;
    return tc_gemm(A, rows, P, cols, ld, k_len, nullptr, out, accumulate, 0, st);
}

}  // namespace nk
