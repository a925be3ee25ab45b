// Metropolis-Hastings sampler for the RBM (Sec. 3.4):
//   P_acc(s -> s') = min(1, |psi(s')|^2 / |psi(s)|^2)       Eq. (20) L709 (local flips / exchanges: symmetric kernels)
//   MetropolisLocal: negate one spin; MetropolisExchange: swap the spins of one pair of a cluster list     L713
// One warp owns one chain for the whole call (n_chains = n_samples, L1583): theta_s = KAPPA theta lives in registers
// exactly as in the fused local-energy kernel (rbm_lane_state.cuh), a proposal costs one row of the table Dtab
// (theta' = theta - 2 s_k W[:,k], or - 2 s_i (W[:,i] - W[:,j])).  Every chain needs a different row at every
// transition, so rows are not shared between warps; instead each warp owns two row buffers in shared memory and,
// while it evaluates one proposal, a bulk async copy (TMA engine, completing on the warp's own mbarrier) already
// brings the row of its next non-trivial proposal from L2 — proposal indices do not depend on the state, and whether
// a coming exchange is trivial is judged on the current spins (a rare misjudgement costs one wasted or one late
// copy, never a wrong result; rows of <= 4 KB are read straight from L2 by 16 warps instead, which measured faster).
// An accepted move re-reads the row and overwrites theta in place.  ln psi is never formed: the ratio psi'/psi comes
// out of the same 1-MUFU-per-pair product as in fused_eloc.cu.
//
// Random numbers (S1-S3): Philox4x32-10, counter = (chain lo, hi, transition lo, hi), key = (seed lo, hi)
//   proposal index = umulhi(r0, n);  u = ((r1 >> 9) + 1/2) 2^-23;  accept iff u < |psi'/psi|^2 (fp32).
// Lane l draws for transition t0 + l, so one Philox evaluation per lane serves 32 transitions of the chain.
#include <type_traits>

#include "nk_internal.h"
#include "ptx_helpers.cuh"
#include "rbm_lane_state.cuh"

namespace nk {

constexpr int SW = 16;                       // most warps (chains) per CTA; fewer when two rows per warp do not fit

struct SamplerParams {
    int8_t* sigma;
    int64_t nb;
    int N, n_words;
    const float* theta;
    int M_pad, M_eff;
    const float* Dtab;
    const int32_t* pairs;
    const float* a;
    int rule, n_idx, sw;                     // sw = warps per CTA of this launch
    int64_t n_steps;
    uint32_t key0, key1;
    uint64_t step_offset, chain0;
    int32_t* accepted;
};

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t& r0, uint32_t& r1) {
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        c0 = hi1 ^ c1 ^ k0; c1 = lo1;
        c2 = hi0 ^ c3 ^ k1; c3 = lo0;
        k0 += W0; k1 += W1;
    }
    r0 = c0; r1 = c1;
}

template <int V, bool CPLX>
constexpr int sampler_min_blocks() { return ((CPLX ? 8 : 4) * V <= 16) ? 2 : 1; }
// warps per CTA: two row buffers of V * 512 B (x2 complex) per warp must fit; 12 warps leave 168 registers per thread
// Rows are staged through shared memory (STAGED) only where that was measured to win: rows of 8 KB (config 5:
// 40.3 -> 35.6 ms per sweep, with 12 warps); for rows of <= 4 KB the direct L2 reads of 16 warps were faster
// (configs 3, 4: 1.51 vs 1.68 ms, 0.66 vs 0.71 ms).
// The wide variants (a lane's theta beyond 64 registers: M_pad > 2048 real, > 1024 complex) run 8 warps with 255 registers
// and read their rows straight from L2.
template <int V, bool CPLX>
__host__ __device__ constexpr int sampler_warps() {
    return lane_state_warps(V, CPLX) == 8 ? 8 : ((16 * 2 * V * 512 * (CPLX ? 2 : 1) <= 216 * 1024) ? 16 : 12);
}
template <int V, bool CPLX>
__host__ __device__ constexpr bool sampler_staged() { return sampler_warps<V, CPLX>() == 12; }

template <int V, bool CPLX>
__global__ void __launch_bounds__(sampler_warps<V, CPLX>() * 32, (sampler_min_blocks<V, CPLX>())) metropolis_kernel(const SamplerParams p) {
    extern __shared__ __align__(128) uint8_t smem_s[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t c_loc = (int64_t)blockIdx.x * p.sw + warp;
    if (c_loc >= p.nb) return;                         // no CTA-wide synchronisation below
    // shared memory: [sw warps][2 row buffers][M_eff floats] | [sw][n_words] spin bits | [sw][2] mbarriers
    const uint32_t row_bytes = (uint32_t)p.M_eff * 4u;
    const size_t rows_bytes = sampler_staged<V, CPLX>() ? (size_t)p.sw * 2 * row_bytes : 0;
    float* rowbuf = reinterpret_cast<float*>(smem_s) + (size_t)warp * 2 * p.M_eff;
    uint32_t* bits = reinterpret_cast<uint32_t*>(smem_s + rows_bytes) + (size_t)warp * p.n_words;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_s + rows_bytes + (size_t)p.sw * p.n_words * 4) +
                     warp * 2;                          // bit i of `bits` set <=> sigma_i = -1
    const uint32_t bar0 = smem_u32(bars), row0 = smem_u32(rowbuf);
    constexpr bool STAGED = sampler_staged<V, CPLX>();
    if (STAGED && lane == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar0 + 8, 1);
        mbar_fence_init();
    }
    uint32_t phase = 0u;                               // bit `slot` = parity the next wait on that slot expects
    auto issue_row = [&](int slot, int row) {          // all lanes are past their reads of this slot (warp converged)
        __syncwarp();
        if (lane == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_arrive_expect_tx(bar0 + 8 * slot, row_bytes);
            bulk_g2s(row0 + slot * row_bytes, p.Dtab + (size_t)row * p.M_eff, row_bytes, bar0 + 8 * slot);
        }
    };
    auto wait_row = [&](int slot) {
        mbar_wait(bar0 + 8 * slot, (phase >> slot) & 1u);
        phase ^= 1u << slot;
    };
    int8_t* sp = p.sigma + c_loc * p.N;
    for (int wi = lane; wi < p.n_words; wi += 32) {
        uint32_t w = 0;
        const int base = wi * 32;
        const int cnt = (p.N - base < 32) ? (p.N - base) : 32;
        for (int t = 0; t < cnt; ++t) w |= (uint32_t)(sp[base + t] < 0) << t;
        bits[wi] = w;
    }
    typename std::conditional<CPLX, CplxState<V>, RealState<V>>::type st;
    st.load(p.theta + c_loc * p.M_eff, lane, p.M_pad);
    __syncwarp();

    const uint64_t chain = p.chain0 + (uint64_t)c_loc;
    const uint32_t ch_lo = (uint32_t)chain, ch_hi = (uint32_t)(chain >> 32);
    int n_acc = 0;
    for (int64_t t0 = 0; t0 < p.n_steps; t0 += 32) {
        // ---- this lane's draw for transition t0 + lane ----
        const uint64_t step = p.step_offset + (uint64_t)(t0 + lane);
        uint32_t r0, r1;
        philox4x32_10(ch_lo, ch_hi, (uint32_t)step, (uint32_t)(step >> 32), p.key0, p.key1, r0, r1);
        const int idx_l = (int)__umulhi(r0, (uint32_t)p.n_idx);
        const float u_l = ((float)(r1 >> 9) + 0.5f) * 1.1920928955078125e-07f;   // 2^-23
        int i_l = idx_l, j_l = -1;
        if (p.rule == NK_RULE_EXCHANGE) { i_l = p.pairs[2 * idx_l]; j_l = p.pairs[2 * idx_l + 1]; }
        float a2_l = 0.f;                             // 2 log2(e) Re(a_i - a_j): visible-bias exponent
        if (p.a != nullptr) {
            const int stride = CPLX ? 2 : 1;
            a2_l = p.a[stride * i_l];
            if (j_l >= 0) a2_l -= p.a[stride * j_l];
            a2_l *= 2.f * LOG2E;
        }
        const int cnt = (p.n_steps - t0 < 32) ? (int)(p.n_steps - t0) : 32;
        // Transitions of the batch are visited through a ballot of the proposals that are non-trivial on the CURRENT
        // spins (lane l tests its own transition): runs of trivial exchanges (s' = s, ratio 1, accepted) are counted
        // and skipped in one step, and the same mask names the next row to prefetch.
        int pend_tt = -1, pend_slot = 0;              // a row copy in flight for transition pend_tt of this batch
        int pos = 0;
        while (true) {
            const uint32_t bi_l = (bits[i_l >> 5] >> (i_l & 31)) & 1u;
            const uint32_t bj_l = (j_l >= 0) ? ((bits[j_l >> 5] >> (j_l & 31)) & 1u) : (bi_l ^ 1u);
            const unsigned cand = __ballot_sync(0xffffffffu, lane >= pos && lane < cnt && bi_l != bj_l);
            if (cand == 0u) {
                n_acc += cnt - pos;
                if (STAGED && pend_tt >= 0) wait_row(pend_slot);          // misjudged: drop the row
                break;
            }
            const int tt = __ffs(cand) - 1;
            n_acc += tt - pos;                        // the trivial exchanges in between
            pos = tt + 1;
            const int idx = __shfl_sync(0xffffffffu, idx_l, tt);
            const int i = __shfl_sync(0xffffffffu, i_l, tt);
            const int j = __shfl_sync(0xffffffffu, j_l, tt);
            const float u = __shfl_sync(0xffffffffu, u_l, tt);
            const float a2 = __shfl_sync(0xffffffffu, a2_l, tt);
            const uint32_t bi = __shfl_sync(0xffffffffu, bi_l, tt);
            int slot = 0;
            if constexpr (STAGED) {
                if (pend_tt == tt) slot = pend_slot;  // the prefetched row is this transition's
                else {
                    if (pend_tt >= 0) wait_row(pend_slot);                // misjudged: drop the row
                    issue_row(0, idx);                // first of a batch, or misjudged: fetch now
                }
                pend_tt = -1;
                const unsigned next = cand & (cand - 1u);                 // next non-trivial proposal on the current spins
                if (next) {
                    pend_tt = __ffs(next) - 1;
                    pend_slot = slot ^ 1;
                    issue_row(pend_slot, __shfl_sync(0xffffffffu, idx_l, pend_tt));
                }
                wait_row(slot);
            }
            const float s = bi ? 1.f : -1.f;          // s = -sigma_i
            const float* drow = STAGED ? rowbuf + (size_t)slot * p.M_eff : p.Dtab + (size_t)idx * p.M_eff;
            bool accept;
            if constexpr (!CPLX) {
                float praw, acc;
                st.partial_raw(drow, lane, s, praw, acc);
                // this lane's share with its exponent folded in: one butterfly instead of two; every lane ends with
                // the same bits (each level multiplies the same two operands in both lanes of a pair)
                const float z = warp_prod_f((praw * st.qinv) * ex2_approx(0.5f * acc));
                const float ratio = z * ex2_approx(s * a2);
                accept = u < ratio * ratio;
                if (accept) st.commit(drow, lane, s, praw);
            } else {
                float pr, pi, acc;
                st.partial_raw(drow, lane, p.M_pad, s, pr, pi, acc);
                float cr = pr, ci = pi;
                cmul_f(cr, ci, st.qr, st.qi);
                const float m = ex2_approx(0.5f * acc);   // exponent folded into the lane's factor
                cr *= m; ci *= m;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const float orr = __shfl_xor_sync(0xffffffffu, cr, o), oi = __shfl_xor_sync(0xffffffffu, ci, o);
                    cmul_f(cr, ci, orr, oi);
                }
                const float mag2 = fmaf(cr, cr, ci * ci) * ex2_approx(2.f * s * a2);
                accept = __shfl_sync(0xffffffffu, (int)(u < mag2), 0) != 0;   // complex products differ in rounding per lane
                if (accept) st.commit(drow, lane, p.M_pad, s, pr, pi);
            }
            if (accept) {
                ++n_acc;
                __syncwarp();
                if (lane == 0) {
                    bits[i >> 5] ^= 1u << (i & 31);
                    if (j >= 0) bits[j >> 5] ^= 1u << (j & 31);
                }
                __syncwarp();
            }
        }
    }
    __syncwarp();
    for (int k = lane; k < p.N; k += 32) sp[k] = ((bits[k >> 5] >> (k & 31)) & 1u) ? (int8_t)-1 : (int8_t)1;
    if (lane == 0 && p.accepted != nullptr) p.accepted[c_loc] = n_acc;
}

using SamplerFn = void (*)(const SamplerParams);
template <int V>
static SamplerFn pick_sreal(int v) {
    if (v == V) return metropolis_kernel<V, false>;
    if constexpr (V < MAX_V_REAL) return pick_sreal<V + 1>(v);
    return nullptr;
}
template <int V>
static SamplerFn pick_scplx(int v) {
    if (v == V) return metropolis_kernel<V, true>;
    if constexpr (V < MAX_V_CPLX) return pick_scplx<V + 1>(v);
    return nullptr;
}

cudaError_t launch_metropolis(const Geometry& g, int dtype, int8_t* sigma, int64_t nb, const float* theta,
                              const float* Dtab, const SamplerArgs& sa, int32_t* accepted, cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    const bool cplx = dtype == NK_C64;
    const int V = g.M_pad / MPAD_ALIGN;
    SamplerFn fn = cplx ? pick_scplx<1>(V) : pick_sreal<1>(V);
    if (fn == nullptr) return cudaErrorInvalidValue;
    // as many warps per CTA (a multiple of 4, one chain each) as fit with two row buffers per warp
    int sw = lane_state_warps(V, cplx) == 8 ? 8 : ((16 * 2 * (size_t)g.M_eff * 4 <= (size_t)216 * 1024) ? 16 : 12);   // = sampler_warps<V, CPLX>()
    const bool staged = sw == 12;
    const size_t per_warp = (staged ? (size_t)2 * g.M_eff * 4 : 0) + (size_t)g.n_words * 4 + 16;
    while (sw > 4 && sw * per_warp + 128 > (size_t)220 * 1024) sw -= 4;
    const size_t smem = sw * per_warp + 128;
    if (smem > (size_t)227 * 1024) return cudaErrorInvalidValue;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    SamplerParams p;
    p.sigma = sigma; p.nb = nb; p.N = g.N; p.n_words = g.n_words;
    p.theta = theta; p.M_pad = g.M_pad; p.M_eff = g.M_eff; p.Dtab = Dtab;
    p.pairs = sa.pairs; p.a = (const float*)sa.a; p.rule = sa.rule; p.n_idx = sa.n_idx; p.sw = sw; p.n_steps = sa.n_steps;
    p.key0 = (uint32_t)sa.seed; p.key1 = (uint32_t)(sa.seed >> 32);
    p.step_offset = sa.step_offset; p.chain0 = sa.chain0; p.accepted = accepted;
    const int64_t grid = (nb + sw - 1) / sw;
    fn<<<(unsigned)grid, sw * 32, smem, st>>>(p);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
