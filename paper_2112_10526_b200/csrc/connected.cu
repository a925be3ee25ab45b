// nk_connected: get_conn(sigma) -> (eta, mels) on the device  (Eq. (3); the paper runs this on
// the CPU through NUMBA and names it as the GPU bottleneck, footnote 5 L225).  One warp per sample enumerates the
// device bond table; the list has fixed width C with the slot convention of include/nkb200.h (Q9).
// This is the inspection / parity call: the fused kernel (fused_eloc.cu) enumerates the same list in registers
// and never writes it out.
#include "nk_internal.h"

namespace nk {

__global__ void __launch_bounds__(256)
connected_kernel(const int8_t* __restrict__ sigma, int64_t B, int N, int kind, int n_bonds,
                 const int32_t* __restrict__ bonds, const int32_t* __restrict__ colors,
                 const double* __restrict__ Jd, double h, unsigned flags, int32_t* __restrict__ flips,
                 float* __restrict__ mels, int32_t* __restrict__ n_conn, int8_t* __restrict__ sprime) {
    extern __shared__ int8_t smem_sigma[];            // [warps][N_pad]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t s = (int64_t)blockIdx.x * (blockDim.x >> 5) + warp;
    if (s >= B) return;
    const int N_pad = (N + 15) & ~15;
    int8_t* sg = smem_sigma + warp * N_pad;
    for (int i = lane; i < N; i += 32) sg[i] = sigma[s * N + i];
    __syncwarp();
    const int C = (kind == NK_HEISENBERG ? n_bonds : N) + 1;
    const double off = (flags & NK_FLAG_MARSHALL) ? -2.0 : 2.0;

    // diagonal: sum_b J_c(b) s_i s_j in fp64 (both models), and the number of active slots
    double diag = 0.0;
    int count = 0;
    for (int b = lane; b < n_bonds; b += 32) {
        const int i = bonds[2 * b], j = bonds[2 * b + 1];
        const int si = sg[i], sj = sg[j];
        diag += Jd[colors[b]] * (double)(si * sj);
        if (kind == NK_HEISENBERG) {
            const bool act = si != sj;
            count += act;
            const int64_t slot = s * C + 1 + b;
            if (flips) { flips[2 * slot] = act ? i : -1; flips[2 * slot + 1] = act ? j : -1; }
            if (mels) mels[slot] = act ? (float)(off * Jd[colors[b]]) : 0.f;
        }
    }
    if (kind == NK_ISING) {
        for (int k = lane; k < N; k += 32) {
            const int64_t slot = s * C + 1 + k;
            if (flips) { flips[2 * slot] = k; flips[2 * slot + 1] = -1; }
            if (mels) mels[slot] = (float)(-h);
        }
        count = (lane == 0) ? N : 0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        diag += __shfl_xor_sync(0xffffffffu, diag, o);
        count += __shfl_xor_sync(0xffffffffu, count, o);
    }
    if (lane == 0) {
        if (flips) { flips[2 * s * C] = -1; flips[2 * s * C + 1] = -1; }
        if (mels) mels[s * C] = (float)diag;
        if (n_conn) n_conn[s] = count + 1;
    }
    if (sprime == nullptr) return;
    // materialised sigma' (only asked for on small batches): slot c is a copy of sigma with <= 2 entries changed
    int8_t* out = sprime + s * (int64_t)C * N;
    for (int c = 0; c < C; ++c) {
        int fi = -1, fj = -1;
        if (c > 0) {
            if (kind == NK_HEISENBERG) {
                const int i = bonds[2 * (c - 1)], j = bonds[2 * (c - 1) + 1];
                if (sg[i] != sg[j]) { fi = i; fj = j; }
            } else fi = c - 1;
        }
        for (int k = lane; k < N; k += 32) {
            int8_t v = sg[k];
            if (k == fi || k == fj) v = (int8_t)(-v);   // exchange of antiparallel spins = negate both
            out[(int64_t)c * N + k] = v;
        }
    }
}

cudaError_t launch_connected(const Operator* op, const int8_t* sigma, int64_t B, int32_t* flips, float* mels,
                             int32_t* n_conn, int8_t* sigma_prime, cudaStream_t st) {
    if (B <= 0) return cudaSuccess;
    const int N_pad = (op->n_sites + 15) & ~15;
    int wpb = 8;
    while (wpb > 1 && (size_t)wpb * N_pad > 48 * 1024) wpb >>= 1;
    if ((size_t)wpb * N_pad > 48 * 1024) return cudaErrorInvalidConfiguration;
    const unsigned grid = (unsigned)((B + wpb - 1) / wpb);
    connected_kernel<<<grid, wpb * 32, (size_t)wpb * N_pad, st>>>(sigma, B, op->n_sites, op->kind, op->n_bonds,
                                                                 op->d_bonds, op->d_colors, op->d_Jd, op->h,
                                                                 op->flags, flips, mels, n_conn, sigma_prime);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
