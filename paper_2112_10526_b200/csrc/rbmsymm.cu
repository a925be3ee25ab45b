// Fully symmetric RBM (RBMSymm), second workload.
//   ln psi = sum_{i, g in G} ln cosh f_g^(i),   f_g^(i) = sum_r W^(i)_r s_{g r} + b^(i)      PAPER.md Eq. (41), Eq. (56)
// is an RBM with M = F |G| hidden units and tied weights:  hidden unit (i, g) = row i |G| + g has
//   W_full[(i,g)][g r] = W^(i)_r,   b_full[(i,g)] = b^(i),
// so every call of this library (ln psi, local energies, sampler, QGT) applies to the expanded parameters, and
// derivatives with respect to the tied parameters are orbit sums of the expanded ones (the map is linear):
//   g_W^(i)_r = sum_g g_Wfull[(i,g)][g r],   g_b^(i) = sum_g g_bfull[(i,g)].
#include "nk_internal.h"

namespace nk {

// one block per expanded row (i, g); E = floats per element (1 real, 2 complex)
template <int E>
__global__ void rbmsymm_expand_kernel(const float* __restrict__ Wsym, const float* __restrict__ bsym,
                                      const int32_t* __restrict__ perms, int G, int N, float* __restrict__ W,
                                      float* __restrict__ b) {
    const int row = blockIdx.x, i = row / G, g = row - i * G;
    for (int r = threadIdx.x; r < N; r += blockDim.x) {
        const int k = perms[(size_t)g * N + r];
        if (k < 0 || k >= N) continue;                 // malformed table: stay inside the buffers
#pragma unroll
        for (int e = 0; e < E; ++e) W[((size_t)row * N + k) * E + e] = Wsym[((size_t)i * N + r) * E + e];
    }
    if (threadIdx.x < E && b != nullptr) b[(size_t)row * E + threadIdx.x] = bsym ? bsym[(size_t)i * E + threadIdx.x] : 0.f;
}

// one block per feature i; thread r sums over the group in order (deterministic), fp64 accumulation
template <int E>
__global__ void rbmsymm_reduce_kernel(const float* __restrict__ gW, const float* __restrict__ gb,
                                      const int32_t* __restrict__ perms, int G, int N, float* __restrict__ gWsym,
                                      float* __restrict__ gbsym) {
    const int i = blockIdx.x;
    for (int r = threadIdx.x; r < N; r += blockDim.x) {
        double acc[E];
#pragma unroll
        for (int e = 0; e < E; ++e) acc[e] = 0.0;
        for (int g = 0; g < G; ++g) {
            const int k = perms[(size_t)g * N + r];
            if (k < 0 || k >= N) continue;             // malformed table: stay inside the buffers
#pragma unroll
            for (int e = 0; e < E; ++e) acc[e] += (double)gW[(((size_t)i * G + g) * N + k) * E + e];
        }
#pragma unroll
        for (int e = 0; e < E; ++e) gWsym[((size_t)i * N + r) * E + e] = (float)acc[e];
    }
    if (threadIdx.x < E && gb != nullptr && gbsym != nullptr) {
        double acc = 0.0;
        for (int g = 0; g < G; ++g) acc += (double)gb[((size_t)i * G + g) * E + threadIdx.x];
        gbsym[(size_t)i * E + threadIdx.x] = (float)acc;
    }
}

cudaError_t launch_rbmsymm_expand(int F, int G, int N, int dtype, const void* Wsym, const void* bsym,
                                  const int32_t* perms, void* W, void* b, cudaStream_t st) {
    const unsigned rows = (unsigned)F * (unsigned)G;
    if (dtype == NK_C64)
        rbmsymm_expand_kernel<2><<<rows, 128, 0, st>>>((const float*)Wsym, (const float*)bsym, perms, G, N, (float*)W,
                                                       (float*)b);
    else
        rbmsymm_expand_kernel<1><<<rows, 128, 0, st>>>((const float*)Wsym, (const float*)bsym, perms, G, N, (float*)W,
                                                       (float*)b);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_rbmsymm_reduce(int F, int G, int N, int dtype, const void* gW, const void* gb,
                                  const int32_t* perms, void* gWsym, void* gbsym, cudaStream_t st) {
    if (dtype == NK_C64)
        rbmsymm_reduce_kernel<2><<<F, 256, 0, st>>>((const float*)gW, (const float*)gb, perms, G, N, (float*)gWsym,
                                                    (float*)gbsym);
    else
        rbmsymm_reduce_kernel<1><<<F, 256, 0, st>>>((const float*)gW, (const float*)gb, perms, G, N, (float*)gWsym,
                                                    (float*)gbsym);
    count_launch();
    return cudaGetLastError();
}

}  // namespace nk
