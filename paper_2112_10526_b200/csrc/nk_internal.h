// Internal declarations shared by the translation units of libnkb200.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "nkb200.h"

namespace nk {

// automatic form of the amplitude ratios (nk_local_energy_ex without a NK_FORM_* flag, real parameters): the product
// form runs iff max |tanh delta| over the table is at most this — every factor 1 +- t tau then lies in [1/2, 3/2] and its
// relative rounding error is amplified by at most (1 + tau) / (1 - tau) <= 3
#define NK_FORM_TAU_MAX 0.5f


// tensor-core series form (series_tc.cu): highest power of the series, 16-bit segments per operand row, the bound on the
// truncation error of a log-ratio (natural-log units) the automatic choice accepts, and the smallest problem it is
// used for.  Like NK_FORM_TAU_MAX these depend on the parameters / operator only, never on sigma, B or chunk_size.
#define SERIES_K_MAX 6
#define SERIES_SEGS (SERIES_K_MAX + 1)
#define SERIES_TOL 1e-5f
#define SERIES_TAU_MAX 0.5f
#define SERIES_MIN_ROWS 128
#define SERIES_MIN_MPAD 256

// theta is kept in the fused kernel as theta_s = KAPPA * theta, so that exp(-2|theta|) = 2^(-|theta_s|)
// is a bare MUFU.EX2 (no multiply).  KAPPA = 2 log2(e).
constexpr float KAPPA = 2.8853900817779268f;
constexpr float LOG2E = 1.4426950408889634f;

constexpr int MPAD_ALIGN = 128;      // hidden units padded to a multiple of 128: one float4 per lane per 128
constexpr int MAX_V_REAL = 32;       // M_pad <= 4096 (real)
constexpr int MAX_V_CPLX = 16;       // M_pad <= 2048 (complex, two planes)
// warps (samples / chains in flight) per CTA of the warp-per-sample kernels: 16 while a lane's share of theta fits 64
// registers (128 registers x 512 threads = the register file); the wide variants (up to 128 registers of theta per lane)
// run 8 warps with 255 registers per thread
__host__ __device__ constexpr int lane_state_warps(int V, bool cplx) { return ((cplx ? 2 : 1) * V > 16) ? 8 : 16; }

// One row of the bond-difference table D: which sites it touches and the scalar data the fused kernel needs.
struct __align__(32) RowInfo {
    int32_t i;        // site whose spin gives the sign (s = -sigma_i)
    int32_t j;        // exchange partner, or -1 for a single flip / padded row
    float coef;       // matrix element of the connected configuration (+-2 J_c, or -h)
    float jdiag;      // Heisenberg: J_c of the bond (diagonal term J s_i s_j); Ising: 0
    float a2_re;      // log2(e) * 2 (a_i - a_j)   [or 2 a_i]: exponent contribution of the visible bias
    float a2_im;      // complex: 2 Im(a_i - a_j) in radians; real: 0
    float c2_re;      // product form: sum_j ln|cosh d_j| in log2 units (filled by rowc_kernel, else 0)
    float c2_im;      // product form, complex: sum_j arg cosh d_j in radians
};

struct Operator {
    int kind, n_sites, n_bonds, n_colors;
    unsigned flags;
    double h;
    int32_t* d_bonds;    // [n_bonds][2]
    int32_t* d_colors;   // [n_bonds]
    float* d_Jf;         // [n_colors]
    double* d_Jd;        // [n_colors]
};

// per-device one-time state (function attributes, SM counts) is kept in arrays indexed by the device ordinal
constexpr int NK_MAX_DEVICES = 64;
inline int current_device() {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= NK_MAX_DEVICES) d = 0;
    return d;
}

inline int round_up(int x, int m) { return (x + m - 1) / m * m; }
inline size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

// Geometry derived from (op, N, M, dtype).
struct Geometry {
    int N, n_words, M, M_pad, M_eff, planes; // M_eff = planes * M_pad; n_words = ceil(N / 32)
    int K_pad;                               // N rounded up to 128: k extent (bytes per row) of the int8 tensor-core operands
    int n_rows, tile_rows, n_tiles, n_rows_pad;
    int stages, ctas_per_sm;                 // shared-memory ring plan of the fused kernel
    size_t smem_bytes;
    bool ok;                                 // false: sizes beyond what this version supports
};
int fused_ctas_per_sm(int M_pad, bool cplx);
int fused_consumer_warps(int M_pad, bool cplx);
Geometry make_geometry(const Operator* op, int N, int M, int dtype);

// ---- launchers (each returns cudaGetLastError() of its launches) -----------------------------------------
// pack.cu
cudaError_t launch_pack(const Operator* op, const Geometry& g, int dtype, const void* W, const void* a, const void* b,
                        float* Wg, float* bg, float* Wt, float* Dtab, RowInfo* rows, cudaStream_t st);
cudaError_t launch_pack_gemm_only(const Geometry& g, int dtype, const void* W, const void* b, float* Wg, float* bg,
                                  cudaStream_t st);
cudaError_t launch_pack_product(const Operator* op, const Geometry& g, int dtype, const float* Wt, float* tab,
                                RowInfo* rows, cudaStream_t st, unsigned* taumax_bits = nullptr,
                                unsigned* series_ctl = nullptr);
cudaError_t launch_pack_table(const Geometry& g, int dtype, const void* W, const void* b, const int32_t* pairs_dev,
                              int n_rows, float* Wg, float* bg, float* Wt, float* Dtab, cudaStream_t st);
// sampler.cu : Metropolis-Hastings transitions with in-register incremental theta
struct SamplerArgs {
    int rule, n_idx;                 // NK_RULE_*; number of proposals (N sites or n_clusters pairs)
    const int32_t* pairs;            // dev [n_idx][2] (exchange) or nullptr (local)
    const void* a;                   // dev visible bias in the parameter dtype, or nullptr
    int64_t n_steps;
    uint64_t seed, step_offset, chain0;
};
cudaError_t launch_metropolis(const Geometry& g, int dtype, int8_t* sigma, int64_t nb, const float* theta,
                              const float* Dtab, const SamplerArgs& sa, int32_t* accepted, cudaStream_t st);
// theta_tc.cu : the same contraction on tcgen05 tensor cores (kind::i8, three int8 digit planes of W, three int32
// TMEM accumulators); Ws = the planes + scale, A = scratch for a padded int8 copy of the spins when N % 128 != 0
cudaError_t theta_tc_init();
cudaError_t launch_split_w(const float* Wg, int M_eff, int N, int K_pad, void* Ws, cudaStream_t st);
cudaError_t launch_theta_tc(const int8_t* sigma, int64_t B, int N, int M_eff, int K_pad, const void* Ws,
                            void* A, const float* bg, float* theta, cudaStream_t st);
cudaError_t launch_sigma_operand(const int8_t* sigma, int64_t B, int N, int K_pad, void* A_i8, cudaStream_t st);
cudaError_t launch_theta_tc_pre(const void* A_i8, int64_t B, int M_eff, int K_pad, const void* Ws,
                                const float* bg, float* theta, cudaStream_t st);   // launch_theta_tc without the spin conversion
cudaError_t launch_tc_gemm_pieces(const void* A_bf16, int64_t rows, const void* P_bf16, int cols, int ld, int k_len,
                                  float* out, int accumulate, cudaStream_t st);
// gradient.cu : force vector / energy gradient of the RBM
struct GradWs {
    float *Wg, *bg, *theta, *Gacc;
    uint16_t *Ws, *A, *TwT, *sigT;
    double *gb_acc, *ga_acc;
    double* part;               // [ceil(chunk / grad_slab())][M_eff] per-slab partial column sums (grad_b)
    double* part_a;             // [ceil(chunk / grad_slab())][2 N] the same for grad_a
    unsigned* absmax;
    int ld;                     // k extent (samples per chunk, rounded up to 64) of TwT / sigT
};
int grad_slab();
cudaError_t launch_gradient_chunk(const Geometry& g, int dtype, const int8_t* sigma, int64_t nb, int64_t B_total,
                                  const void* eloc, const double* stats, const GradWs& w, int first_chunk,
                                  float real_scale, cudaStream_t st, const float* theta_in = nullptr,
                                  const void* sigT_ready = nullptr, int phase = 0);
// real_scale: 2 (gradient 2 Re f~) | 1 (QGT).  theta_in: read theta from there (w.theta receives v) instead of in
// place; sigT_ready: the chunk's transposed bf16 spins prepared earlier by launch_sigma_T (w.sigT is not touched).
cudaError_t launch_sigma_T(const int8_t* sigma, int64_t nb, int N, int ld, void* sigT, cudaStream_t st);
cudaError_t launch_gradient_finalize(const Geometry& g, int dtype, const GradWs& w, void* grad_a, void* grad_b,
                                     void* grad_W, cudaStream_t st);
// qgt.cu : pieces of the QGT-vector product
cudaError_t launch_qgt_w(const Geometry& g, int dtype, const int8_t* sigma, int64_t nb, const float* theta,
                         const float* Y, const void* v_a, void* w_out, cudaStream_t st);
cudaError_t launch_qgt_shift(void* out, const void* v, double shift, int64_t n_floats, cudaStream_t st);
// cg.cu : conjugate-gradient pieces of the SR solve
int cg_partials();
cudaError_t launch_cg_dot(const float* x, const float* y, int64_t n, double* part, double* out, cudaStream_t st);
cudaError_t launch_cg_step(float* x, float* r, const float* p, const float* Ap, int64_t n, const double* rr,
                           const double* pAp, cudaStream_t st);
cudaError_t launch_cg_dir(float* p, const float* r, int64_t n, const double* rr_new, const double* rr_old,
                          cudaStream_t st);
// rbmsymm.cu : weight tying of the fully symmetric RBM
cudaError_t launch_rbmsymm_expand(int F, int G, int N, int dtype, const void* Wsym, const void* bsym,
                                  const int32_t* perms, void* W, void* b, cudaStream_t st);
cudaError_t launch_rbmsymm_reduce(int F, int G, int N, int dtype, const void* gW, const void* gb,
                                  const int32_t* perms, void* gWsym, void* gbsym, cudaStream_t st);
// logpsi.cu
cudaError_t launch_logpsi(const int8_t* sigma, int64_t B, const Geometry& g, int dtype, const float* theta,
                          const void* a, void* logpsi_out, bool out_f64, void* theta_out, cudaStream_t st,
                          const unsigned* series_ctl = nullptr, uint16_t* series_Ap = nullptr);
// connected.cu
cudaError_t launch_connected(const Operator* op, const int8_t* sigma, int64_t B, int32_t* flips, float* mels,
                             int32_t* n_conn, int8_t* sigma_prime, cudaStream_t st);
// series_tc.cu : amplitude ratios as a short series of tensor-core GEMMs (product form, logarithm expanded)
struct SeriesWs {
    unsigned* ctl;              // [16] control block written per call: ctl[0] = K (0 = path off), scales, row bounds
    uint16_t* Bp;               // [n_rows][SERIES_SEGS][M_pad] 16-bit operand rows of the table (per call)
    // per-group buffers (a group = `group` consecutive chunks contracted by one launch), two sets when there is more
    // than one group (api.cu pipelines them over two streams):
    uint16_t* Ap[2];            // [group_rows][SERIES_SEGS][M_pad] 16-bit operand rows of the samples
    uint32_t* sigT[2];          // [N][w32] transposed bit-packed spins of the group
    float* part;                // [n_nt][part_stride] partial local energies per column tile, whole batch
    int w32, n_nt, group, n_sets;
    int64_t group_rows;
    int64_t part_stride;
};
bool series_possible(const Geometry& g, int dtype);
SeriesWs carve_series(uint8_t* base, size_t* off, const Geometry& g, int64_t chunk, int64_t B);
cudaError_t launch_series_prep(const Geometry& g, const int8_t* sigma, int64_t nb, const SeriesWs& w, int set,
                               cudaStream_t st);
cudaError_t launch_series_ctl_reset(const SeriesWs& w, cudaStream_t st);
cudaError_t launch_series_pack(const Geometry& g, const float* Ttab, const unsigned* taumax_bits, const SeriesWs& w,
                               bool force, cudaStream_t st);
cudaError_t launch_series_gemm(const Geometry& g, int64_t s0, int64_t nb, const RowInfo* rows, const SeriesWs& w, int set,
                               cudaStream_t st);
cudaError_t launch_series_finish(const Operator* op, const Geometry& g, const int8_t* sigma, int64_t B, const SeriesWs& w,
                                 float* eloc_out, cudaStream_t st);
// fused_eloc.cu
cudaError_t launch_fused_eloc(const Operator* op, const Geometry& g, int dtype, const int8_t* sigma, int64_t B,
                              const float* theta, const float* Dtab, const RowInfo* rows, void* eloc_out,
                              bool product_form, cudaStream_t st, const unsigned* gate = nullptr, int gate_mode = 0,
                              const unsigned* series_ctl = nullptr);
cudaError_t fused_eloc_init();   // one-time cudaFuncSetAttribute calls
// stats.cu
cudaError_t launch_check_spins(const int8_t* sigma, int64_t n, int* flag, cudaStream_t st);
cudaError_t launch_stats(const void* eloc, int64_t B, int dtype, double* stats_out, cudaStream_t st);

void count_launch(int n = 1);

// optional per-phase event timing (nk_profile_enable / nk_profile_read): brackets a group of launches on `st`
enum Phase { PH_PACK = 0, PH_GEMM, PH_LOGPSI, PH_FUSED, PH_STATS, PH_SERIES_GEMM, PH_SERIES_PREP, PH_COUNT };
struct ProfScope {
    cudaStream_t st; int phase; cudaEvent_t a, b; bool on;
    ProfScope(int phase, cudaStream_t st);
    ~ProfScope();
};

}  // namespace nk
