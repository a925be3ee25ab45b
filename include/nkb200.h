/* nkb200.h — C ABI of libnkb200.so: batched RBM local energies for lattice spin Hamiltonians on one B200.
 *
 * The calls follow the paper's statement of the problem (citations: PAPER.md lines of arxiv 2112.10526):
 *   get_conn(sigma) -> (eta, mels)                         Eq. (3)  L215-219      -> nk_connected
 *   apply(params, sigma_batch) -> ln psi, batched           Eq. (6)  L273, L410    -> nk_rbm_logpsi
 *   local estimator A~(s) = sum_s' psi(s')/psi(s) <s|A|s'>  Eq. (12) L652          -> nk_local_energy
 *   sample mean over the batch                              Eq. (17) L675          -> nk_local_energy (stats_out)
 *   chunk_size bounds the configurations evaluated at once  Sec. 3.3.1 L689-695    -> nk_local_energy (chunk_size)
 * Ansatz (RBM, L575; ln cosh form Eq. (41); shapes W in C^{MxN}, b in C^M from Eq. (7)):
 *   ln psi(s) = sum_i a_i s_i + sum_j ln cosh(theta_j),  theta = W s + b.
 * Operators (hard-coded matrix elements, the style of L201-203):
 *   NK_HEISENBERG  H = sum_b J_c(b) sigma_i . sigma_j (Pauli matrices, Eq. (50)): diagonal J s_i s_j,
 *                  antiparallel bond -> exchanged configuration with element 2 J  (-2 J with NK_FLAG_MARSHALL)
 *   NK_ISING       H = J sum_b sz_i sz_j - h sum_i sx_i (Eq. (54)): diagonal J s_i s_j, every single-spin
 *                  flip with element -h
 *
 * Conventions
 *   - "dev" pointers are CUDA device pointers, "host" pointers are ordinary host memory.  All buffers belong to
 *     the caller.  The library allocates device memory only inside nk_operator_create and frees it only in
 *     nk_operator_destroy (nk_local_energy_plan_create additionally owns a CUDA graph).
 *   - Every call that takes a stream is asynchronous on that stream (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) and never synchronises the device, except nk_local_energy_host (see there).
 *   - Spins are int8 with values +1 / -1, row-major [B][N].  W is row-major [M][N] (theta = W s + b); a is [N],
 *     b is [M].  dtype NK_F32: float; NK_C64: interleaved (re, im) float pairs.  a and b may be NULL (= zeros).
 *   - Return value: NK_OK (0) or a negative nk_status.  Argument errors are detected on the host before any
 *     launch.  No exceptions, no exit(), no CPU fallback: without a CUDA device every compute call returns
 *     NK_ERR_CUDA.
 *   - Limits of this version: M <= 4096 (NK_F32) or M <= 2048 (NK_C64); N <= 65535; larger -> NK_ERR_UNSUPPORTED.
 */
#ifndef NKB200_H
#define NKB200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nk_operator_s* nk_operator_t;   /* opaque; device-resident bond table + couplings */
typedef void* nk_stream_t;                      /* a cudaStream_t */
typedef struct nk_plan_s* nk_plan_t;            /* opaque; one nk_local_energy_ex call captured into a CUDA graph */

enum nk_status {
    NK_OK = 0,
    NK_ERR_INVALID_ARG = -1,   /* NULL / out-of-range / inconsistent argument */
    NK_ERR_BAD_SPIN = -2,      /* a sigma value is not +1 / -1; only reported under NK_CHECK_SPINS (nk_local_energy_ex) */
    NK_ERR_WORKSPACE = -3,     /* workspace NULL, misaligned (256 B) or smaller than the *_workspace_bytes query */
    NK_ERR_UNSUPPORTED = -4,   /* sizes beyond the limits above */
    NK_ERR_CUDA = -5           /* a CUDA runtime call failed; see nk_last_cuda_error() */
};
enum nk_kind { NK_HEISENBERG = 0, NK_ISING = 1 };
enum nk_dtype { NK_F32 = 0, NK_C64 = 1 };
enum nk_rule { NK_RULE_LOCAL = 0, NK_RULE_EXCHANGE = 1 };
enum nk_flags {
    NK_FLAG_MARSHALL = 1u,     /* nk_operator_create: off-diagonal Heisenberg element -2J on EVERY bond (default +2J, Eq. (50)).
                                  This is the sublattice rotation U H U, U = prod_{i in A} sz_i, only if every bond joins
                                  the two sublattices; with same-sublattice bonds in the list (e.g. next-nearest neighbours)
                                  it defines a different Hamiltonian — give such bonds a colour with the sign folded into J */
    NK_OUT_F64 = 2u,           /* nk_rbm_logpsi: logpsi_out is double / (re,im) double instead of float */
    NK_FORM_PRODUCT = 4u,      /* nk_local_energy_ex: product-form amplitude ratios (see there) */
    NK_CHECK_SPINS = 8u,       /* nk_local_energy_ex: validate sigma in {+1,-1} first (one extra pass over sigma and one
                                  stream synchronisation); NK_ERR_BAD_SPIN before any other launch if it is not */
    NK_FORM_LOGCOSH = 16u,     /* nk_local_energy_ex: log-cosh amplitude ratios (see there) */
    NK_FORM_SERIES = 32u,      /* nk_local_energy_ex: product form with the logarithm expanded into a short series of
                                  tensor-core GEMMs (see there); real parameters only */
    NK_SERIAL_CHUNKS = 64u     /* nk_local_energy_ex: keep every kernel of the chunk loop on `stream` (no internal second
                                  stream); same results, used to time kernels in isolation */
};

/* Static, never-NULL description of a status code. */
const char* nk_status_string(int status);
/* The cudaError_t (as int) of the most recent NK_ERR_CUDA on this thread, 0 if none. */
int nk_last_cuda_error(void);
/* Library version, e.g. 100 = 0.1.0. */
int nk_version(void);

/* ---- operator ------------------------------------------------------------------------------------------
 * Copies the bond table to the device.  bonds_host [n_bonds][2] with 0 <= i,j < n_sites and i != j (each
 * undirected pair listed once; the ORDER of the table fixes the order of the connected list).  colors_host
 * [n_bonds] in [0, n_colors) or NULL (all 0).  J_host [n_colors].  h is used by NK_ISING only.
 * Synchronous (cudaMalloc + cudaMemcpy).  Errors: NK_ERR_INVALID_ARG on a bad table, NK_ERR_CUDA. */
int nk_operator_create(nk_operator_t* out, int kind, int n_sites, int n_bonds, const int32_t* bonds_host,
                       const int32_t* colors_host, int n_colors, const double* J_host, double h, unsigned flags);
int nk_operator_destroy(nk_operator_t op);
/* Width C of the connected list: n_bonds + 1 (Heisenberg) or n_sites + 1 (Ising). */
int nk_operator_max_conn(nk_operator_t op, int* C_out);

/* ---- ln psi ---------------------------------------------------------------------------------------------
 * logpsi_out dev [B]: float | (re,im) float, or double | (re,im) double with NK_OUT_F64.  The imaginary part
 * is returned modulo 2 pi (a sum of principal logs).  theta_out: NULL, or dev [B][M] (float | (re,im) float)
 * receiving theta = W s + b.  theta is contracted on the tensor cores from an exact fixed-point split of W (|W - W_fixed|
 * <= 2^-23 max|W|) with exact +-1 products and exact integer accumulation; the ln cosh
 * terms and their sum are evaluated in fp64 (Q12).  workspace: dev, 256-B aligned, at least
 * nk_rbm_logpsi_workspace_bytes(B, N, M, dtype) bytes. */
size_t nk_rbm_logpsi_workspace_bytes(int64_t B, int N, int M, int dtype);
int nk_rbm_logpsi(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* a,
                  const void* b, void* logpsi_out, void* theta_out, unsigned flags, void* workspace,
                  size_t workspace_bytes, nk_stream_t stream);

/* nk_rbm_logpsi for callers that cannot allocate device memory (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same inputs, outputs, arithmetic and errors, no workspace argument.  The scratch
 * is a static device array of NK_STATIC_SCRATCH_BYTES (16 MiB) inside the library, which EVERY GPU that loads the
 * library holds until the process exits; the call itself makes no cudaMalloc / cudaFree and calls no allocating
 * library routine.  Limit: nk_rbm_logpsi_workspace_bytes(B, N, M, dtype) <= NK_STATIC_SCRATCH_BYTES (also returned by
 * nk_rbm_logpsi_static_max_bytes), e.g. B = 4096 samples of config 2 (N = M = 100: 3.2 MiB) or B = 1024 at N = 400,
 * M = 800 (7 MiB); a larger problem is rejected with NK_ERR_WORKSPACE before anything is launched — use
 * nk_rbm_logpsi with your own workspace there.  All calls on a device share the one array, which keeps the last
 * call's contents (every buffer in it is rewritten in full by the call before it is read, so nothing needs clearing):
 * calls that may OVERLAP on the GPU — different streams, or graphs replayed concurrently — race on it; order them on
 * one stream or with events.  The array's address is resolved per device on the first call there
 * (cudaGetSymbolAddress), with that device current.  Asynchronous on `stream` like nk_rbm_logpsi. */
#define NK_STATIC_SCRATCH_BYTES (16u << 20)
size_t nk_rbm_logpsi_static_max_bytes(void);
int nk_rbm_logpsi_static(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* a,
                         const void* b, void* logpsi_out, void* theta_out, unsigned flags, nk_stream_t stream);

/* ---- connected configurations (inspection / parity call; the fused path never materialises sigma') --------
 * Fixed-width list per sample, C = nk_operator_max_conn:
 *   slot 0      diagonal: flips (-1,-1), mel = H_ss (always present)
 *   Heisenberg  slot 1+b <-> bond b = (i,j): antiparallel -> flips (i,j), mel = +-2 J_c(b), sigma' = sigma with
 *               s_i, s_j exchanged; parallel -> PADDED: flips (-1,-1), mel 0, sigma' = sigma
 *   Ising       slot 1+k <-> site k: flips (k,-1), mel = -h, sigma' = sigma with s_k negated
 * flips_out dev int32 [B][C][2]; mels_out dev float [B][C]; n_conn_out dev int32 [B] = number of non-padded
 * slots; sigma_prime_out NULL or dev int8 [B][C][N].  Any of the three outputs flips/mels/n_conn may be NULL. */
int nk_connected(nk_operator_t op, const int8_t* sigma, int64_t B, int32_t* flips_out, float* mels_out,
                 int32_t* n_conn_out, int8_t* sigma_prime_out, nk_stream_t stream);

/* ---- local energy ---------------------------------------------------------------------------------------
 * E_loc(s) = H_ss + sum_{s' != s} H_ss' psi(s')/psi(s) for every row of sigma, evaluated chunk_size samples at a
 * time (0 = whole batch) inside a workspace whose size is set by min(B, chunk_size), not by B: where the tensor-core
 * series form can run (see nk_local_energy_ex) the library works on groups of up to 8 consecutive chunks — as many as
 * make its launches whole waves, at most 1 GiB of operand rows per buffer — so the bound is a small multiple of
 * chunk_size there, plus 64 bytes per sample (at 2048 table rows) for partial sums, and theta = W sigma + b is kept for a window of
 * groups (up to 1 GiB of fp32 activations: 4 M_pad bytes per sample until that cap) so that one launch contracts the
 * whole window.  Always size the workspace with the query.  Per-sample results do not depend on chunk_size.
 *   eloc_out    dev [B] float | (re,im) float
 *   logpsi_out  NULL or dev [B] float | (re,im) float  (ln psi(s), as nk_rbm_logpsi)
 *   stats_out   NULL or dev double[4]: mean_re, mean_im, population variance mean|E - mean|^2, count
 * W/a/b packing (transposes, bond-difference table) is redone on every call — the parameters change every VMC
 * step — and is part of the call's time. */
size_t nk_local_energy_workspace_bytes(nk_operator_t op, int64_t B, int N, int M, int dtype, int64_t chunk_size);
int nk_local_energy(nk_operator_t op, const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W,
                    const void* a, const void* b, int64_t chunk_size, void* eloc_out, void* logpsi_out,
                    double* stats_out, void* workspace, size_t workspace_bytes, nk_stream_t stream);

/* nk_local_energy with flags.  Two evaluations of the same Eq. (12) ratios:
 *  - NK_FORM_LOGCOSH: every ratio as exp(ln psi' - ln psi) from stable ln cosh terms (BASELINE.json north_star (3));
 *    one exponential per (amplitude, hidden unit) pair.
 *  - NK_FORM_PRODUCT: each ratio written as a product,
 *      cosh(theta_j + s d_j) / cosh(theta_j) = cosh(d_j) (1 + s tanh(theta_j) tanh(d_j)),   s = +-1,
 *      psi'/psi = e^{s da} prod_j cosh(d_j) prod_j (1 + s tanh(theta_j) tanh(d_j)),
 *    d the change of theta under the flip / exchange; tanh(d) and prod_j cosh(d_j) depend on the parameters only and
 *    are tabulated per call, tanh(theta) once per sample, so a pair costs two FP32 operations and no transcendental.
 *    Same outputs and tolerances for |d| up to ~2 (parameters of the five configs x5); beyond, the factors
 *    1 - |tanh(theta) tanh(d)| cancel and the fp32 rounding of the two tanh shows (~5e-4 at x10).  For complex
 *    parameters tanh(theta) is unbounded next to the zeros of cosh (Q18).
 *  - NK_FORM_SERIES: the product form with its logarithm expanded,
 *      ln prod_j (1 + s t_j tau_j) = sum_k ((-1)^(k+1) / k) s^k sum_j t_j^k tau_j^k,   t = tanh(theta), tau = tanh(d),
 *    so that the log-ratios of a chunk against all table rows are a short series of GEMMs over the hidden units, run
 *    on the tensor cores (tcgen05, fp16 hi/lo split of the k = 1 term, fp32 accumulation) with the exponential, the
 *    matrix element, the spin masks and the sum over connected configurations fused into the epilogue.  The series is
 *    cut after K <= 6 terms, K chosen on the device so that the remainder bound
 *    max_rows sum_j |tau_j|^(K+1) / ((K+1)(1 - tau_max)) <= 1e-5 (a property of the parameters).  Real parameters,
 *    M_pad >= 256 and >= 128 table rows only (else NK_ERR_UNSUPPORTED when forced); forced, it uses K = 6 when the
 *    bound cannot be met.
 *  - no form flag (flags = 0, and nk_local_energy): automatic.  Real parameters: the tables are packed, the device
 *    finds tau_max = max |tanh(d)| over the table; the series form runs if the sizes allow it, tau_max <= 0.5 and its
 *    bound can be met; else the product form iff tau_max <= 0.5 (every factor then lies in [1/2, 3/2]; its rounding
 *    error is amplified at most (1 + tau_max) / (1 - tau_max) <= 3 times); else the log-cosh form.  No host
 *    synchronisation (every kernel is launched, those on the wrong side of the gates return at once).  Complex
 *    parameters: always the log-cosh form.  The choice depends on the parameters only, never on sigma, B or chunk_size.
 *  The NK_FORM_* flags are mutually exclusive (NK_ERR_INVALID_ARG).
 * Streams: when the series form may run and the batch has more than one chunk, the preparation of chunk c + 1 (theta
 * contraction, the ln psi / operand pass, spin bits) is issued on one internal high-priority stream per calling thread
 * (created on first use, with five events) beside the tensor-core kernel of chunk c on `stream`; the internal stream
 * forks from and joins `stream` through events, so everything the caller observes is ordered on `stream` and the call
 * stays capturable in a CUDA graph.  The per-chunk buffers then exist twice in the workspace.  NK_SERIAL_CHUNKS keeps
 * everything on `stream`.
 * NK_CHECK_SPINS: validate sigma first (see enum nk_flags); may be combined with a form flag. */
int nk_local_energy_ex(nk_operator_t op, const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W,
                       const void* a, const void* b, int64_t chunk_size, unsigned flags, void* eloc_out,
                       void* logpsi_out, double* stats_out, void* workspace, size_t workspace_bytes,
                       nk_stream_t stream);

/* The same call as a PLAN: nk_local_energy_plan_create runs nk_local_energy_ex once (so every error it can report is
 * reported here; synchronises an internal stream), then captures its launches — both streams of the pipelined chunk loop
 * included — into a CUDA graph; nk_local_energy_plan_run replays that graph on `stream`: one launch per step instead of
 * ~85 (config 5) or ~15 (configs 1-2, which are launch-bound), the same kernels on the same buffers, the form of the
 * ratios still chosen on the device from the CURRENT parameters.  The plan is bound to the addresses and sizes given
 * at creation; the CONTENTS of sigma / W / a / b may change between runs, and the outputs are rewritten by every run.
 * The buffers must outlive the plan.  NK_CHECK_SPINS cannot be planned (NK_ERR_INVALID_ARG).  Besides
 * nk_operator_create this is the only call that allocates (a graph, its executable instance, one stream), released by
 * nk_local_energy_plan_destroy.  nk_launch_count advances by the number of kernels in the graph on every run. */
int nk_local_energy_plan_create(nk_plan_t* out, nk_operator_t op, const int8_t* sigma, int64_t B, int N, int M, int dtype,
                                const void* W, const void* a, const void* b, int64_t chunk_size, unsigned flags,
                                void* eloc_out, void* logpsi_out, double* stats_out, void* workspace,
                                size_t workspace_bytes);
int nk_local_energy_plan_run(nk_plan_t plan, nk_stream_t stream);
int nk_local_energy_plan_destroy(nk_plan_t plan);

/* Which form the most recent automatic nk_local_energy / nk_local_energy_ex call on `workspace` took (same op, B, N,
 * M, dtype, chunk_size as that call): *form_host = NK_FORM_SERIES, NK_FORM_PRODUCT or NK_FORM_LOGCOSH, *tau_max_host
 * (may be NULL) = max |tanh(d)| of the table, *series_terms_host (may be NULL) = the K of the series form (0 if it did
 * not run).  Reads two words of the workspace and SYNCHRONISES `stream`.  Undefined after a call with a forced
 * product or log-cosh form (the words are only written by automatic and forced-series calls). */
int nk_local_energy_form(nk_operator_t op, int64_t B, int N, int M, int dtype, int64_t chunk_size, const void* workspace,
                         size_t workspace_bytes, nk_stream_t stream, int* form_host, float* tau_max_host,
                         int* series_terms_host);

/* Same computation with HOST inputs and outputs (the end-to-end call): copies sigma/W/a/b host->device into
 * `scratch`, runs nk_local_energy, copies eloc / logpsi / stats back and SYNCHRONISES `stream` before returning.
 * Host buffers should be pinned for the copies to be asynchronous.  scratch: dev, 256-B aligned, at least
 * nk_local_energy_host_scratch_bytes(...) bytes (inputs + outputs + workspace).  eloc_host [B], logpsi_host [B]
 * or NULL, stats_host double[4] or NULL.  The host->device copies run on one internal non-blocking stream per calling
 * thread (created on first use, with a few events) so that sigma of chunk k + 1 is copied while chunk k is computed;
 * everything the caller observes is still ordered on `stream`. */
size_t nk_local_energy_host_scratch_bytes(nk_operator_t op, int64_t B, int N, int M, int dtype, int64_t chunk_size);
int nk_local_energy_host(nk_operator_t op, const int8_t* sigma_host, int64_t B, int N, int M, int dtype,
                         const void* W_host, const void* a_host, const void* b_host, int64_t chunk_size,
                         void* eloc_host, void* logpsi_host, double* stats_host, void* scratch,
                         size_t scratch_bytes, nk_stream_t stream);

/* ---- energy gradient / force vector of the RBM -------------------------------------
 * PAPER.md Eq. (13) L656 (log-derivatives O_i), Eq. (14) L660 / (26) L910 (force f~_i = E[O_i^* (H~ - E[H~])]),
 * Eq. (15)/(16) L664-668 and (27)/(28) L918-922: the gradient of <H> is 2 Re f~ for real parameters (NK_F32) and
 * f~ for the complex, holomorphic RBM (NK_C64).  O_a = s, O_b = tanh(theta), O_W = tanh(theta) s^T; E[.] is the
 * mean over the B samples.
 *   eloc   dev [B] float | (re,im) float, and stats dev double[4] (mean in [0],[1]) — as written by nk_local_energy
 *   grad_a_out dev [N] or NULL, grad_b_out dev [M] or NULL, grad_W_out dev [M][N]; parameter dtype
 * Samples are processed chunk_size at a time (0 = whole batch); the workspace scales with min(B, chunk_size).
 * The contraction over samples runs on the tensor cores with exact products; results are bit-reproducible. */
size_t nk_energy_gradient_workspace_bytes(int64_t B, int N, int M, int dtype, int64_t chunk_size);
int nk_energy_gradient(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* b,
                       const void* eloc, const double* stats, int64_t chunk_size, void* grad_a_out,
                       void* grad_b_out, void* grad_W_out, void* workspace, size_t workspace_bytes,
                       nk_stream_t stream);

/* The same for ONE SHARD of a batch that is spread over several ranks (samples are
 * distributed, expectation values reduced): sigma / eloc hold this rank's B samples, `stats` the statistics of the
 * WHOLE batch (nk_stats_combine of the all-gathered per-rank statistics) and B_global >= B its size.  The outputs are
 * this rank's share  (1 / B_global) sum_{s in shard} O_s^* (E_s - mean)  (x 2 Re for NK_F32), so the gradient of the
 * union is the plain SUM of the ranks' outputs: one all-reduce per block, no arithmetic outside the library. */
int nk_energy_gradient_sharded(const int8_t* sigma, int64_t B, int64_t B_global, int N, int M, int dtype,
                               const void* W, const void* b, const void* eloc, const double* stats,
                               int64_t chunk_size, void* grad_a_out, void* grad_b_out, void* grad_W_out,
                               void* workspace, size_t workspace_bytes, nk_stream_t stream);

/* Statistics of the union of n_parts shards from their (mean_re, mean_im, population variance, count) quadruples
 * (Eq. (17) L675 across shards; the pairwise update of Chan et al., applied in the order given).  Host arithmetic on
 * host pointers: parts_host [n_parts][4], out4_host [4].  Shards with count 0 are skipped. */
int nk_stats_combine(const double* parts_host, int n_parts, double* out4_host);

/* ---- quantum geometric tensor times a vector, on the fly -----------------------------
 * PAPER.md Eq. (23): G_ij = E[O_i^* O_j] - E[O_i^*] E[O_j] with the log-derivatives O of Eq. (13); its
 * product with a vector without forming G, Eq. (75) L2219 (QGTOnTheFly):
 *     w = (1/N_s) J v;   dw = w - <w>;   v~ = J^dagger dw;          out = v~ + diag_shift * v   (Eq. (25))
 * E[.] is the mean over the B rows of sigma.  Parameter vectors are given block-wise in the parameter dtype:
 * (v_a [N], v_b [M], v_W [M][N]) -> (out_a, out_b, out_W).  v_a / v_b may be NULL (= zeros), out_a / out_b may be
 * NULL (not wanted).  NK_F32: G is real (the Re[G] of Eq. (30)); NK_C64: the full Hermitian G of the holomorphic
 * RBM (Eq. (31)).  Samples are processed chunk_size at a time; the three contractions (theta, V_W sigma, J^dagger dw)
 * run on the tensor cores with exact products, as in nk_rbm_logpsi / nk_energy_gradient.
 * Single rank only: <w> is the mean over THIS call's samples, so the outputs of several shards do not add up to the
 * product of the union's G (the between-shard term of the covariance is missing); multi-rank stochastic
 * reconfiguration is not supported by this version. */
size_t nk_qgt_matvec_workspace_bytes(int64_t B, int N, int M, int dtype, int64_t chunk_size);
int nk_qgt_matvec(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* b,
                  const void* v_a, const void* v_b, const void* v_W, double diag_shift, int64_t chunk_size,
                  void* out_a, void* out_b, void* out_W, void* workspace, size_t workspace_bytes,
                  nk_stream_t stream);

/* Stochastic reconfiguration: solves  sum_j (G_ij + diag_shift delta_ij) delta_j = f_i  (Eq. (25) L886 with
 * Eq. (30) L961 for real parameters — G = Re[G], f = 2 Re f~ — and Eq. (31) for the holomorphic complex RBM) by
 * conjugate gradients (the paper's default solver, L969) started from zero; every iteration is one nk_qgt_matvec.
 * f and delta are block-wise in the parameter dtype, all six pointers required (device).  Stops when
 * |r| <= tol |f| or after max_iter iterations.  SYNCHRONISES `stream` (the residual is read back every few
 * iterations).  info_host (host double[2], or NULL): iterations performed, final |r| / |f| of the CG recurrence. */
size_t nk_sr_solve_workspace_bytes(int64_t B, int N, int M, int dtype, int64_t chunk_size);
int nk_sr_solve(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* b,
                const void* f_a, const void* f_b, const void* f_W, double diag_shift, double tol, int max_iter,
                int64_t chunk_size, void* delta_a, void* delta_b, void* delta_W, double* info_host, void* workspace,
                size_t workspace_bytes, nk_stream_t stream);

/* ---- fully symmetric RBM (RBMSymm, second workload) ----------------------------------
 * PAPER.md Eq. (41): ln psi = sum_{i, g in G} ln cosh f_g^(i), with the embedding of Eq. (56),
 * f_g^(i) = sum_r W^(i)_r s_{g r} + b^(i).  This is an RBM with M = n_features * n_group tied hidden units; hidden
 * unit (i, g) is row i * n_group + g:   W[(i,g)][g r] = W_sym[i][r],  b[(i,g)] = b_sym[i].
 *   perms  dev int32 [n_group][N], perms[g][r] = the site g r; every row must be a permutation of 0..N-1 (caller's
 *          responsibility; the table lives on the device, so the calls cannot check it without synchronising:
 *          out-of-range entries are skipped, a repeated image leaves a column of the expansion unwritten)
 * nk_rbmsymm_expand writes the expanded (W [M][N], b [M] or NULL) to pass to any other call of this library (no
 * visible bias: a = NULL); nk_rbmsymm_reduce_gradient maps a gradient / force / QGT-vector block of the expanded
 * parameters to the tied ones by summing over orbits (the tying is linear):
 *   grad_W_sym[i][r] = sum_g grad_W[(i,g)][g r],   grad_b_sym[i] = sum_g grad_b[(i,g)]   (fp64 sums, fixed order). */
int nk_rbmsymm_expand(int n_features, int n_group, int N, int dtype, const void* W_sym, const void* b_sym,
                      const int32_t* perms, void* W_out, void* b_out, nk_stream_t stream);
int nk_rbmsymm_reduce_gradient(int n_features, int n_group, int N, int dtype, const void* grad_W, const void* grad_b,
                               const int32_t* perms, void* grad_W_sym, void* grad_b_sym, nk_stream_t stream);

/* ---- Metropolis-Hastings sampler for the RBM ------------------------------------------
 * PAPER.md Sec. 3.4: a proposal s -> s' is accepted with probability min(1, |psi(s')|^2 / |psi(s)|^2) (Eq. (20)
 * L709; both rules are symmetric kernels, L711).  Every row of sigma is one chain (n_chains = n_samples, L1583);
 * the call advances each chain by n_steps transitions IN PLACE (one sweep = N transitions, footnote 20 L1590).
 *   NK_RULE_LOCAL     negate one uniformly drawn spin (MetropolisLocal, L713); clusters_host = NULL, n_clusters = 0
 *   NK_RULE_EXCHANGE  swap the spins of one uniformly drawn pair of clusters_host [n_clusters][2] (HOST pointer,
 *                     0 <= i != j < N; e.g. the lattice bonds: MetropolisExchange with graph=lattice, L1600); a
 *                     pair of equal spins proposes s' = s, which is accepted and counted
 * Random numbers are a pure function of (seed, chain index, transition index): Philox4x32-10 with counter
 * (chain lo, hi, transition lo, hi) and key (seed lo, hi) gives (r0, r1, ..); proposal = (r0 * n) >> 32,
 * u = ((r1 >> 9) + 1/2) 2^-23, accept iff u < |psi'/psi|^2 evaluated in fp32.  Row r of sigma is chain
 * chain_offset + r; its t-th transition of this call has index step_offset + t, so consecutive calls continue a
 * stream and a sharded batch reproduces the unsharded one.  Results do not depend on chunk_size (chains are
 * processed chunk_size at a time, 0 = all at once; the workspace scales with min(B, chunk_size)).
 *   sigma         dev [B][N] int8, in/out        accepted_out  NULL or dev int32 [B]: accepted transitions of this call
 * theta is contracted once per call from sigma and then updated incrementally in registers (fp32). */
size_t nk_metropolis_workspace_bytes(int rule, int n_clusters, int64_t B, int N, int M, int dtype, int64_t chunk_size);
int nk_metropolis_sample(int rule, const int32_t* clusters_host, int n_clusters, int8_t* sigma, int64_t B, int N,
                         int M, int dtype, const void* W, const void* a, const void* b, int64_t n_steps,
                         uint64_t seed, uint64_t step_offset, uint64_t chain_offset, int64_t chunk_size,
                         int32_t* accepted_out, void* workspace, size_t workspace_bytes, nk_stream_t stream);

/* Per-phase device timing (bench accounting).  With nk_profile_enable(1), nk_local_energy brackets each phase
 * of each chunk with CUDA events on the call's stream (a few microseconds of timeline each).  nk_profile_read
 * synchronises on those events, adds up the elapsed milliseconds per phase since the last read and writes
 * out[0..6] = ms in {pack, theta contraction, ln psi, local-energy phase (every kernel of it), statistics, the series
 * form's tensor-core kernel alone, the series form's operand preparation alone}, out[7..13] = the number of bracketed
 * launch groups per phase; then clears the record.  Thread-local, like nk_launch_count. */
int nk_profile_enable(int on);
int nk_profile_read(double* out14_host);

/* Pipe-peak microbenchmarks for the roofline denominators (bench accounting; nothing of the hot path runs here): three
 * kernels that saturate one pipe each — MUFU.EX2 (the log-cosh form's bound), FFMA (the product form's arithmetic),
 * LDS.128 (the product form's shared-memory bound) — timed with CUDA events, the SM clock measured inside each launch.
 * out8_host: [0] MUFU lanes / clk / SM, [1] FFMA lanes / clk / SM, [2] LDS bytes / clk / SM, [3..5] the SM clock (GHz)
 * in each of the three, [6] SM count, [7] total milliseconds.  scratch_dev: >= 256 device bytes.  SYNCHRONISES `stream`. */
int nk_pipe_peaks(double* out8_host, void* scratch_dev, nk_stream_t stream);

/* Number of kernels the library launched on this thread since the last call with reset != 0 (bench accounting). */
int64_t nk_launch_count(int reset);

#ifdef __cplusplus
}
#endif
#endif /* NKB200_H */
