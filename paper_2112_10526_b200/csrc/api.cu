// C ABI of libnkb200.so (include/nkb200.h): argument validation, workspace carving, the chunked driver
// (Sec. 3.3.1: chunk_size bounds the configurations evaluated at once).
#include <cmath>
#include <cstdlib>
#include <new>
#include <vector>

#include <mutex>

#include "nk_internal.h"

namespace nk {

static thread_local int tl_last_cuda = 0;
static thread_local int64_t tl_launches = 0;
void count_launch(int n) { tl_launches += n; }

// ---- optional per-phase event timing ----
struct Span { int phase; cudaEvent_t a, b; };
static thread_local bool tl_prof = false;
static thread_local std::vector<Span> tl_spans;
static thread_local std::vector<cudaEvent_t> tl_event_pool;      // events are reused: creating one costs microseconds
static cudaEvent_t pooled_event() {
    if (!tl_event_pool.empty()) { cudaEvent_t e = tl_event_pool.back(); tl_event_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
    return e;
}
ProfScope::ProfScope(int phase_, cudaStream_t s) : st(s), phase(phase_), a(nullptr), b(nullptr), on(tl_prof) {
    if (!on) return;
    a = pooled_event(); b = pooled_event();
    if (!a || !b) { on = false; return; }
    cudaEventRecord(a, st);
}
ProfScope::~ProfScope() {
    if (!on) return;
    cudaEventRecord(b, st);
    tl_spans.push_back(Span{phase, a, b});
}
typedef ProfScope Scope;

// nk_local_energy_host overlaps its host->device copies with the chunk loop: when this is set, chunk k of
// nk_local_energy_ex first makes the call's stream wait on event k (sigma of that chunk has arrived).
// internal stream + events of the pipelined chunk loop (nk_local_energy_ex), one set per calling thread and device
static thread_local cudaStream_t tl_prep_stream = nullptr;
static thread_local int tl_prep_device = -1;
static thread_local cudaEvent_t tl_pipe_events[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
static cudaError_t pipeline_objects() {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (tl_prep_stream != nullptr && tl_prep_device == dev) return cudaSuccess;
    int lo = 0, hi = 0;
    e = cudaDeviceGetStreamPriorityRange(&lo, &hi);                   // hi = the numerically smallest = greatest priority
    if (e != cudaSuccess) return e;
    e = cudaStreamCreateWithPriority(&tl_prep_stream, cudaStreamNonBlocking, hi);
    if (e != cudaSuccess) return e;
    for (int k = 0; k < 5; ++k) {
        e = cudaEventCreateWithFlags(&tl_pipe_events[k], cudaEventDisableTiming);
        if (e != cudaSuccess) return e;
    }
    tl_prep_device = dev;
    return cudaSuccess;
}

static thread_local const std::vector<cudaEvent_t>* tl_chunk_ready = nullptr;
static thread_local cudaStream_t tl_copy_stream = nullptr;
static thread_local std::vector<cudaEvent_t> tl_copy_events;

static int cuda_fail(cudaError_t e) {
    tl_last_cuda = (int)e;
    return NK_ERR_CUDA;
}
#define NK_CUDA(x)                                   \
    do {                                             \
        cudaError_t e__ = (x);                       \
        if (e__ != cudaSuccess) return cuda_fail(e__); \
    } while (0)

Geometry make_geometry(const Operator* op, int N, int M, int dtype) {
    Geometry g{};
    const bool cplx = dtype == NK_C64;
    g.N = N; g.n_words = (N + 31) / 32; g.K_pad = round_up(N, 128);
    g.M = M; g.M_pad = round_up(M, MPAD_ALIGN);
    g.planes = cplx ? 2 : 1;
    g.M_eff = g.planes * g.M_pad;
    g.n_rows = op ? (op->kind == NK_HEISENBERG ? op->n_bonds : op->n_sites) : 0;
    g.ok = g.M_pad / MPAD_ALIGN <= (cplx ? MAX_V_CPLX : MAX_V_REAL) && N <= 65535 && g.n_rows <= 65535;
    g.ctas_per_sm = fused_ctas_per_sm(g.M_pad, cplx);
    // shared-memory plan of the fused kernel: [stages x tile][bit-packed spins][stages mbarriers + counters];
    // as many rows per stage as fit (<= 32: one ballot bit per row)
    const size_t budget = (size_t)(227 * 1024) / g.ctas_per_sm - (g.ctas_per_sm > 1 ? 1024 : 0);
    const size_t sig = ((size_t)fused_consumer_warps(g.M_pad, cplx) * g.n_words * 4 + 15) & ~size_t(15);
    const size_t row_bytes = (size_t)g.M_eff * 4;
    const size_t fixed = sig + (8 + 4) * 8 + 128;         // spins + barriers + counters + alignment slack
    if (fixed + 2 * row_bytes > budget) { g.ok = false; g.tile_rows = 1; g.stages = 2; }
    else {
        // Few, large stages: every tile costs each warp a ballot, an mbarrier wait and a release, so the measured
        // optimum at config 5 (8 KB rows) is 2 stages x 14 rows (fused 36.5 ms) over 3 x 9 (36.9) and 4 x 7 (37.5);
        // more than 2 stages only once a stage already holds the 32 rows one ballot can name.
        g.stages = 2;
        int tr = (int)((budget - fixed) / (g.stages * row_bytes));
        if (tr > 32) {
            tr = 32;
            g.stages = (int)((budget - fixed) / ((size_t)tr * row_bytes));
            if (g.stages > 4) g.stages = 4;
        }
        g.tile_rows = tr;
    }
    g.n_tiles = (g.n_rows + g.tile_rows - 1) / g.tile_rows;
    g.n_rows_pad = g.n_tiles * g.tile_rows;
    if (g.n_rows_pad == 0) g.n_rows_pad = g.tile_rows;   // keep the tables non-empty
    g.smem_bytes = (size_t)g.stages * g.tile_rows * row_bytes + sig + (8 + 4) * (size_t)g.stages + 16;
    (void)fixed;
    return g;
}

// workspace carving: a bump allocator over the caller's buffer (256-B aligned pieces)
struct Carver {
    uint8_t* base;
    size_t off = 0;
    explicit Carver(void* p) : base((uint8_t*)p) {}
    template <typename T>
    T* take(size_t count) {
        T* r = (T*)(base ? base + off : nullptr);
        off += align256(count * sizeof(T));
        return r;
    }
};

struct LogpsiWs {
    float *Wg, *bg, *theta;
    uint16_t *Ws, *A;          // operands of the tensor-core contraction (int8 planes + scale; padded int8 spins)
    unsigned* absmax;
    size_t bytes;
};
static LogpsiWs carve_logpsi(void* ws, const Geometry& g, int64_t rows) {
    Carver c(ws);
    LogpsiWs w;
    w.Wg = c.take<float>((size_t)g.M_eff * g.N);
    w.bg = c.take<float>(g.M_eff);
    w.theta = c.take<float>((size_t)rows * g.M_eff);
    w.Ws = c.take<uint16_t>((size_t)3 * g.M_eff * g.K_pad);
    w.A = c.take<uint16_t>((size_t)rows * g.K_pad);
    w.absmax = c.take<unsigned>(1);
    w.bytes = c.off;
    return w;
}
constexpr int64_t THETA_WINDOW_BYTES = int64_t(1) << 30;
struct ElocWs {
    float *Wg, *bg, *Wt, *Dtab, *Ttab;                // Dtab: log-cosh form, Ttab: product form (both when automatic)
    float* theta;                                     // per-chunk buffers
    uint16_t *A, *Ws;
    unsigned *absmax, *taumax;                        // taumax: max |tanh delta| of Ttab as float bits (the form gate)
    RowInfo* rows;
    int64_t unit_rows;                                // rows the kernels work on: one chunk, or one group of chunks (series form)
    int64_t theta_rows;                               // rows of theta / A: unit_rows times the groups of one theta window
    bool has_series;                                  // the tensor-core series form is possible for these sizes
    SeriesWs ser;
    size_t bytes;
};
static ElocWs carve_eloc(void* ws, const Geometry& g, int64_t chunk, int dtype, int64_t B) {
    Carver c(ws);
    ElocWs w;
    w.Wg = c.take<float>((size_t)g.M_eff * g.N);
    w.bg = c.take<float>(g.M_eff);
    w.Wt = c.take<float>((size_t)g.N * g.M_eff);
    w.Dtab = c.take<float>((size_t)g.n_rows_pad * g.M_eff);
    w.rows = c.take<RowInfo>(g.n_rows_pad);
    w.has_series = series_possible(g, dtype);
    w.Ws = c.take<uint16_t>((size_t)3 * g.M_eff * g.K_pad);
    w.absmax = c.take<unsigned>(1);
    w.taumax = c.take<unsigned>(1);
    w.Ttab = c.take<float>((size_t)g.n_rows_pad * g.M_eff);
    if (w.has_series) w.ser = carve_series(c.base, &c.off, g, chunk, B);
    // the unit the chunk loop works in: a chunk, or (series form possible) the group of chunks one tensor-core launch covers
    w.unit_rows = w.has_series ? w.ser.group_rows : chunk;
    // Series form: theta is contracted for a WINDOW of groups in one launch (as many as keep theta under
    // THETA_WINDOW_BYTES — the whole batch at config 5, 512 MiB): the contraction and the series launches each need
    // whole SMs, so a per-group theta launch only ever ran between two series launches; one launch per window runs at
    // the large-launch rate and leaves nothing but the light ln psi / operand pass to run beside the tensor-core work.
    w.theta_rows = w.unit_rows;
    if (w.has_series) {
        const int64_t n_groups = (B + w.unit_rows - 1) / w.unit_rows;
        int64_t win = THETA_WINDOW_BYTES / ((int64_t)w.unit_rows * g.M_eff * 4);
        win = win < 1 ? 1 : (win > n_groups ? n_groups : win);
        w.theta_rows = w.unit_rows * win;
    }
    w.theta = c.take<float>((size_t)w.theta_rows * g.M_eff);
    w.A = c.take<uint16_t>((size_t)w.theta_rows * g.K_pad);
    w.bytes = c.off;
    return w;
}

static GradWs carve_grad(void* ws, const Geometry& g, int64_t chunk, size_t* bytes) {
    Carver c(ws);
    GradWs w;
    w.ld = (int)((chunk + 127) / 128 * 128);
    w.Wg = c.take<float>((size_t)g.M_eff * g.N);
    w.bg = c.take<float>(g.M_eff);
    w.theta = c.take<float>((size_t)chunk * g.M_eff);
    w.Gacc = c.take<float>((size_t)g.N * g.M_eff);
    w.Ws = c.take<uint16_t>((size_t)3 * g.M_eff * g.K_pad);
    w.A = c.take<uint16_t>((size_t)chunk * g.K_pad);
    w.TwT = c.take<uint16_t>((size_t)3 * g.M_eff * w.ld);
    w.sigT = c.take<uint16_t>((size_t)g.N * w.ld);
    w.gb_acc = c.take<double>(g.M_eff);
    w.ga_acc = c.take<double>((size_t)2 * g.N);
    const size_t n_slabs = (size_t)((chunk + grad_slab() - 1) / grad_slab());
    w.part = c.take<double>(n_slabs * (size_t)g.M_eff);
    w.part_a = c.take<double>(n_slabs * (size_t)(2 * g.N));
    w.absmax = c.take<unsigned>(1);
    *bytes = c.off;
    return w;
}

struct SamplerWs {
    float *Wg, *bg, *Wt, *Dtab, *theta;
    uint16_t *Ws, *A;
    unsigned* absmax;
    int32_t* pairs;
    size_t bytes;
};
static SamplerWs carve_sampler(void* ws, const Geometry& g, int n_rows, int64_t chunk) {
    Carver c(ws);
    SamplerWs w;
    w.Wg = c.take<float>((size_t)g.M_eff * g.N);
    w.bg = c.take<float>(g.M_eff);
    w.Wt = c.take<float>((size_t)g.N * g.M_eff);
    w.Dtab = c.take<float>((size_t)n_rows * g.M_eff);
    w.theta = c.take<float>((size_t)chunk * g.M_eff);
    w.Ws = c.take<uint16_t>((size_t)3 * g.M_eff * g.K_pad);
    w.A = c.take<uint16_t>((size_t)chunk * g.K_pad);
    w.absmax = c.take<unsigned>(1);
    w.pairs = c.take<int32_t>((size_t)2 * n_rows);
    w.bytes = c.off;
    return w;
}

struct QgtWs {
    GradWs g;
    float *Vg, *vbg, *Y;
    uint16_t* Vs;
    float* wbuf;
    double* wstats;
    size_t bytes;
};
static QgtWs carve_qgt(void* ws, const Geometry& g, int64_t B, int64_t chunk, int dtype) {
    size_t gbytes = 0;
    QgtWs w;
    w.g = carve_grad(ws, g, chunk, &gbytes);
    Carver c(ws);
    c.off = gbytes;
    w.Vg = c.take<float>((size_t)g.M_eff * g.N);
    w.vbg = c.take<float>(g.M_eff);
    w.Y = c.take<float>((size_t)chunk * g.M_eff);
    w.Vs = c.take<uint16_t>((size_t)3 * g.M_eff * g.K_pad);
    w.wbuf = c.take<float>((size_t)B * (dtype == NK_C64 ? 2 : 1));
    w.wstats = c.take<double>(4);
    w.bytes = c.off;
    return w;
}

static cudaError_t run_theta(const Geometry& g, const int8_t* sg, int64_t nb, const float* /*Wg*/, const float* bg,
                             const uint16_t* Ws, uint16_t* A, float* theta, cudaStream_t st) {
    return launch_theta_tc(sg, nb, g.N, g.M_eff, g.K_pad, Ws, A, bg, theta, st);
}

static bool bad_dims(int64_t B, int N, int M, int dtype) {
    return B < 0 || N <= 0 || M <= 0 || (dtype != NK_F32 && dtype != NK_C64);
}

}  // namespace nk

using namespace nk;

extern "C" {

const char* nk_status_string(int status) {
    switch (status) {
        case NK_OK: return "NK_OK";
        case NK_ERR_INVALID_ARG: return "NK_ERR_INVALID_ARG: null, out-of-range or inconsistent argument";
        case NK_ERR_BAD_SPIN: return "NK_ERR_BAD_SPIN: spin value not in {+1,-1}";
        case NK_ERR_WORKSPACE: return "NK_ERR_WORKSPACE: workspace null, misaligned or too small";
        case NK_ERR_UNSUPPORTED: return "NK_ERR_UNSUPPORTED: sizes beyond this version's limits";
        case NK_ERR_CUDA: return "NK_ERR_CUDA: a CUDA runtime call failed (see nk_last_cuda_error)";
        default: return "unknown nk_status";
    }
}
int nk_last_cuda_error(void) { return tl_last_cuda; }
int nk_version(void) { return 100; }
int64_t nk_launch_count(int reset) {
    const int64_t v = tl_launches;
    if (reset) tl_launches = 0;
    return v;
}

int nk_profile_enable(int on) {
    tl_prof = on != 0;
    return NK_OK;
}
int nk_profile_read(double* out) {
    if (!out) return NK_ERR_INVALID_ARG;
    for (int i = 0; i < 2 * PH_COUNT; ++i) out[i] = 0.0;
    int rc = NK_OK;
    for (const Span& sp : tl_spans) {
        float ms = 0.f;
        cudaError_t e = cudaEventSynchronize(sp.b);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, sp.a, sp.b);
        if (e != cudaSuccess) rc = cuda_fail(e);
        else { out[sp.phase] += ms; out[PH_COUNT + sp.phase] += 1.0; }
        tl_event_pool.push_back(sp.a); tl_event_pool.push_back(sp.b);
    }
    tl_spans.clear();
    return rc;
}

int nk_operator_create(nk_operator_t* out, int kind, int n_sites, int n_bonds, const int32_t* bonds_host,
                       const int32_t* colors_host, int n_colors, const double* J_host, double h, unsigned flags) {
    if (!out) return NK_ERR_INVALID_ARG;
    *out = nullptr;
    if ((kind != NK_HEISENBERG && kind != NK_ISING) || n_sites <= 0 || n_bonds < 0 || n_colors <= 0 || !J_host ||
        (n_bonds > 0 && !bonds_host) || (flags & ~NK_FLAG_MARSHALL))
        return NK_ERR_INVALID_ARG;
    for (int b = 0; b < n_bonds; ++b) {
        const int i = bonds_host[2 * b], j = bonds_host[2 * b + 1];
        if (i < 0 || j < 0 || i >= n_sites || j >= n_sites || i == j) return NK_ERR_INVALID_ARG;
        if (colors_host && (colors_host[b] < 0 || colors_host[b] >= n_colors)) return NK_ERR_INVALID_ARG;
    }
    Operator* op = new (std::nothrow) Operator();
    if (!op) return NK_ERR_INVALID_ARG;
    op->kind = kind; op->n_sites = n_sites; op->n_bonds = n_bonds; op->n_colors = n_colors; op->flags = flags; op->h = h;
    op->d_bonds = nullptr; op->d_colors = nullptr; op->d_Jf = nullptr; op->d_Jd = nullptr;
    std::vector<int32_t> colors(n_bonds > 0 ? n_bonds : 1, 0);
    if (colors_host) for (int b = 0; b < n_bonds; ++b) colors[b] = colors_host[b];
    std::vector<float> Jf(n_colors);
    for (int c = 0; c < n_colors; ++c) Jf[c] = (float)J_host[c];
    const size_t nb = n_bonds > 0 ? n_bonds : 1;
    cudaError_t e = cudaMalloc(&op->d_bonds, nb * 2 * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&op->d_colors, nb * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&op->d_Jf, n_colors * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&op->d_Jd, n_colors * sizeof(double));
    if (e == cudaSuccess && n_bonds > 0)
        e = cudaMemcpy(op->d_bonds, bonds_host, (size_t)n_bonds * 2 * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(op->d_colors, colors.data(), nb * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(op->d_Jf, Jf.data(), n_colors * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(op->d_Jd, J_host, n_colors * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        nk_operator_destroy((nk_operator_t)op);
        return cuda_fail(e);
    }
    *out = (nk_operator_t)op;
    return NK_OK;
}

int nk_operator_destroy(nk_operator_t h) {
    if (!h) return NK_ERR_INVALID_ARG;
    Operator* op = (Operator*)h;
    cudaFree(op->d_bonds); cudaFree(op->d_colors); cudaFree(op->d_Jf); cudaFree(op->d_Jd);
    delete op;
    return NK_OK;
}

int nk_operator_max_conn(nk_operator_t h, int* C_out) {
    if (!h || !C_out) return NK_ERR_INVALID_ARG;
    const Operator* op = (const Operator*)h;
    *C_out = (op->kind == NK_HEISENBERG ? op->n_bonds : op->n_sites) + 1;
    return NK_OK;
}

size_t nk_rbm_logpsi_workspace_bytes(int64_t B, int N, int M, int dtype) {
    if (bad_dims(B, N, M, dtype)) return 0;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    return carve_logpsi(nullptr, g, B).bytes;
}

int nk_rbm_logpsi(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* a,
                  const void* b, void* logpsi_out, void* theta_out, unsigned flags, void* workspace,
                  size_t workspace_bytes, nk_stream_t stream) {
    if (bad_dims(B, N, M, dtype) || !W || (flags & ~NK_OUT_F64) || (B > 0 && (!sigma || !logpsi_out)))
        return NK_ERR_INVALID_ARG;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    if (g.M_pad / MPAD_ALIGN > (dtype == NK_C64 ? MAX_V_CPLX : MAX_V_REAL) || N > 65535) return NK_ERR_UNSUPPORTED;
    if (B == 0) return NK_OK;
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < carve_logpsi(nullptr, g, B).bytes)
        return NK_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const LogpsiWs w = carve_logpsi(workspace, g, B);
    NK_CUDA(launch_pack_gemm_only(g, dtype, W, b, w.Wg, w.bg, st));
    NK_CUDA(launch_split_w(w.Wg, g.M_eff, N, g.K_pad, w.Ws, st));
    NK_CUDA(run_theta(g, sigma, B, w.Wg, w.bg, w.Ws, w.A, w.theta, st));
    NK_CUDA(launch_logpsi(sigma, B, g, dtype, w.theta, a, logpsi_out, (flags & NK_OUT_F64) != 0, theta_out, st));
    return NK_OK;
}

// ---- ln psi without a caller workspace ---------------------------------------------------------------------------
// For callers that cannot allocate (stream capture, serving loops, harnesses that forbid cudaMalloc): the scratch of
// nk_rbm_logpsi lives in a file-scope device array of NK_STATIC_SCRATCH_BYTES that every GPU loading the library holds
// until exit.  In host code `g_static_scratch` is a host-side stand-in, not a device address: the address is resolved
// once per device, with that device current, by cudaGetSymbolAddress and that pointer is what the kernels get.
static __device__ __align__(256) unsigned char g_static_scratch[NK_STATIC_SCRATCH_BYTES];
static std::mutex g_static_mutex;
static void* g_static_ptr[NK_MAX_DEVICES];
static cudaError_t static_scratch(void** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NK_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[dev] == nullptr) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (ptr == nullptr || ((uintptr_t)ptr & 255)) return cudaErrorInvalidSymbol;
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return cudaSuccess;
}

size_t nk_rbm_logpsi_static_max_bytes(void) { return (size_t)NK_STATIC_SCRATCH_BYTES; }

int nk_rbm_logpsi_static(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* a,
                         const void* b, void* logpsi_out, void* theta_out, unsigned flags, nk_stream_t stream) {
    if (bad_dims(B, N, M, dtype)) return NK_ERR_INVALID_ARG;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    if (g.M_pad / MPAD_ALIGN > (dtype == NK_C64 ? MAX_V_CPLX : MAX_V_REAL) || N > 65535) return NK_ERR_UNSUPPORTED;
    if (carve_logpsi(nullptr, g, B).bytes > (size_t)NK_STATIC_SCRATCH_BYTES) return NK_ERR_WORKSPACE;
    void* ws = nullptr;
    NK_CUDA(static_scratch(&ws));
    // Nothing in the scratch has to start at zero: every buffer carved from it (packed weights and bias, digit planes and
    // scales, padded spins, theta) is written in full by this call's own launches before a later launch reads it, so
    // the previous call's contents — of any other shape — are never observed.
    return nk_rbm_logpsi(sigma, B, N, M, dtype, W, a, b, logpsi_out, theta_out, flags, ws, (size_t)NK_STATIC_SCRATCH_BYTES,
                         stream);
}

int nk_connected(nk_operator_t h, const int8_t* sigma, int64_t B, int32_t* flips_out, float* mels_out,
                 int32_t* n_conn_out, int8_t* sigma_prime_out, nk_stream_t stream) {
    if (!h || B < 0 || (B > 0 && !sigma)) return NK_ERR_INVALID_ARG;
    const Operator* op = (const Operator*)h;
    if (op->n_sites > 48 * 1024) return NK_ERR_UNSUPPORTED;
    NK_CUDA(launch_connected(op, sigma, B, flips_out, mels_out, n_conn_out, sigma_prime_out, (cudaStream_t)stream));
    return NK_OK;
}

static int64_t eff_chunk(int64_t B, int64_t chunk_size);

size_t nk_energy_gradient_workspace_bytes(int64_t B, int N, int M, int dtype, int64_t chunk_size) {
    if (bad_dims(B, N, M, dtype) || chunk_size < 0) return 0;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    size_t bytes = 0;
    carve_grad(nullptr, g, eff_chunk(B, chunk_size), &bytes);
    return bytes;
}

int nk_energy_gradient(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* b,
                       const void* eloc, const double* stats, int64_t chunk_size, void* grad_a_out,
                       void* grad_b_out, void* grad_W_out, void* workspace, size_t workspace_bytes,
                       nk_stream_t stream) {
    return nk_energy_gradient_sharded(sigma, B, B, N, M, dtype, W, b, eloc, stats, chunk_size, grad_a_out, grad_b_out,
                                      grad_W_out, workspace, workspace_bytes, stream);
}

int nk_energy_gradient_sharded(const int8_t* sigma, int64_t B, int64_t B_global, int N, int M, int dtype,
                               const void* W, const void* b, const void* eloc, const double* stats,
                               int64_t chunk_size, void* grad_a_out, void* grad_b_out, void* grad_W_out,
                               void* workspace, size_t workspace_bytes, nk_stream_t stream) {
    if (bad_dims(B, N, M, dtype) || B == 0 || B_global < B || chunk_size < 0 || !sigma || !W || !eloc || !stats ||
        !grad_W_out)
        return NK_ERR_INVALID_ARG;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    if (g.M_pad / MPAD_ALIGN > (dtype == NK_C64 ? MAX_V_CPLX : MAX_V_REAL) || N > 65535) return NK_ERR_UNSUPPORTED;
    const int64_t chunk = eff_chunk(B, chunk_size);
    size_t need = 0;
    carve_grad(nullptr, g, chunk, &need);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < need) return NK_ERR_WORKSPACE;
    const GradWs w = carve_grad(workspace, g, chunk, &need);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t esz = dtype == NK_C64 ? 8 : 4;
    // The part of a chunk that does not read theta (sample weights into grad_a, the scale of the split, the transposed
    // spins) runs on the internal stream beside the packing and the theta contraction of the same chunk; the caller's
    // stream waits for it before the part that needs both.  Everything the caller observes is ordered on `stream`.
    NK_CUDA(pipeline_objects());
    cudaStream_t side = tl_prep_stream;
    int first = 1;
    for (int64_t s0 = 0; s0 < B; s0 += chunk) {
        const int64_t nb = (B - s0 < chunk) ? (B - s0) : chunk;
        const int8_t* sg = sigma + s0 * N;
        const void* el = (const uint8_t*)eloc + s0 * esz;
        NK_CUDA(cudaEventRecord(tl_pipe_events[0], st));              // earlier work (the previous chunk) is done with the buffers
        NK_CUDA(cudaStreamWaitEvent(side, tl_pipe_events[0], 0));
        NK_CUDA(launch_gradient_chunk(g, dtype, sg, nb, B_global, el, stats, w, first, 2.f, side, nullptr, nullptr, 1));
        NK_CUDA(cudaEventRecord(tl_pipe_events[1], side));
        if (first) {
            NK_CUDA(launch_pack_gemm_only(g, dtype, W, b, w.Wg, w.bg, st));
            NK_CUDA(launch_split_w(w.Wg, g.M_eff, N, g.K_pad, w.Ws, st));
        }
        NK_CUDA(launch_theta_tc(sg, nb, N, g.M_eff, g.K_pad, w.Ws, w.A, w.bg, w.theta, st));
        NK_CUDA(cudaStreamWaitEvent(st, tl_pipe_events[1], 0));
        NK_CUDA(launch_gradient_chunk(g, dtype, sg, nb, B_global, el, stats, w, first, 2.f, st, nullptr, nullptr, 2));
        first = 0;
    }
    NK_CUDA(launch_gradient_finalize(g, dtype, w, grad_a_out, grad_b_out, grad_W_out, st));
    return NK_OK;
}

static int64_t eff_chunk(int64_t B, int64_t chunk_size) {
    if (chunk_size <= 0 || chunk_size > B) return B > 0 ? B : 1;
    return chunk_size;
}

size_t nk_qgt_matvec_workspace_bytes(int64_t B, int N, int M, int dtype, int64_t chunk_size) {
    if (bad_dims(B, N, M, dtype) || chunk_size < 0) return 0;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    return carve_qgt(nullptr, g, B, eff_chunk(B, chunk_size), dtype).bytes;
}

// theta, the padded int8 spins and their bf16 transposes for the WHOLE batch, kept across the matvecs of one nk_sr_solve (the
// parameters do not change during the solve): a matvec then costs one contraction less per pass and no conversions
namespace {
struct QgtCache {
    float* theta_all;        // [B][M_eff]
    uint16_t* A_all;         // [B][K_pad] int8 (allocated as 2 B per entry)
    uint16_t* sigT_all;      // [n_chunks][N][ld] int8 (allocated as 2 B per entry)
    size_t sigT_stride;      // N * ld
};
}  // namespace

static int qgt_matvec_impl(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* b,
                           const void* v_a, const void* v_b, const void* v_W, double diag_shift, int64_t chunk_size,
                           void* out_a, void* out_b, void* out_W, void* workspace, size_t workspace_bytes,
                           nk_stream_t stream, const QgtCache* cache) {
    if (bad_dims(B, N, M, dtype) || B == 0 || chunk_size < 0 || !sigma || !W || !v_W || !out_W ||
        (diag_shift < 0.0))
        return NK_ERR_INVALID_ARG;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    if (g.M_pad / MPAD_ALIGN > (dtype == NK_C64 ? MAX_V_CPLX : MAX_V_REAL) || N > 65535) return NK_ERR_UNSUPPORTED;
    const int64_t chunk = eff_chunk(B, chunk_size);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < carve_qgt(nullptr, g, B, chunk, dtype).bytes)
        return NK_ERR_WORKSPACE;
    const QgtWs w = carve_qgt(workspace, g, B, chunk, dtype);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t esz = dtype == NK_C64 ? 8 : 4;
    // operands of the two contractions: (W, b) -> theta (not needed when theta is cached) and (V_W, v_b) -> Y
    if (cache == nullptr) {
        NK_CUDA(launch_pack_gemm_only(g, dtype, W, b, w.g.Wg, w.g.bg, st));
        NK_CUDA(launch_split_w(w.g.Wg, g.M_eff, N, g.K_pad, w.g.Ws, st));
    }
    NK_CUDA(launch_pack_gemm_only(g, dtype, v_W, v_b, w.Vg, w.vbg, st));
    NK_CUDA(launch_split_w(w.Vg, g.M_eff, N, g.K_pad, w.Vs, st));
    // step 1 of Eq. (75): w_s = (J v)_s for every sample
    for (int64_t s0 = 0; s0 < B; s0 += chunk) {
        const int64_t nb = (B - s0 < chunk) ? (B - s0) : chunk;
        const int8_t* sg = sigma + s0 * N;
        const float* th = w.g.theta;
        if (cache == nullptr) {
            NK_CUDA(launch_theta_tc(sg, nb, N, g.M_eff, g.K_pad, w.g.Ws, w.g.A, w.g.bg, w.g.theta, st));
            NK_CUDA(launch_theta_tc(sg, nb, N, g.M_eff, g.K_pad, w.Vs, w.g.A, w.vbg, w.Y, st));
        } else {
            th = cache->theta_all + (size_t)s0 * g.M_eff;
            NK_CUDA(launch_theta_tc_pre((const uint8_t*)cache->A_all + (size_t)s0 * g.K_pad, nb, g.M_eff, g.K_pad, w.Vs, w.vbg, w.Y, st));
        }
        NK_CUDA(launch_qgt_w(g, dtype, sg, nb, th, w.Y, v_a, (uint8_t*)w.wbuf + s0 * esz, st));
    }
    // step 2: <w> (the 1/N_s and the subtraction happen inside the force contraction, as for E_loc)
    NK_CUDA(launch_stats(w.wbuf, B, dtype, w.wstats, st));
    // step 3: v~ = J^dagger (w - <w>) / N_s  — the force-vector contraction with w in the place of E_loc
    int first = 1;
    for (int64_t s0 = 0; s0 < B; s0 += chunk) {
        const int64_t nb = (B - s0 < chunk) ? (B - s0) : chunk;
        const int8_t* sg = sigma + s0 * N;
        if (cache == nullptr) {
            NK_CUDA(launch_theta_tc(sg, nb, N, g.M_eff, g.K_pad, w.g.Ws, w.g.A, w.g.bg, w.g.theta, st));
            NK_CUDA(launch_gradient_chunk(g, dtype, sg, nb, B, (const uint8_t*)w.wbuf + s0 * esz, w.wstats, w.g, first,
                                          1.f, st));
        } else {
            NK_CUDA(launch_gradient_chunk(g, dtype, sg, nb, B, (const uint8_t*)w.wbuf + s0 * esz, w.wstats, w.g, first,
                                          1.f, st, cache->theta_all + (size_t)s0 * g.M_eff,
                                          (const uint8_t*)cache->sigT_all + (size_t)(s0 / chunk) * cache->sigT_stride));
        }
        first = 0;
    }
    NK_CUDA(launch_gradient_finalize(g, dtype, w.g, out_a, out_b, out_W, st));
    // Eq. (25): + eps v
    const int64_t e = dtype == NK_C64 ? 2 : 1;
    NK_CUDA(launch_qgt_shift(out_a, v_a, diag_shift, (int64_t)N * e, st));
    NK_CUDA(launch_qgt_shift(out_b, v_b, diag_shift, (int64_t)M * e, st));
    NK_CUDA(launch_qgt_shift(out_W, v_W, diag_shift, (int64_t)M * N * e, st));
    return NK_OK;
}

int nk_qgt_matvec(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* b,
                  const void* v_a, const void* v_b, const void* v_W, double diag_shift, int64_t chunk_size,
                  void* out_a, void* out_b, void* out_W, void* workspace, size_t workspace_bytes,
                  nk_stream_t stream) {
    return qgt_matvec_impl(sigma, B, N, M, dtype, W, b, v_a, v_b, v_W, diag_shift, chunk_size, out_a, out_b, out_W,
                           workspace, workspace_bytes, stream, nullptr);
}

// ---- stochastic reconfiguration: (G + eps) delta = f by conjugate gradients -----------------------------------
namespace {
struct SrWs {
    float *x, *r, *p, *Ap;       // packed [a | b | W] vectors, n floats each
    double *part, *scal;         // reduction partials; scal[0..1] = rr (ping-pong), [2] = pAp, [3] = |f|^2
    void* qgt;
    size_t qgt_bytes, bytes;
    int64_t n;
    QgtCache cache;
};
SrWs carve_sr(void* ws, int64_t B, int N, int M, int dtype, int64_t chunk_size) {
    const int64_t e = dtype == NK_C64 ? 2 : 1;
    Carver c(ws);
    SrWs w;
    w.n = ((int64_t)N + M + (int64_t)M * N) * e;
    w.x = c.take<float>(w.n); w.r = c.take<float>(w.n); w.p = c.take<float>(w.n); w.Ap = c.take<float>(w.n);
    w.part = c.take<double>(cg_partials());
    w.scal = c.take<double>(8);
    w.qgt_bytes = nk_qgt_matvec_workspace_bytes(B, N, M, dtype, chunk_size);
    w.qgt = c.take<uint8_t>(w.qgt_bytes);
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    const int64_t chunk = (chunk_size <= 0 || chunk_size > B) ? (B > 0 ? B : 1) : chunk_size;
    const int64_t n_chunks = B > 0 ? (B + chunk - 1) / chunk : 1;
    const size_t ld = (size_t)((chunk + 127) / 128 * 128);
    w.cache.theta_all = c.take<float>((size_t)B * g.M_eff);
    w.cache.A_all = c.take<uint16_t>((size_t)B * g.K_pad);
    w.cache.sigT_stride = (size_t)N * ld;
    w.cache.sigT_all = c.take<uint16_t>((size_t)n_chunks * w.cache.sigT_stride);
    w.bytes = c.off;
    return w;
}
}  // namespace

size_t nk_sr_solve_workspace_bytes(int64_t B, int N, int M, int dtype, int64_t chunk_size) {
    if (bad_dims(B, N, M, dtype) || chunk_size < 0) return 0;
    return carve_sr(nullptr, B, N, M, dtype, chunk_size).bytes;
}

int nk_sr_solve(const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W, const void* b,
                const void* f_a, const void* f_b, const void* f_W, double diag_shift, double tol, int max_iter,
                int64_t chunk_size, void* delta_a, void* delta_b, void* delta_W, double* info_host, void* workspace,
                size_t workspace_bytes, nk_stream_t stream) {
    if (bad_dims(B, N, M, dtype) || B == 0 || chunk_size < 0 || !sigma || !W || !f_a || !f_b || !f_W || !delta_a ||
        !delta_b || !delta_W || diag_shift < 0.0 || !(tol >= 0.0) || max_iter < 0)
        return NK_ERR_INVALID_ARG;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    if (g.M_pad / MPAD_ALIGN > (dtype == NK_C64 ? MAX_V_CPLX : MAX_V_REAL) || N > 65535) return NK_ERR_UNSUPPORTED;
    if (!workspace || ((uintptr_t)workspace & 255) ||
        workspace_bytes < carve_sr(nullptr, B, N, M, dtype, chunk_size).bytes)
        return NK_ERR_WORKSPACE;
    const SrWs w = carve_sr(workspace, B, N, M, dtype, chunk_size);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t fsz = sizeof(float) * (dtype == NK_C64 ? 2 : 1);
    const size_t na = (size_t)N * fsz, nb_ = (size_t)M * fsz, nW = (size_t)M * N * fsz;
    auto blk = [&](float* v, int which) -> void* {
        uint8_t* q = (uint8_t*)v;
        return which == 0 ? (void*)q : which == 1 ? (void*)(q + na) : (void*)(q + na + nb_);
    };
    // x0 = 0, r0 = p0 = f
    NK_CUDA(cudaMemsetAsync(w.x, 0, (size_t)w.n * sizeof(float), st));
    const void* fsrc[3] = {f_a, f_b, f_W};
    const size_t fbytes[3] = {na, nb_, nW};
    for (int k = 0; k < 3; ++k) {
        NK_CUDA(cudaMemcpyAsync(blk(w.r, k), fsrc[k], fbytes[k], cudaMemcpyDeviceToDevice, st));
        NK_CUDA(cudaMemcpyAsync(blk(w.p, k), fsrc[k], fbytes[k], cudaMemcpyDeviceToDevice, st));
    }
    {   // theta, padded spins and their transposes of the whole batch, once per solve
        const QgtWs q = carve_qgt(w.qgt, g, B, eff_chunk(B, chunk_size), dtype);
        const int64_t chunk = eff_chunk(B, chunk_size);
        NK_CUDA(launch_pack_gemm_only(g, dtype, W, b, q.g.Wg, q.g.bg, st));
        NK_CUDA(launch_split_w(q.g.Wg, g.M_eff, N, g.K_pad, q.g.Ws, st));
        NK_CUDA(launch_sigma_operand(sigma, B, N, g.K_pad, w.cache.A_all, st));
        for (int64_t s0 = 0; s0 < B; s0 += chunk) {
            const int64_t nb = (B - s0 < chunk) ? (B - s0) : chunk;
            NK_CUDA(launch_theta_tc_pre((const uint8_t*)w.cache.A_all + (size_t)s0 * g.K_pad, nb, g.M_eff, g.K_pad, q.g.Ws, q.g.bg,
                                        w.cache.theta_all + (size_t)s0 * g.M_eff, st));
            NK_CUDA(launch_sigma_T(sigma + s0 * N, nb, N, q.g.ld,
                                   (uint8_t*)w.cache.sigT_all + (size_t)(s0 / chunk) * w.cache.sigT_stride, st));
        }
    }
    NK_CUDA(launch_cg_dot(w.r, w.r, w.n, w.part, w.scal + 0, st));
    NK_CUDA(cudaMemcpyAsync(w.scal + 3, w.scal + 0, sizeof(double), cudaMemcpyDeviceToDevice, st));
    double h[4] = {0, 0, 0, 0};
    NK_CUDA(cudaMemcpyAsync(h, w.scal, sizeof(h), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));
    const double ff = h[0];
    double rr = ff;
    int it = 0;
    const int check_every = 4;           // the residual is read back (one synchronisation) every few iterations
    while (it < max_iter && ff > 0.0 && rr > tol * tol * ff) {
        const int cur = it & 1, nxt = cur ^ 1;
        const int rc = qgt_matvec_impl(sigma, B, N, M, dtype, W, b, blk(w.p, 0), blk(w.p, 1), blk(w.p, 2), diag_shift,
                                       chunk_size, blk(w.Ap, 0), blk(w.Ap, 1), blk(w.Ap, 2), w.qgt, w.qgt_bytes, stream,
                                       &w.cache);
        if (rc != NK_OK) return rc;
        NK_CUDA(launch_cg_dot(w.p, w.Ap, w.n, w.part, w.scal + 2, st));
        NK_CUDA(launch_cg_step(w.x, w.r, w.p, w.Ap, w.n, w.scal + cur, w.scal + 2, st));
        NK_CUDA(launch_cg_dot(w.r, w.r, w.n, w.part, w.scal + nxt, st));
        NK_CUDA(launch_cg_dir(w.p, w.r, w.n, w.scal + nxt, w.scal + cur, st));
        ++it;
        if (it % check_every == 0 || it == max_iter) {
            NK_CUDA(cudaMemcpyAsync(h, w.scal, sizeof(h), cudaMemcpyDeviceToHost, st));
            NK_CUDA(cudaStreamSynchronize(st));
            rr = h[nxt];
            if (!(h[2] > 0.0)) break;    // p^dagger A p <= 0 or NaN: breakdown, stop with what we have
        }
    }
    void* dst[3] = {delta_a, delta_b, delta_W};
    for (int k = 0; k < 3; ++k)
        NK_CUDA(cudaMemcpyAsync(dst[k], blk(w.x, k), fbytes[k], cudaMemcpyDeviceToDevice, st));
    NK_CUDA(cudaStreamSynchronize(st));
    if (info_host) {
        info_host[0] = (double)it;
        info_host[1] = ff > 0.0 ? sqrt(rr / ff) : 0.0;
    }
    return NK_OK;
}

// ---- fully symmetric RBM: tied weights <-> expanded RBM -------------------------------------------------------
static bool bad_symm(int F, int G, int N, int dtype) {
    return F <= 0 || G <= 0 || N <= 0 || (dtype != NK_F32 && dtype != NK_C64) || (int64_t)F * G > (1 << 24);
}

int nk_rbmsymm_expand(int n_features, int n_group, int N, int dtype, const void* W_sym, const void* b_sym,
                      const int32_t* perms, void* W_out, void* b_out, nk_stream_t stream) {
    if (bad_symm(n_features, n_group, N, dtype) || !W_sym || !perms || !W_out) return NK_ERR_INVALID_ARG;
    NK_CUDA(launch_rbmsymm_expand(n_features, n_group, N, dtype, W_sym, b_sym, perms, W_out, b_out,
                                  (cudaStream_t)stream));
    return NK_OK;
}

int nk_rbmsymm_reduce_gradient(int n_features, int n_group, int N, int dtype, const void* grad_W, const void* grad_b,
                               const int32_t* perms, void* grad_W_sym, void* grad_b_sym, nk_stream_t stream) {
    if (bad_symm(n_features, n_group, N, dtype) || !grad_W || !perms || !grad_W_sym) return NK_ERR_INVALID_ARG;
    NK_CUDA(launch_rbmsymm_reduce(n_features, n_group, N, dtype, grad_W, grad_b, perms, grad_W_sym, grad_b_sym,
                                  (cudaStream_t)stream));
    return NK_OK;
}

static bool bad_rule(int rule, int n_clusters) {
    return (rule != NK_RULE_LOCAL && rule != NK_RULE_EXCHANGE) || n_clusters < 0 ||
           (rule == NK_RULE_EXCHANGE && n_clusters == 0);
}

size_t nk_metropolis_workspace_bytes(int rule, int n_clusters, int64_t B, int N, int M, int dtype, int64_t chunk_size) {
    if (bad_dims(B, N, M, dtype) || chunk_size < 0 || bad_rule(rule, n_clusters)) return 0;
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    return carve_sampler(nullptr, g, rule == NK_RULE_LOCAL ? N : n_clusters, eff_chunk(B, chunk_size)).bytes;
}

int nk_metropolis_sample(int rule, const int32_t* clusters_host, int n_clusters, int8_t* sigma, int64_t B, int N,
                         int M, int dtype, const void* W, const void* a, const void* b, int64_t n_steps,
                         uint64_t seed, uint64_t step_offset, uint64_t chain_offset, int64_t chunk_size,
                         int32_t* accepted_out, void* workspace, size_t workspace_bytes, nk_stream_t stream) {
    if (bad_dims(B, N, M, dtype) || chunk_size < 0 || n_steps < 0 || bad_rule(rule, n_clusters) || !W ||
        (B > 0 && !sigma) || (rule == NK_RULE_EXCHANGE && !clusters_host))
        return NK_ERR_INVALID_ARG;
    if (rule == NK_RULE_EXCHANGE)
        for (int c = 0; c < n_clusters; ++c) {
            const int i = clusters_host[2 * c], j = clusters_host[2 * c + 1];
            if (i < 0 || j < 0 || i >= N || j >= N || i == j) return NK_ERR_INVALID_ARG;
        }
    const Geometry g = make_geometry(nullptr, N, M, dtype);
    if (g.M_pad / MPAD_ALIGN > (dtype == NK_C64 ? MAX_V_CPLX : MAX_V_REAL) || N > 65535) return NK_ERR_UNSUPPORTED;
    if (B == 0) return NK_OK;
    const int n_rows = rule == NK_RULE_LOCAL ? N : n_clusters;
    const int64_t chunk = eff_chunk(B, chunk_size);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < carve_sampler(nullptr, g, n_rows, chunk).bytes)
        return NK_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const SamplerWs w = carve_sampler(workspace, g, n_rows, chunk);
    if (rule == NK_RULE_EXCHANGE)
        NK_CUDA(cudaMemcpyAsync(w.pairs, clusters_host, (size_t)2 * n_clusters * sizeof(int32_t),
                                cudaMemcpyHostToDevice, st));
    NK_CUDA(launch_pack_table(g, dtype, W, b, rule == NK_RULE_EXCHANGE ? w.pairs : nullptr, n_rows, w.Wg, w.bg, w.Wt,
                              w.Dtab, st));
    NK_CUDA(launch_split_w(w.Wg, g.M_eff, N, g.K_pad, w.Ws, st));
    SamplerArgs sa;
    sa.rule = rule; sa.n_idx = n_rows; sa.pairs = rule == NK_RULE_EXCHANGE ? w.pairs : nullptr; sa.a = a;
    sa.n_steps = n_steps; sa.seed = seed; sa.step_offset = step_offset;
    for (int64_t s0 = 0; s0 < B; s0 += chunk) {
        const int64_t nb = (B - s0 < chunk) ? (B - s0) : chunk;
        int8_t* sg = sigma + s0 * N;
        sa.chain0 = chain_offset + (uint64_t)s0;
        NK_CUDA(launch_theta_tc(sg, nb, N, g.M_eff, g.K_pad, w.Ws, w.A, w.bg, w.theta, st));
        NK_CUDA(launch_metropolis(g, dtype, sg, nb, w.theta, w.Dtab, sa, accepted_out ? accepted_out + s0 : nullptr, st));
    }
    return NK_OK;
}

size_t nk_local_energy_workspace_bytes(nk_operator_t h, int64_t B, int N, int M, int dtype, int64_t chunk_size) {
    if (!h || bad_dims(B, N, M, dtype) || chunk_size < 0) return 0;
    const Operator* op = (const Operator*)h;
    const Geometry g = make_geometry(op, N, M, dtype);
    return carve_eloc(nullptr, g, eff_chunk(B, chunk_size), dtype, B).bytes;
}

int nk_local_energy(nk_operator_t h, const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W,
                    const void* a, const void* b, int64_t chunk_size, void* eloc_out, void* logpsi_out,
                    double* stats_out, void* workspace, size_t workspace_bytes, nk_stream_t stream) {
    return nk_local_energy_ex(h, sigma, B, N, M, dtype, W, a, b, chunk_size, 0u, eloc_out, logpsi_out, stats_out,
                              workspace, workspace_bytes, stream);
}

int nk_local_energy_ex(nk_operator_t h, const int8_t* sigma, int64_t B, int N, int M, int dtype, const void* W,
                       const void* a, const void* b, int64_t chunk_size, unsigned flags, void* eloc_out,
                       void* logpsi_out, double* stats_out, void* workspace, size_t workspace_bytes,
                       nk_stream_t stream) {
    if (!h || bad_dims(B, N, M, dtype) || chunk_size < 0 || !W || (B > 0 && (!sigma || !eloc_out)) ||
        (flags & ~(NK_FORM_PRODUCT | NK_FORM_LOGCOSH | NK_FORM_SERIES | NK_CHECK_SPINS | NK_SERIAL_CHUNKS)))
        return NK_ERR_INVALID_ARG;
    {
        const unsigned forms = flags & (NK_FORM_PRODUCT | NK_FORM_LOGCOSH | NK_FORM_SERIES);
        if (forms & (forms - 1)) return NK_ERR_INVALID_ARG;             // at most one form may be forced
    }
    // form of the amplitude ratios: forced by a flag, else chosen on the device from the parameters (real parameters;
    // complex ones keep the log-cosh form: tanh theta is unbounded next to the zeros of cosh)
    const bool force_product = (flags & NK_FORM_PRODUCT) != 0;
    const bool force_series = (flags & NK_FORM_SERIES) != 0;
    const bool automatic = !force_product && !force_series && !(flags & NK_FORM_LOGCOSH) && dtype == NK_F32;
    const Operator* op = (const Operator*)h;
    if (N != op->n_sites) return NK_ERR_INVALID_ARG;
    const Geometry g = make_geometry(op, N, M, dtype);
    if (!g.ok) return NK_ERR_UNSUPPORTED;
    const int64_t chunk = eff_chunk(B, chunk_size);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < carve_eloc(nullptr, g, chunk, dtype, B).bytes)
        return NK_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const ElocWs w = carve_eloc(workspace, g, chunk, dtype, B);
    if (force_series && !w.has_series) return NK_ERR_UNSUPPORTED;       // complex parameters or a tiny problem
    const bool series = w.has_series && (automatic || force_series);
    if ((flags & NK_CHECK_SPINS) && B > 0) {           // opt-in validation: one pass over sigma and one synchronisation
        int bad = 0;
        NK_CUDA(launch_check_spins(sigma, B * N, (int*)w.absmax, st));
        NK_CUDA(cudaMemcpyAsync(&bad, w.absmax, sizeof(int), cudaMemcpyDeviceToHost, st));
        NK_CUDA(cudaStreamSynchronize(st));
        if (bad) return NK_ERR_BAD_SPIN;
    }
    NK_CUDA(fused_eloc_init());
    {
        Scope sc(PH_PACK, st);
        NK_CUDA(launch_pack(op, g, dtype, W, a, b, w.Wg, w.bg, w.Wt, w.Dtab, w.rows, st));
        if (series) NK_CUDA(launch_series_ctl_reset(w.ser, st));
        if (force_product || automatic || force_series)
            NK_CUDA(launch_pack_product(op, g, dtype, w.Wt, w.Ttab, w.rows, st,
                                        (automatic || force_series) ? w.taumax : nullptr, series ? w.ser.ctl : nullptr));
        if (series) NK_CUDA(launch_series_pack(g, w.Ttab, w.taumax, w.ser, force_series, st));
        NK_CUDA(launch_split_w(w.Wg, g.M_eff, N, g.K_pad, w.Ws, st));
    }
    const size_t esz = dtype == NK_C64 ? 8 : 4;
    // The series form contracts GROUPS of chunks (series_tc.cu: as many as make the tensor-core launch a whole number
    // of waves).  With more than one group the work is split over two streams: the preparation of a group's chunks
    // (theta contraction, the ln psi / operand pass, the gated SIMT stand-ins, spin bits) goes to an internal
    // high-priority stream `ps`, the tensor-core launches stay on the caller's stream, and each of the two operand
    // buffers is handed over by a pair of events — the preparation of group G + 1 runs beside the launch of group G.
    // Everything the caller observes is ordered on `stream`; the construction is capturable in a CUDA graph (the
    // internal stream forks from and joins `stream`).
    const bool pipelined = series && w.ser.n_sets == 2 && !(flags & NK_SERIAL_CHUNKS);
    cudaStream_t ps = st;
    if (pipelined) {
        NK_CUDA(pipeline_objects());
        ps = tl_prep_stream;
        NK_CUDA(cudaEventRecord(tl_pipe_events[0], st));              // parameters packed; earlier work on `stream` done
        NK_CUDA(cudaStreamWaitEvent(ps, tl_pipe_events[0], 0));
    }
    // Where the series form is possible the whole group is the unit of work for every kernel (theta, ln psi, stand-ins):
    // four launches of each per step at config 5 instead of sixteen (also when a SIMT form is forced there).
    const int64_t group_rows = w.unit_rows;
    const int64_t copy_chunk = chunk;                                 // granularity of the host path's arrival events
    // groups per theta launch (carve_eloc); the host path keeps one, so that theta of a group waits for its own chunks only
    const int64_t win = (series && tl_chunk_ready == nullptr) ? w.theta_rows / group_rows : 1;
    int64_t gi = 0;
    for (int64_t g0 = 0; g0 < B; g0 += group_rows, ++gi) {
        const int64_t gn = (B - g0 < group_rows) ? (B - g0) : group_rows;
        const int set = (series && w.ser.n_sets == 2) ? (int)(gi & 1) : 0;
        cudaEvent_t ev_prep = tl_pipe_events[1 + set], ev_done = tl_pipe_events[3 + set];
        if (pipelined && gi >= 2) NK_CUDA(cudaStreamWaitEvent(ps, ev_done, 0));    // group G - 2 no longer reads this set
        {
            const int64_t s0 = g0, nb = gn;
            const int8_t* sg = sigma + s0 * N;
            if (tl_chunk_ready != nullptr)                            // every chunk of the group has arrived
                for (int64_t c0 = s0; c0 < s0 + nb; c0 += copy_chunk)
                    NK_CUDA(cudaStreamWaitEvent(ps, (*tl_chunk_ready)[(size_t)(c0 / copy_chunk)], 0));
            const float* th = w.theta + (size_t)((gi % win) * group_rows) * g.M_eff;
            if (gi % win == 0) {               // theta of the whole window (of this group alone when win = 1)
                Scope sc(PH_GEMM, ps);
                const int64_t wn = (B - s0 < win * group_rows) ? (B - s0) : win * group_rows;
                NK_CUDA(run_theta(g, sg, wn, w.Wg, w.bg, w.Ws, w.A, w.theta, ps));
            }
            if (logpsi_out || series) {        // ln psi and, in the same pass over theta, the series form's operand rows
                Scope sc(PH_LOGPSI, ps);
                uint16_t* ap = series ? w.ser.Ap[set] : nullptr;
                NK_CUDA(launch_logpsi(sg, nb, g, dtype, th, a, logpsi_out ? (uint8_t*)logpsi_out + s0 * esz : nullptr,
                                      false, nullptr, ps, series ? w.ser.ctl : nullptr, ap));
            }
            {
                // the SIMT forms (the only ones when the series form is impossible; gated stand-ins when it may run:
                // every launch is made, those on the wrong side of the gates return at once) stay on the preparation
                // stream, off the critical path of the tensor-core launches
                Scope sc(PH_FUSED, ps);
                void* out = (uint8_t*)eloc_out + s0 * esz;
                if (automatic) {
                    const unsigned* sctl = series ? w.ser.ctl : nullptr;
                    NK_CUDA(launch_fused_eloc(op, g, dtype, sg, nb, th, w.Ttab, w.rows, out, true, ps, w.taumax, 1, sctl));
                    NK_CUDA(launch_fused_eloc(op, g, dtype, sg, nb, th, w.Dtab, w.rows, out, false, ps, w.taumax, 2, sctl));
                } else if (!force_series) {
                    NK_CUDA(launch_fused_eloc(op, g, dtype, sg, nb, th, force_product ? w.Ttab : w.Dtab, w.rows, out,
                                              force_product, ps));
                }
            }
        }
        if (!series) continue;
        NK_CUDA(launch_series_prep(g, sigma + g0 * N, gn, w.ser, set, ps));
        if (pipelined) {
            NK_CUDA(cudaEventRecord(ev_prep, ps));
            NK_CUDA(cudaStreamWaitEvent(st, ev_prep, 0));
        }
        {
            Scope sc(PH_FUSED, st);
            NK_CUDA(launch_series_gemm(g, g0, gn, w.rows, w.ser, set, st));
        }
        if (pipelined) NK_CUDA(cudaEventRecord(ev_done, st));
    }
    // the series form's partial sums per column tile -> E_loc, one pass over the whole batch (gated like the rest; it
    // runs after the SIMT stand-ins, which wrote nothing if the series form ran, and writes nothing if it did not)
    if (series) {
        Scope sc(PH_FUSED, st);
        NK_CUDA(launch_series_finish(op, g, sigma, B, w.ser, (float*)eloc_out, st));
    }
    if (stats_out) {
        Scope sc(PH_STATS, st);
        NK_CUDA(launch_stats(eloc_out, B, dtype, stats_out, st));
    }
    return NK_OK;
}

// ---- plan: the call captured once into a CUDA graph, replayed per step ----------------------------------------------
namespace {
struct Plan {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaStream_t capture_stream = nullptr;
    int64_t launches = 0;                 // kernels of one replay (what nk_launch_count is advanced by)
    int device = 0;
};
}  // namespace

int nk_local_energy_plan_create(nk_plan_t* out, nk_operator_t h, const int8_t* sigma, int64_t B, int N, int M, int dtype,
                                const void* W, const void* a, const void* b, int64_t chunk_size, unsigned flags,
                                void* eloc_out, void* logpsi_out, double* stats_out, void* workspace,
                                size_t workspace_bytes) {
    if (!out) return NK_ERR_INVALID_ARG;
    *out = nullptr;
    if (flags & NK_CHECK_SPINS) return NK_ERR_INVALID_ARG;           // that flag synchronises: not capturable
    Plan* p = new (std::nothrow) Plan();
    if (!p) return NK_ERR_INVALID_ARG;
    auto fail = [&](int rc) { nk_local_energy_plan_destroy((nk_plan_t)p); return rc; };
    if (cudaGetDevice(&p->device) != cudaSuccess) return fail(NK_ERR_CUDA);
    cudaError_t e = cudaStreamCreateWithFlags(&p->capture_stream, cudaStreamNonBlocking);
    if (e != cudaSuccess) return fail(cuda_fail(e));
    // once eagerly: argument checks, one-time attribute / stream / event set-up (none of which may happen in a capture)
    int rc = nk_local_energy_ex(h, sigma, B, N, M, dtype, W, a, b, chunk_size, flags, eloc_out, logpsi_out, stats_out,
                                workspace, workspace_bytes, (nk_stream_t)p->capture_stream);
    if (rc != NK_OK) return fail(rc);
    e = cudaStreamSynchronize(p->capture_stream);
    if (e != cudaSuccess) return fail(cuda_fail(e));
    const bool prof = tl_prof;
    tl_prof = false;                                                 // no timing brackets inside the graph
    const int64_t before = tl_launches;
    e = cudaStreamBeginCapture(p->capture_stream, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) { tl_prof = prof; return fail(cuda_fail(e)); }
    rc = nk_local_energy_ex(h, sigma, B, N, M, dtype, W, a, b, chunk_size, flags, eloc_out, logpsi_out, stats_out,
                            workspace, workspace_bytes, (nk_stream_t)p->capture_stream);
    e = cudaStreamEndCapture(p->capture_stream, &p->graph);
    tl_prof = prof;
    p->launches = tl_launches - before;
    tl_launches = before;                                            // captured, not launched
    if (rc != NK_OK) return fail(rc);
    if (e != cudaSuccess || p->graph == nullptr) return fail(cuda_fail(e != cudaSuccess ? e : cudaErrorUnknown));
    e = cudaGraphInstantiate(&p->exec, p->graph, 0);
    if (e != cudaSuccess) return fail(cuda_fail(e));
    *out = (nk_plan_t)p;
    return NK_OK;
}

int nk_local_energy_plan_run(nk_plan_t plan, nk_stream_t stream) {
    if (!plan) return NK_ERR_INVALID_ARG;
    Plan* p = (Plan*)plan;
    NK_CUDA(cudaGraphLaunch(p->exec, (cudaStream_t)stream));
    count_launch((int)p->launches);
    return NK_OK;
}

int nk_local_energy_plan_destroy(nk_plan_t plan) {
    if (!plan) return NK_ERR_INVALID_ARG;
    Plan* p = (Plan*)plan;
    if (p->exec) cudaGraphExecDestroy(p->exec);
    if (p->graph) cudaGraphDestroy(p->graph);
    if (p->capture_stream) cudaStreamDestroy(p->capture_stream);
    delete p;
    return NK_OK;
}

int nk_stats_combine(const double* parts_host, int n_parts, double* out4_host) {
    if (!parts_host || n_parts < 0 || !out4_host) return NK_ERR_INVALID_ARG;
    // Chan et al. pairwise update of (mean, M2) in the order given: the statistics of the union of the shards
    double n_tot = 0.0, mr = 0.0, mi = 0.0, m2 = 0.0;
    for (int k = 0; k < n_parts; ++k) {
        const double pr = parts_host[4 * k], pi = parts_host[4 * k + 1], pv = parts_host[4 * k + 2],
                     n = parts_host[4 * k + 3];
        if (!(n >= 0.0)) return NK_ERR_INVALID_ARG;
        if (n == 0.0) continue;
        const double dr = pr - mr, di = pi - mi, new_n = n_tot + n;
        m2 += pv * n + (dr * dr + di * di) * n_tot * n / new_n;
        mr += dr * n / new_n;
        mi += di * n / new_n;
        n_tot = new_n;
    }
    out4_host[0] = mr; out4_host[1] = mi; out4_host[2] = n_tot > 0.0 ? m2 / n_tot : 0.0; out4_host[3] = n_tot;
    return NK_OK;
}

int nk_local_energy_form(nk_operator_t h, int64_t B, int N, int M, int dtype, int64_t chunk_size, const void* workspace,
                         size_t workspace_bytes, nk_stream_t stream, int* form_host, float* tau_max_host,
                         int* series_terms_host) {
    if (!h || bad_dims(B, N, M, dtype) || chunk_size < 0 || !form_host) return NK_ERR_INVALID_ARG;
    const Operator* op = (const Operator*)h;
    if (N != op->n_sites) return NK_ERR_INVALID_ARG;
    const Geometry g = make_geometry(op, N, M, dtype);
    if (!g.ok) return NK_ERR_UNSUPPORTED;
    const int64_t chunk = eff_chunk(B, chunk_size);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < carve_eloc(nullptr, g, chunk, dtype, B).bytes)
        return NK_ERR_WORKSPACE;
    const ElocWs w = carve_eloc(const_cast<void*>(workspace), g, chunk, dtype, B);
    float tau = 0.f;
    unsigned K = 0;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == NK_F32) {                              // complex parameters never pack the product table
        NK_CUDA(cudaMemcpyAsync(&tau, w.taumax, sizeof(float), cudaMemcpyDeviceToHost, st));
        if (w.has_series) NK_CUDA(cudaMemcpyAsync(&K, w.ser.ctl, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
        NK_CUDA(cudaStreamSynchronize(st));
    }
    *form_host = K > 0 ? (int)NK_FORM_SERIES
                       : (dtype == NK_F32 && tau <= NK_FORM_TAU_MAX) ? (int)NK_FORM_PRODUCT : (int)NK_FORM_LOGCOSH;
    if (tau_max_host) *tau_max_host = tau;
    if (series_terms_host) *series_terms_host = (int)K;
    return NK_OK;
}

// ---- host-buffer entry point ---------------------------------------------------------------------------
namespace {
struct HostScratch {
    int8_t* sigma;
    void *W, *a, *b, *eloc, *logpsi, *ws;
    double* stats;
    size_t ws_bytes, bytes;
};
HostScratch carve_host(void* scratch, nk_operator_t h, int64_t B, int N, int M, int dtype, int64_t chunk_size) {
    const size_t esz = dtype == NK_C64 ? 8 : 4;
    Carver c(scratch);
    HostScratch s;
    s.sigma = c.take<int8_t>((size_t)B * N);
    s.W = c.take<uint8_t>((size_t)M * N * esz);
    s.a = c.take<uint8_t>((size_t)N * esz);
    s.b = c.take<uint8_t>((size_t)M * esz);
    s.eloc = c.take<uint8_t>((size_t)B * esz);
    s.logpsi = c.take<uint8_t>((size_t)B * esz);
    s.stats = c.take<double>(4);
    s.ws_bytes = nk_local_energy_workspace_bytes(h, B, N, M, dtype, chunk_size);
    s.ws = c.take<uint8_t>(s.ws_bytes);
    s.bytes = c.off;
    return s;
}
}  // namespace

size_t nk_local_energy_host_scratch_bytes(nk_operator_t h, int64_t B, int N, int M, int dtype, int64_t chunk_size) {
    if (!h || bad_dims(B, N, M, dtype) || chunk_size < 0) return 0;
    return carve_host(nullptr, h, B, N, M, dtype, chunk_size).bytes;
}

int nk_local_energy_host(nk_operator_t h, const int8_t* sigma_host, int64_t B, int N, int M, int dtype,
                         const void* W_host, const void* a_host, const void* b_host, int64_t chunk_size,
                         void* eloc_host, void* logpsi_host, double* stats_host, void* scratch, size_t scratch_bytes,
                         nk_stream_t stream) {
    if (!h || bad_dims(B, N, M, dtype) || chunk_size < 0 || !W_host || (B > 0 && (!sigma_host || !eloc_host)))
        return NK_ERR_INVALID_ARG;
    if (!scratch || ((uintptr_t)scratch & 255)) return NK_ERR_WORKSPACE;
    const HostScratch s = carve_host(scratch, h, B, N, M, dtype, chunk_size);
    if (scratch_bytes < s.bytes) return NK_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t esz = dtype == NK_C64 ? 8 : 4;
    // Copies run on an internal stream so that sigma of chunk k + 1 travels while chunk k is computed: parameters
    // first (the packing kernels need them), then sigma chunk by chunk, one event each.
    if (tl_copy_stream == nullptr) NK_CUDA(cudaStreamCreateWithFlags(&tl_copy_stream, cudaStreamNonBlocking));
    const int64_t chunk = (chunk_size <= 0 || chunk_size > B) ? (B > 0 ? B : 1) : chunk_size;
    const size_t n_chunks = B > 0 ? (size_t)((B + chunk - 1) / chunk) : 0;
    while (tl_copy_events.size() < n_chunks + 2) {
        cudaEvent_t ev;
        NK_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        tl_copy_events.push_back(ev);
    }
    cudaStream_t cs = tl_copy_stream;
    const cudaEvent_t ev_start = tl_copy_events[n_chunks], ev_params = tl_copy_events[n_chunks + 1];
    NK_CUDA(cudaEventRecord(ev_start, st));                 // earlier work on the caller's stream may still use scratch
    NK_CUDA(cudaStreamWaitEvent(cs, ev_start, 0));
    NK_CUDA(cudaMemcpyAsync(s.W, W_host, (size_t)M * N * esz, cudaMemcpyHostToDevice, cs));
    if (a_host) NK_CUDA(cudaMemcpyAsync(s.a, a_host, (size_t)N * esz, cudaMemcpyHostToDevice, cs));
    if (b_host) NK_CUDA(cudaMemcpyAsync(s.b, b_host, (size_t)M * esz, cudaMemcpyHostToDevice, cs));
    NK_CUDA(cudaEventRecord(ev_params, cs));
    for (size_t k = 0; k < n_chunks; ++k) {
        const int64_t s0 = (int64_t)k * chunk, nb = (B - s0 < chunk) ? (B - s0) : chunk;
        NK_CUDA(cudaMemcpyAsync(s.sigma + s0 * N, sigma_host + s0 * N, (size_t)nb * N, cudaMemcpyHostToDevice, cs));
        NK_CUDA(cudaEventRecord(tl_copy_events[k], cs));
    }
    NK_CUDA(cudaStreamWaitEvent(st, ev_params, 0));
    tl_chunk_ready = &tl_copy_events;
    const int rc = nk_local_energy(h, s.sigma, B, N, M, dtype, s.W, a_host ? s.a : nullptr, b_host ? s.b : nullptr,
                                   chunk_size, s.eloc, logpsi_host ? s.logpsi : nullptr, stats_host ? s.stats : nullptr,
                                   s.ws, s.ws_bytes, stream);
    tl_chunk_ready = nullptr;
    if (rc != NK_OK) return rc;
    if (B > 0) NK_CUDA(cudaMemcpyAsync(eloc_host, s.eloc, (size_t)B * esz, cudaMemcpyDeviceToHost, st));
    if (B > 0 && logpsi_host) NK_CUDA(cudaMemcpyAsync(logpsi_host, s.logpsi, (size_t)B * esz, cudaMemcpyDeviceToHost, st));
    if (stats_host) NK_CUDA(cudaMemcpyAsync(stats_host, s.stats, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));
    return NK_OK;
}

}  // extern "C"
