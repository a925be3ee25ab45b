/* ORACLE, second route — test infrastructure, NOT the product.
 *
 * Float64 INCREMENTAL local energy of the RBM (last paragraph): the same
 * estimator as oracle/nk_oracle.py `local_energy`, Eq. (12)
 *     E_loc(s) = sum_s' <s|H|s'> psi(s') / psi(s),
 * but ln psi(s') is NOT recomputed from scratch: with theta = W s + b (Eq. (7); RBM L575, ln cosh Eq. (41)
 * L1292) a flipped site k changes theta to theta' = theta - 2 s_k W[:,k] and an exchange of antiparallel spins
 * (i, j) to theta' = theta - 2 s_i (W[:,i] - W[:,j]), so
 *     ln psi(s') - ln psi(s) = -2 s_k a_k [- 2 s_i (a_i - a_j)] + sum_j [ lc(theta'_j) - lc(theta_j) ],
 * lc(z) = ln cosh z evaluated stably (Q11: z <- z sign(Re z); lc = z + log1p(exp(-2z)) - ln 2).
 * Matrix elements: Heisenberg Eq. (50) L1556 (diagonal J s_i s_j, exchange 2J, -2J with the Marshall flag),
 * Ising Eq. (54) L1881 (diagonal J s_i s_j, flip -h).  Statistics: Eq. (17) L675 stays in nk_oracle.stats.
 *
 * Written separately from oracle/nk_oracle.py (which materialises every s' and calls a matmul per sample) and from
 * paper_2112_10526_b200/csrc (no shared code, headers, tables or helpers).  Pinned in tests/test_oracle_incremental.py
 * against the from-scratch oracle to 1e-12 relative on configs 1-4 and a fixed 256-sample subset of config 5; its
 * job is (i) to cover ALL samples of config 5 in the GPU parity tests, (ii) to be the fair "plain CPU" baseline
 * beside the from-scratch one in bench.py.  Plain loops, double precision; POSIX threads over samples only (a shared atomic
 * counter hands out blocks of 4 samples; this image's gcc has no usable OpenMP runtime).
 *
 * Build (oracle/nk_incremental.py does it on demand): gcc -O2 -pthread -shared -fPIC nk_incremental.c -lm
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <pthread.h>
#include <unistd.h>

#define NK_INC_HEISENBERG 0
#define NK_INC_ISING 1
#define NK_INC_FLAG_MARSHALL 1u

static const double LN2 = 0.69314718055994530942;

static double lc_real(double x) {
    const double t = fabs(x);
    return t + log1p(exp(-2.0 * t)) - LN2;
}
static double complex lc_cplx(double complex z) {
    if (creal(z) < 0.0) z = -z;
    const double complex w = cexp(-2.0 * z);           /* |w| <= 1 */
    /* principal log1p(w) = ln|1 + w| + i arg(1 + w); Re(1 + w) >= 0 */
    const double re = 0.5 * log1p(creal(w) * (2.0 + creal(w)) + cimag(w) * cimag(w));
    const double im = atan2(cimag(w), 1.0 + creal(w));
    return z + (re + im * I) - LN2;
}

/* ---- threading: n_threads workers pull blocks of 4 samples from a shared counter ------------------------------ */
typedef struct {
    int kind, N, M, n_bonds;
    int64_t B;
    const int8_t* sigma;
    const int32_t *bonds, *colors;
    const double* J;
    double h;
    unsigned flags;
    const void* Wt;                 /* [N][M] column-major copy of W: double or double complex */
    const double *a, *b;
    double *eloc_out, *logpsi_out;
    int64_t next;                   /* shared block counter */
    int fail;
} job_t;

static int64_t take_block(job_t* jb) { return __atomic_fetch_add(&jb->next, 4, __ATOMIC_RELAXED); }

static int default_threads(void) {
    long n = sysconf(_SC_NPROCESSORS_ONLN);
    return n < 1 ? 1 : (n > 256 ? 256 : (int)n);
}
int nk_inc_num_threads(void) { return default_threads(); }

static int run_threads(void* (*fn)(void*), job_t* jb) {
    const int nt = default_threads();
    pthread_t th[256];
    int started = 0;
    for (int t = 0; t < nt - 1; ++t) {
        if (pthread_create(&th[started], NULL, fn, jb) != 0) break;
        ++started;
    }
    fn(jb);                                          /* the calling thread works too */
    for (int t = 0; t < started; ++t) pthread_join(th[t], NULL);
    return jb->fail ? -1 : 0;
}

/* one sample, real parameters */
static void one_sample_real(const job_t* jb, int64_t n, double* theta, double* lc0) {
    const int N = jb->N, M = jb->M;
    const double* Wt = (const double*)jb->Wt;
    const double *a = jb->a, *b = jb->b, *J = jb->J;
    const int32_t *bonds = jb->bonds, *colors = jb->colors;
    const int8_t* s = jb->sigma + n * N;
    /* theta = W s + b */
    for (int j = 0; j < M; ++j) theta[j] = b ? b[j] : 0.0;
    for (int k = 0; k < N; ++k) {
        const double sk = (double)s[k];
        const double* col = Wt + (size_t)k * M;
        for (int j = 0; j < M; ++j) theta[j] += sk * col[j];
    }
    double lp = 0.0;
    for (int j = 0; j < M; ++j) { lc0[j] = lc_real(theta[j]); lp += lc0[j]; }
    if (a) for (int k = 0; k < N; ++k) lp += a[k] * (double)s[k];
    if (jb->logpsi_out) jb->logpsi_out[n] = lp;
    /* diagonal: sz_i sz_j term of every bond (both models) */
    double e = 0.0;
    for (int q = 0; q < jb->n_bonds; ++q) {
        const double Jq = J[colors ? colors[q] : 0];
        e += Jq * (double)s[bonds[2 * q]] * (double)s[bonds[2 * q + 1]];
    }
    if (jb->kind == NK_INC_HEISENBERG) {
        for (int q = 0; q < jb->n_bonds; ++q) {
            const int i = bonds[2 * q], jj = bonds[2 * q + 1];
            if (s[i] == s[jj]) continue;                       /* parallel bond: no off-diagonal element */
            const double mel = ((jb->flags & NK_INC_FLAG_MARSHALL) ? -2.0 : 2.0) * J[colors ? colors[q] : 0];
            const double si = (double)s[i];
            const double* ci = Wt + (size_t)i * M;
            const double* cj = Wt + (size_t)jj * M;
            double d = a ? -2.0 * si * (a[i] - a[jj]) : 0.0;
            for (int j = 0; j < M; ++j) d += lc_real(theta[j] - 2.0 * si * (ci[j] - cj[j])) - lc0[j];
            e += mel * exp(d);
        }
    } else {
        for (int k = 0; k < N; ++k) {
            const double sk = (double)s[k];
            const double* ck = Wt + (size_t)k * M;
            double d = a ? -2.0 * sk * a[k] : 0.0;
            for (int j = 0; j < M; ++j) d += lc_real(theta[j] - 2.0 * sk * ck[j]) - lc0[j];
            e += -jb->h * exp(d);
        }
    }
    jb->eloc_out[n] = e;
}

static void* worker_real(void* arg) {
    job_t* jb = (job_t*)arg;
    double* theta = (double*)malloc((size_t)jb->M * sizeof(double));
    double* lc0 = (double*)malloc((size_t)jb->M * sizeof(double));
    if (!theta || !lc0) __atomic_store_n(&jb->fail, 1, __ATOMIC_RELAXED);
    else
        for (int64_t n0 = take_block(jb); n0 < jb->B; n0 = take_block(jb))
            for (int64_t n = n0; n < n0 + 4 && n < jb->B; ++n) one_sample_real(jb, n, theta, lc0);
    free(theta); free(lc0);
    return NULL;
}

/* Real parameters.  W [M][N], a [N] or NULL, b [M] or NULL, all float64 (the caller up-casts the fp32 storage
 * exactly).  sigma [B][N] int8 +-1.  bonds [n_bonds][2], colors [n_bonds] or NULL, J [n_colors].
 * eloc_out [B], logpsi_out [B] or NULL.  Returns 0, or -1 on a bad argument / allocation failure. */
int nk_inc_local_energy_real(int kind, int64_t B, int N, int M, const int8_t* sigma, int n_bonds,
                             const int32_t* bonds, const int32_t* colors, const double* J, double h, unsigned flags,
                             const double* W, const double* a, const double* b, double* eloc_out,
                             double* logpsi_out) {
    if ((kind != NK_INC_HEISENBERG && kind != NK_INC_ISING) || B < 0 || N <= 0 || M <= 0 || !sigma || !W || !eloc_out)
        return -1;
    /* column k of W as a contiguous row: Wt[k][j] = W[j][k] */
    double* Wt = (double*)malloc((size_t)N * M * sizeof(double));
    if (!Wt) return -1;
    for (int j = 0; j < M; ++j)
        for (int k = 0; k < N; ++k) Wt[(size_t)k * M + j] = W[(size_t)j * N + k];
    job_t jb = {kind, N, M, n_bonds, B, sigma, bonds, colors, J, h, flags, Wt, a, b, eloc_out, logpsi_out, 0, 0};
    const int rc = run_threads(worker_real, &jb);
    free(Wt);
    return rc;
}

/* one sample, complex parameters (a, b interleaved (re, im) pairs) */
static void one_sample_cplx(const job_t* jb, int64_t n, double complex* theta, double complex* lc0) {
    const int N = jb->N, M = jb->M;
    const double complex* Wt = (const double complex*)jb->Wt;
    const double *a = jb->a, *b = jb->b, *J = jb->J;
    const int32_t *bonds = jb->bonds, *colors = jb->colors;
    const int8_t* s = jb->sigma + n * N;
    for (int j = 0; j < M; ++j) theta[j] = b ? b[2 * j] + b[2 * j + 1] * I : 0.0;
    for (int k = 0; k < N; ++k) {
        const double sk = (double)s[k];
        const double complex* col = Wt + (size_t)k * M;
        for (int j = 0; j < M; ++j) theta[j] += sk * col[j];
    }
    double complex lp = 0.0;
    for (int j = 0; j < M; ++j) { lc0[j] = lc_cplx(theta[j]); lp += lc0[j]; }
    if (a) for (int k = 0; k < N; ++k) lp += (a[2 * k] + a[2 * k + 1] * I) * (double)s[k];
    if (jb->logpsi_out) { jb->logpsi_out[2 * n] = creal(lp); jb->logpsi_out[2 * n + 1] = cimag(lp); }
    double complex e = 0.0;
    for (int q = 0; q < jb->n_bonds; ++q) {
        const double Jq = J[colors ? colors[q] : 0];
        e += Jq * (double)s[bonds[2 * q]] * (double)s[bonds[2 * q + 1]];
    }
    if (jb->kind == NK_INC_HEISENBERG) {
        for (int q = 0; q < jb->n_bonds; ++q) {
            const int i = bonds[2 * q], jj = bonds[2 * q + 1];
            if (s[i] == s[jj]) continue;
            const double mel = ((jb->flags & NK_INC_FLAG_MARSHALL) ? -2.0 : 2.0) * J[colors ? colors[q] : 0];
            const double si = (double)s[i];
            const double complex* ci = Wt + (size_t)i * M;
            const double complex* cj = Wt + (size_t)jj * M;
            double complex d = 0.0;
            if (a) d = -2.0 * si * ((a[2 * i] - a[2 * jj]) + (a[2 * i + 1] - a[2 * jj + 1]) * I);
            for (int j = 0; j < M; ++j) d += lc_cplx(theta[j] - 2.0 * si * (ci[j] - cj[j])) - lc0[j];
            e += mel * cexp(d);
        }
    } else {
        for (int k = 0; k < N; ++k) {
            const double sk = (double)s[k];
            const double complex* ck = Wt + (size_t)k * M;
            double complex d = 0.0;
            if (a) d = -2.0 * sk * (a[2 * k] + a[2 * k + 1] * I);
            for (int j = 0; j < M; ++j) d += lc_cplx(theta[j] - 2.0 * sk * ck[j]) - lc0[j];
            e += -jb->h * cexp(d);
        }
    }
    jb->eloc_out[2 * n] = creal(e);
    jb->eloc_out[2 * n + 1] = cimag(e);
}

static void* worker_cplx(void* arg) {
    job_t* jb = (job_t*)arg;
    double complex* theta = (double complex*)malloc((size_t)jb->M * sizeof(double complex));
    double complex* lc0 = (double complex*)malloc((size_t)jb->M * sizeof(double complex));
    if (!theta || !lc0) __atomic_store_n(&jb->fail, 1, __ATOMIC_RELAXED);
    else
        for (int64_t n0 = take_block(jb); n0 < jb->B; n0 = take_block(jb))
            for (int64_t n = n0; n < n0 + 4 && n < jb->B; ++n) one_sample_cplx(jb, n, theta, lc0);
    free(theta); free(lc0);
    return NULL;
}

/* Complex parameters: W, a, b as interleaved (re, im) float64 pairs; eloc_out / logpsi_out [B][2]. */
int nk_inc_local_energy_cplx(int kind, int64_t B, int N, int M, const int8_t* sigma, int n_bonds,
                             const int32_t* bonds, const int32_t* colors, const double* J, double h, unsigned flags,
                             const double* W, const double* a, const double* b, double* eloc_out,
                             double* logpsi_out) {
    if ((kind != NK_INC_HEISENBERG && kind != NK_INC_ISING) || B < 0 || N <= 0 || M <= 0 || !sigma || !W || !eloc_out)
        return -1;
    double complex* Wt = (double complex*)malloc((size_t)N * M * sizeof(double complex));
    if (!Wt) return -1;
    for (int j = 0; j < M; ++j)
        for (int k = 0; k < N; ++k)
            Wt[(size_t)k * M + j] = W[2 * ((size_t)j * N + k)] + W[2 * ((size_t)j * N + k) + 1] * I;
    job_t jb = {kind, N, M, n_bonds, B, sigma, bonds, colors, J, h, flags, Wt, a, b, eloc_out, logpsi_out, 0, 0};
    const int rc = run_threads(worker_cplx, &jb);
    free(Wt);
    return rc;
}
