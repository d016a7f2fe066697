/*
 * zmc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU restatement of the hot path of
 * ZMCintegral-v5 (arXiv 1910.01965): the direct Monte-Carlo estimate
 *     f(x) = \int dy g(y; x)                      (Eq. 1)
 * evaluated independently at every point x of a Cartesian parameter grid
 * ("each parameter x_i takes values from a list"; PAPER.md:61
 * "direct Monte Carlo method"; PAPER.md:65 one integration per grid point;
 * PAPER.md:63 result = "multi-dimensional grid" of integral values).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code, header, table
 * or constant generator with the CUDA path (paper_1910_01965_b200/csrc).
 *
 * Where the paper is silent the readings S1-S8 / Q1-Q18 of SURVEY.md 8(c)
 * (restated in DESIGN.md "Readings") are followed, in the paper's order:
 *   for t in range:  decode (S1);  for s: for k: word(q) (S2,S3) -> u (S4) -> y (S5);
 *                    g (S7); store g_s;   then the two-pass estimator (S6).
 * There is no blocking, fusion or reordering beyond that.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors,
 * the S3 stream values, uniform extremes, param_echo decode, const_one,
 * the n=4 worked example, a pure-Python brute-force enumerator, closed forms
 * of every family (5-sigma coverage, z-score moments, stderr scale); the
 * user-integrand hook (zmc_oracle_set_user) against a closed form
 * (tests/test_user_integrand_cpu.py).
 * Unpinned: the paper's printed Table-1 delta_r values --
 * "parity unpinned": RNG/seed unspecified by the paper.
 *
 * Build: gcc -O2 -std=c11 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_MAX_N 16
#define ORACLE_MAX_M 8

enum { MODE_F64 = 0, MODE_F32_MIRROR = 1 };

enum {
    FAM_C1 = 1, FAM_C2 = 2, FAM_C3 = 3, FAM_C4 = 4, FAM_C5 = 5, FAM_P6 = 6,
    FAM_CONST_ONE = 100, FAM_PARAM_ECHO = 101, FAM_LIN_Y = 102, FAM_POLY = 103
};

/* ---- S2: Philox4x32-10 from the definition (Salmon et al., SC'11) ------- */
void zmc_oracle_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {                   /* key bump before every round but the first */
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ---- S3: stream layout.  Word q = s*N + k of point t lives in block q>>2,
 *      lane q&3; counter = (block lo, block hi, t lo, t hi); key = seed. ---- */
uint32_t zmc_oracle_word(uint64_t seed, uint64_t t, uint64_t q)
{
    uint64_t j = q >> 2;
    uint32_t ctr[4] = { (uint32_t)j, (uint32_t)(j >> 32), (uint32_t)t, (uint32_t)(t >> 32) };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t r[4];
    zmc_oracle_philox(ctr, key, r);
    return r[q & 3];
}

/* ---- S4: uniform in the open interval (0,1), exact in the evaluation type -- */
double zmc_oracle_uniform(uint32_t w, int mode)
{
    if (mode == MODE_F64)
        return (2.0 * (double)w + 1.0) * 0x1p-33;          /* 2^32 levels */
    return (2.0 * (double)(w >> 9) + 1.0) * 0x1p-24;       /* 2^23 levels */
}

/* mirror mode: round an input to float (RN) and promote back (S5) */
static double mirror(double v, int mode)
{
    return mode == MODE_F32_MIRROR ? (double)(float)v : v;
}

/* ---- NEXT-3: a user-defined integrand g(y; x) ("users have a full flexibility to define their
 *      own integrands").  The test harness compiles the user's C expression with gcc and hands the function in;
 *      any integrand id >= FAM_USER evaluates it.  Always evaluated in double (mirror mode rounds its inputs). ---- */
#define FAM_USER 1000
typedef double (*zmc_oracle_user_fn)(const double *y, const double *x, const double *c);
static zmc_oracle_user_fn user_g = 0;
static int user_N = 0, user_M = 0, user_nc = 0;
void zmc_oracle_set_user(zmc_oracle_user_fn g, int N, int M, int n_consts)
{
    user_g = g; user_N = N; user_M = M; user_nc = n_consts;
}

/* ---- S7: the integrand families.  y[k] is 0-based, x[i] holds x_{i+1}. ---- */
static double integrand(int id, int N, int M, const double *y, const double *x,
                        const double *consts)
{
    if (id >= FAM_USER) return user_g(y, x, consts);
    switch (id) {
    case FAM_C1:
        return cos(x[0] * y[0]);
    case FAM_C2:
        return sin(x[0] * y[0] + x[1] * y[1]);
    case FAM_C3: {
        double two_pi = 2.0 * 3.141592653589793;
        double phase = two_pi * consts[0];
        for (int k = 0; k < N; ++k) {
            double ck = x[k % 3] * (double)(k + 1);
            phase += ck * y[k];
        }
        return cos(phase);
    }
    case FAM_C4: {
        double a = x[0], acc = 0.0;
        for (int k = 0; k < N; ++k) {
            double wk = (k < 2) ? x[1] : (k < 4) ? x[2] : x[3];
            double d = y[k] - wk;
            acc += a * a * d * d;
        }
        return exp(-acc);
    }
    case FAM_C5: {
        double r2 = y[0] * y[0] + y[1] * y[1] + y[2] * y[2];
        double ph = x[1] * y[0] + x[2] * y[1] + x[3] * y[2];
        return exp(-x[0] * r2) * cos(ph) * (1.0 + x[4] * y[0] * y[1] * y[2]);
    }
    case FAM_P6: {                       /* PAPER.md:75 Eq. (2), :120 Eq. (4) */
        double arg = 0.0;
        for (int k = 0; k < N; ++k) arg += y[k];
        for (int l = 0; l < M; ++l) arg += x[l];
        return sin(arg);
    }
    case FAM_CONST_ONE:
        return 1.0;
    case FAM_PARAM_ECHO:
        return x[(int)consts[0]];
    case FAM_LIN_Y:
        return y[(int)consts[0]];
    case FAM_POLY: {
        double p = 1.0;
        for (int k = 0; k < N; ++k) p *= y[k];
        return p;
    }
    }
    return NAN;
}

/* accepted (N, M, n_consts) per family; mirrors S7, returns 0 ok */
static int check_shape(int id, int N, int M, int n_consts, const double *consts)
{
    if (id >= FAM_USER) return !user_g ? 2 : (N == user_N && M == user_M && n_consts == user_nc) ? 0 : 3;
    switch (id) {
    case FAM_C1: return (N == 1 && M == 1) ? 0 : 3;
    case FAM_C2: return (N == 2 && M == 2) ? 0 : 3;
    case FAM_C3: return (N >= 1 && M == 3 && n_consts == 1) ? 0 : 3;
    case FAM_C4: return (N == 6 && M == 4) ? 0 : 3;
    case FAM_C5: return (N == 3 && M == 5) ? 0 : 3;
    case FAM_P6: return 0;
    case FAM_CONST_ONE: return 0;
    case FAM_PARAM_ECHO:
        return (n_consts == 1 && consts[0] >= 0 && consts[0] < M && consts[0] == floor(consts[0])) ? 0 : 3;
    case FAM_LIN_Y:
        return (n_consts == 1 && consts[0] >= 0 && consts[0] < N && consts[0] == floor(consts[0])) ? 0 : 3;
    case FAM_POLY: return 0;
    }
    return 2;
}

typedef struct {
    int id, N, M, mode, n_consts;
    const double *bounds;
    const double *const *lists;
    const int64_t *counts;
    uint64_t n, seed;
    const double *consts;
} problem;

/* Q18: the same argument checks as the library boundary. 0 = ok. */
static int validate(const problem *p, uint64_t *G_out)
{
    if (!p->bounds || !p->lists || !p->counts) return 1;
    if (p->N < 1 || p->N > ORACLE_MAX_N || p->M < 1 || p->M > ORACLE_MAX_M) return 1;
    if (p->n < 2 || p->n > 0xFFFFFFFFull) return 1;
    if (p->n_consts < 0 || (p->n_consts > 0 && !p->consts)) return 1;
    for (int k = 0; k < p->N; ++k) {
        double a = p->bounds[2 * k], b = p->bounds[2 * k + 1];
        if (!isfinite(a) || !isfinite(b) || !(a < b)) return 1;
    }
    uint64_t G = 1;
    for (int i = 0; i < p->M; ++i) {
        if (p->counts[i] < 1 || !p->lists[i]) return 1;
        for (int64_t j = 0; j < p->counts[i]; ++j)
            if (!isfinite(p->lists[i][j])) return 1;
        if ((uint64_t)p->counts[i] > (1ull << 48) / G) return 4;
        G *= (uint64_t)p->counts[i];
    }
    int rc = check_shape(p->id, p->N, p->M, p->n_consts, p->consts);
    if (rc) return rc;
    *G_out = G;
    return 0;
}

/* One grid point, literally: decode; for s: for k: word -> u -> y; g; store; S6. */
static int one_point(const problem *p, uint64_t t, double *g_store,
                     double *mean_out, double *stderr_out)
{
    double x[ORACLE_MAX_M], y[ORACLE_MAX_N], a[ORACLE_MAX_N], width[ORACLE_MAX_N];
    double cst[8] = {0};

    /* S1: row-major, last parameter fastest */
    uint64_t rest = t;
    for (int i = p->M - 1; i >= 0; --i) {
        uint64_t L = (uint64_t)p->counts[i];
        uint64_t digit = rest % L;
        rest = rest / L;
        x[i] = mirror(p->lists[i][digit], p->mode);
    }
    /* S5: widths in double, then (mirror mode) rounded to float; V = prod width, k ascending */
    double V = 1.0;
    for (int k = 0; k < p->N; ++k) {
        a[k] = mirror(p->bounds[2 * k], p->mode);
        width[k] = mirror(p->bounds[2 * k + 1] - p->bounds[2 * k], p->mode);
        V *= width[k];
    }
    for (int c = 0; c < p->n_consts && c < 8; ++c) cst[c] = mirror(p->consts[c], p->mode);

    for (uint64_t s = 0; s < p->n; ++s) {
        for (int k = 0; k < p->N; ++k) {
            uint64_t q = s * (uint64_t)p->N + (uint64_t)k;
            uint32_t w = zmc_oracle_word(p->seed, t, q);
            double u = zmc_oracle_uniform(w, p->mode);
            y[k] = fma(u, width[k], a[k]);
        }
        g_store[s] = integrand(p->id, p->N, p->M, y, x, cst);
    }
    /* S6: two-pass estimator, sums in long double */
    long double sum = 0.0L;
    for (uint64_t s = 0; s < p->n; ++s) sum += (long double)g_store[s];
    long double gbar = sum / (long double)p->n;
    long double ss = 0.0L;
    for (uint64_t s = 0; s < p->n; ++s) {
        long double d = (long double)g_store[s] - gbar;
        ss += d * d;
    }
    long double var = ss / (long double)(p->n - 1);
    *mean_out = (double)((long double)V * gbar);
    *stderr_out = (double)((long double)V * sqrtl(var / (long double)p->n));
    return 0;
}

static int run(const problem *p, const uint64_t *indices, uint64_t first, uint64_t count,
               double *out_mean, double *out_stderr, int n_threads)
{
    uint64_t G = 0;
    int rc = validate(p, &G);
    if (rc) return rc;
    if (!out_mean || !out_stderr) return 1;
    if (indices) {
        for (uint64_t r = 0; r < count; ++r) if (indices[r] >= G) return 1;
    } else {
        if (first > G || count > G - first) return 1;
    }
    if (n_threads < 1) n_threads = 1;
    int oom = 0;
#pragma omp parallel num_threads(n_threads)
    {
        double *g_store = (double *)malloc(sizeof(double) * (size_t)p->n);
        if (!g_store) {
#pragma omp atomic write
            oom = 1;
        }
#pragma omp for schedule(static)
        for (int64_t r = 0; r < (int64_t)count; ++r) {
            if (g_store) {
                uint64_t t = indices ? indices[r] : first + (uint64_t)r;
                one_point(p, t, g_store, &out_mean[r], &out_stderr[r]);
            }
        }
        free(g_store);
    }
    return oom ? 5 : 0;
}

/* Contiguous flat range [first_index, first_index+count) of the grid. Outputs are doubles. */
int zmc_oracle_scan(int integrand_id, int N, const double *bounds, int M,
                    const double *const *lists, const int64_t *counts,
                    uint64_t n_samples, uint64_t seed, int mode,
                    const double *consts, int n_consts,
                    uint64_t first_index, uint64_t count,
                    double *out_mean, double *out_stderr, int n_threads)
{
    problem p = { integrand_id, N, M, mode, n_consts, bounds, lists, counts, n_samples, seed, consts };
    return run(&p, NULL, first_index, count, out_mean, out_stderr, n_threads);
}

/* Arbitrary subset of flat indices (duplicates allowed). */
int zmc_oracle_points(int integrand_id, int N, const double *bounds, int M,
                      const double *const *lists, const int64_t *counts,
                      uint64_t n_samples, uint64_t seed, int mode,
                      const double *consts, int n_consts,
                      const uint64_t *indices, uint64_t n_indices,
                      double *out_mean, double *out_stderr, int n_threads)
{
    problem p = { integrand_id, N, M, mode, n_consts, bounds, lists, counts, n_samples, seed, consts };
    if (!indices) return 1;
    return run(&p, indices, 0, n_indices, out_mean, out_stderr, n_threads);
}

/* The g values of one point, in sample order (for the brute-force / prefix pins). */
int zmc_oracle_samples(int integrand_id, int N, const double *bounds, int M,
                       const double *const *lists, const int64_t *counts,
                       uint64_t n_samples, uint64_t seed, int mode,
                       const double *consts, int n_consts,
                       uint64_t t, double *out_g)
{
    problem p = { integrand_id, N, M, mode, n_consts, bounds, lists, counts, n_samples, seed, consts };
    uint64_t G = 0;
    int rc = validate(&p, &G);
    if (rc) return rc;
    if (t >= G || !out_g) return 1;
    double m, e;
    return one_point(&p, t, out_g, &m, &e);
}
