/*
 * afsat_oracle.c -- CPU ORACLE for the AFSAT hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct implementation of what the CUDA path computes, written from
 * the paper's definitions (arxiv/paper_2606_06641, /root/reference/PAPER.md) and the readings
 * listed in DESIGN.md.  It shares NO code with the CUDA library (no headers, helpers, tables or
 * constant generators) and the product path never calls it: only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 *
 * What it computes (all floating point in x87 `long double`, 64-bit significand):
 *   O2  truth table g(tau) of a symmetric constraint on the count tau of true literals,
 *       -1 = satisfied, +1 = violated               (Table 1 :87-97, Table 2 :252-262,
 *                                                    convention True -> -1)
 *   O3  exact integer Fourier coefficients A_j = 2^k * f^(S), |S| = j, grouped by |S|
 *       (symmetric constraint => f^ depends on |S| only):
 *           A_j = sum_tau g(tau) * K_tau(j),  K_tau(j) = sum_a (-1)^a C(j,a) C(k-j,tau-a)
 *       which is f^(S) = 2^-k sum_z f(z) prod_{i in S} z_i with the corners z grouped by the
 *       number tau of -1 entries and the number a of those that fall inside S.  Division by 2^k
 *       is deferred to the very end.
 *   O5  elementary symmetric polynomials e_0..e_k of the literal values by the textbook DP
 *       (the terms of Eq. (1) sharing a coefficient are the ESPs).
 *   O6  FE_C = (sum_j A_j e_j) / 2^k                         -- Eq. (1)
 *   O7  dFE_C/dy_i = (sum_{j>=1} A_j e_{j-1}(y without i)) / 2^k, a fresh DP per literal
 *       (multilinearity of Eq. (1)); scatter with the literal sign; zero rows for fixed
 *       variables (gradient masking).
 *   O8  F[b] = sum_C FE_C                                     -- Eq. (2)
 *   O9  x <- min(1, max(-1, x - eta * G))                      -- Alg. 1
 *   O10 T_v = (x_v < 0); tau = #true literals; integer satisfied count; first solved step;
 *       solved candidates are frozen (Alg. 1 :124-127).
 *   O11 Alg. 1 with its line search (method not given by the paper: DESIGN.md
 *       reading B5 = per-candidate backtracking, Armijo rule along the projection arc): oracle_step_ls.
 *   O12 random re-initialisation for restarts: oracle_restart, the counter-based
 *       generator the C ABI header documents, restated here (the one thing both sides must share by value).
 * No DFT, no prefix/suffix products, no blocking, no reordering.
 *
 * Pins (tests/test_oracle_pins.py, `-m "not gpu"`): brute force of Eq. (1) over all 2^k subsets
 * (k <= 10), FE = g(tau) exactly at every corner, closed forms for OR / XOR / NAE, the
 * Poisson-binomial expectation identity for any k <= 64, the exact affine-gradient identity and
 * central finite differences, Parseval, the mean coefficient, the dualities between constraint
 * types, monotone-gradient closed forms, an independent integer recount for the discrete check,
 * and the worked k=3 values of tests/golden/worked_k3.txt.
 * Parity unpinned by the PAPER (pinned only by DESIGN.md readings): the step size eta, the
 * rounding of x = 0 (reading A9: True iff x < 0), "no-op" semantics of frozen candidates (A12), and
 * the whole of oracle_step_ls (the paper names neither the line-search method nor its constants;
 * its pins check the textbook properties of the rule in reading B5, not the paper).
 *
 * Layout: X, G are variable-major, candidate-minor: x[v*ldb + b].  All arrays are caller-owned.
 * Every function returns 0 on success, a negative number on invalid input.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_KMAX 64
typedef long double real;
typedef __int128 wide;

enum { T_OR = 0, T_XOR = 1, T_ATLEAST = 2, T_ATMOST = 3, T_EXACTLY = 4, T_NAE = 5 };

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* O2: is a constraint of this type satisfied when tau of its k literals are true? */
static int satisfied(int type, int k, int param, int tau)
{
    switch (type) {
    case T_OR:      return tau >= 1;                    /* sum >= 1  */
    case T_XOR:     return (tau & 1) == (param & 1);    /* parity; 1 = odd  */
    case T_ATLEAST: return tau >= param;                /* CARD >= t  */
    case T_ATMOST:  return tau <= param;                /* CARD < t+1 */
    case T_EXACTLY: return tau == param;                /* EK  */
    case T_NAE:     return tau > 0 && tau < k;          /* not all equal  */
    default:        return -1;
    }
}

int oracle_truth_table(int type, int k, int param, int8_t *g /* [k+1] */)
{
    if (k < 1 || k > ORACLE_KMAX || type < 0 || type > T_NAE) return -1;
    for (int tau = 0; tau <= k; ++tau) g[tau] = satisfied(type, k, param, tau) ? -1 : +1;
    return 0;
}

static wide binom(int n, int r)
{
    if (r < 0 || r > n) return 0;
    wide c = 1;
    for (int i = 1; i <= r; ++i) c = c * (n - r + i) / i;   /* exact at every step */
    return c;
}

/* O3: A_j, j = 0..k, exact integers with |A_j| <= 2^k. */
static int coeffs_wide(int type, int k, int param, wide *A)
{
    int8_t g[ORACLE_KMAX + 1];
    if (oracle_truth_table(type, k, param, g)) return -1;
    for (int j = 0; j <= k; ++j) {
        wide acc = 0;
        for (int tau = 0; tau <= k; ++tau) {
            wide K = 0;                                   /* Krawtchouk K_tau(j) */
            for (int a = 0; a <= j && a <= tau; ++a) {
                wide term = binom(j, a) * binom(k - j, tau - a);
                K += (a & 1) ? -term : term;
            }
            acc += (wide)g[tau] * K;
        }
        A[j] = acc;
    }
    return 0;
}

/* Exported for the pins: exact coefficients as int64 (k <= 62 so that 2^k fits). */
int oracle_coeffs(int type, int k, int param, int64_t *A /* [k+1] */)
{
    wide W[ORACLE_KMAX + 1];
    if (k > 62) return -2;
    if (coeffs_wide(type, k, param, W)) return -1;
    for (int j = 0; j <= k; ++j) A[j] = (int64_t)W[j];
    return 0;
}

/* O5: e_0..e_k of y[0..k-1], skipping index `skip` (skip < 0: none). Returns the degree. */
static int esp(const real *y, int k, int skip, real *e)
{
    int d = 0;
    e[0] = 1.0L;
    for (int i = 0; i < k; ++i) {
        if (i == skip) continue;
        e[d + 1] = 0.0L;
        for (int j = d + 1; j >= 1; --j) e[j] += y[i] * e[j - 1];
        ++d;
    }
    return d;
}

/* O6 + O7 for one constraint on literal values y. A = real-valued copies of the integers. */
static void fe_one(const real *A, int k, const real *y, real *fe, real *dfe /* [k] or NULL */)
{
    real e[ORACLE_KMAX + 1];
    esp(y, k, -1, e);
    real s = 0.0L;
    for (int j = 0; j <= k; ++j) s += A[j] * e[j];
    *fe = ldexpl(s, -k);                                 /* the single deferred division */
    if (!dfe) return;
    for (int i = 0; i < k; ++i) {
        esp(y, k, i, e);                                 /* ESPs of the other k-1 literals */
        real d = 0.0L;
        for (int j = 1; j <= k; ++j) d += A[j] * e[j - 1];
        dfe[i] = ldexpl(d, -k);
    }
}

/* Single constraint, literal values given directly (used by the pins). */
int oracle_fe_single(int type, int k, int param, const double *y, double *fe, double *dfe)
{
    wide W[ORACLE_KMAX + 1];
    real A[ORACLE_KMAX + 1], yy[ORACLE_KMAX] = {0}, f, d[ORACLE_KMAX];
    if (coeffs_wide(type, k, param, W)) return -1;
    for (int j = 0; j <= k; ++j) A[j] = (real)W[j];
    for (int i = 0; i < k; ++i) yy[i] = (real)y[i];
    fe_one(A, k, yy, &f, dfe ? d : NULL);
    *fe = (double)f;
    if (dfe) for (int i = 0; i < k; ++i) dfe[i] = (double)d[i];
    return 0;
}

/* ---- instance-level entry points ------------------------------------------------------- */

typedef struct {
    int32_t n, m;
    const int64_t *row_ptr;
    const int32_t *lit_var;
    const int8_t *lit_sign;
    const uint8_t *type;
    const int32_t *param;
    const int8_t *fixed;
    real *A;          /* coefficients, constraint c at offset row_ptr[c] + c, length k+1 */
} inst_t;

static int inst_init(inst_t *I, int32_t n, int32_t m, const int64_t *row_ptr,
                     const int32_t *lit_var, const int8_t *lit_sign, const uint8_t *type,
                     const int32_t *param, const int8_t *fixed, int want_coeffs)
{
    memset(I, 0, sizeof *I);
    if (n < 1 || m < 0 || row_ptr[0] != 0) return -1;
    for (int32_t c = 0; c < m; ++c) {
        int64_t k = row_ptr[c + 1] - row_ptr[c];
        if (k < 1 || k > ORACLE_KMAX || type[c] > T_NAE) return -1;
        for (int64_t p = row_ptr[c]; p < row_ptr[c + 1]; ++p) {
            if (lit_var[p] < 0 || lit_var[p] >= n) return -1;
            if (lit_sign[p] != 1 && lit_sign[p] != -1) return -1;
            for (int64_t q = row_ptr[c]; q < p; ++q)
                if (lit_var[q] == lit_var[p]) return -1;   /* FE is multilinear: distinct vars */
        }
    }
    I->n = n; I->m = m; I->row_ptr = row_ptr; I->lit_var = lit_var; I->lit_sign = lit_sign;
    I->type = type; I->param = param; I->fixed = fixed;
    if (want_coeffs) {
        I->A = (real *)malloc(sizeof(real) * (size_t)(row_ptr[m] + m + 1));
        if (!I->A) return -3;
        for (int32_t c = 0; c < m; ++c) {
            wide W[ORACLE_KMAX + 1];
            int k = (int)(row_ptr[c + 1] - row_ptr[c]);
            coeffs_wide(type[c], k, param[c], W);
            real *A = I->A + row_ptr[c] + c;
            for (int j = 0; j <= k; ++j) A[j] = (real)W[j];
        }
    }
    return 0;
}

static void inst_free(inst_t *I) { free(I->A); I->A = NULL; }

/* value of variable v for this candidate: fixed variables use their fixed value */
static inline double var_value(const inst_t *I, const double *xcol_base, int64_t ldb, int32_t v)
{
    if (I->fixed && I->fixed[v] != 0) return (double)I->fixed[v];
    return xcol_base[(int64_t)v * ldb];
}

/* O4-O8 for one candidate (column pointer x = X + b). g: [n] long double accumulators. */
static real eval_candidate(const inst_t *I, const double *x, int64_t ldb, real *g)
{
    real F = 0.0L;
    if (g) for (int32_t v = 0; v < I->n; ++v) g[v] = 0.0L;
    for (int32_t c = 0; c < I->m; ++c) {
        int64_t lo = I->row_ptr[c];
        int k = (int)(I->row_ptr[c + 1] - lo);
        real y[ORACLE_KMAX], d[ORACLE_KMAX], fe;
        for (int i = 0; i < k; ++i)
            y[i] = (real)I->lit_sign[lo + i] * (real)var_value(I, x, ldb, I->lit_var[lo + i]);
        fe_one(I->A + lo + c, k, y, &fe, g ? d : NULL);
        F += fe;
        if (g) for (int i = 0; i < k; ++i) g[I->lit_var[lo + i]] += (real)I->lit_sign[lo + i] * d[i];
    }
    if (g && I->fixed) for (int32_t v = 0; v < I->n; ++v) if (I->fixed[v] != 0) g[v] = 0.0L;
    return F;
}

/* O10 for one candidate. */
static int32_t check_candidate(const inst_t *I, const double *x, int64_t ldb)
{
    int32_t sat = 0;
    for (int32_t c = 0; c < I->m; ++c) {
        int64_t lo = I->row_ptr[c];
        int k = (int)(I->row_ptr[c + 1] - lo), tau = 0;
        for (int i = 0; i < k; ++i) {
            int var_true = var_value(I, x, ldb, I->lit_var[lo + i]) < 0.0;  /* True iff x < 0 */
            int lit_true = (I->lit_sign[lo + i] > 0) ? var_true : !var_true;
            tau += lit_true;
        }
        sat += satisfied(I->type[c], k, I->param[c], tau) ? 1 : 0;
    }
    return sat;
}

int oracle_eval_grad(int32_t n, int32_t m, const int64_t *row_ptr, const int32_t *lit_var,
                     const int8_t *lit_sign, const uint8_t *type, const int32_t *param,
                     const int8_t *fixed, int32_t B, int64_t ldb, const double *X,
                     double *F /* [B] */, double *G /* [n][ldb] or NULL */)
{
    inst_t I;
    int rc = inst_init(&I, n, m, row_ptr, lit_var, lit_sign, type, param, fixed, 1);
    if (rc) return rc;
    if (B < 0 || ldb < B) { inst_free(&I); return -1; }
#pragma omp parallel
    {
        real *g = G ? (real *)malloc(sizeof(real) * (size_t)n) : NULL;
#pragma omp for schedule(dynamic, 1)
        for (int32_t b = 0; b < B; ++b) {
            real f = eval_candidate(&I, X + b, ldb, g);
            if (F) F[b] = (double)f;
            if (G) for (int32_t v = 0; v < n; ++v) G[(int64_t)v * ldb + b] = (double)g[v];
        }
        free(g);
    }
    inst_free(&I);
    return 0;
}

int oracle_check(int32_t n, int32_t m, const int64_t *row_ptr, const int32_t *lit_var,
                 const int8_t *lit_sign, const uint8_t *type, const int32_t *param,
                 const int8_t *fixed, int32_t B, int64_t ldb, const double *X,
                 int32_t *sat_count /* [B] */, uint8_t *is_solution /* [B] */)
{
    inst_t I;
    int rc = inst_init(&I, n, m, row_ptr, lit_var, lit_sign, type, param, fixed, 0);
    if (rc) return rc;
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t b = 0; b < B; ++b) {
        int32_t s = check_candidate(&I, X + b, ldb);
        sat_count[b] = s;
        is_solution[b] = (uint8_t)(s == m);
    }
    return 0;
}

/*
 * Alg. 1 with a fixed step eta (reading A10), n_steps iterations:
 *   gradient at X(t-1) -> X(t) = clamp(X(t-1) - eta*G) on free variables -> round -> count on
 *   X(t) -> if all m satisfied: is_solution = 1, first_step = step_base + t, candidate frozen.
 * X(0) is not checked (reading A11).  If resume != 0, is_solution / first_step are read as the
 * state left by an earlier call (frozen candidates stay frozen); otherwise they are reset.
 * On return sat_count / F describe the final X of every candidate.
 */
int oracle_step(int32_t n, int32_t m, const int64_t *row_ptr, const int32_t *lit_var,
                const int8_t *lit_sign, const uint8_t *type, const int32_t *param,
                const int8_t *fixed, int32_t B, int64_t ldb, double *X /* in/out */,
                double eta, int32_t n_steps, int32_t step_base, int32_t resume,
                double *F /* [B] or NULL */, int32_t *sat_count, uint8_t *is_solution,
                int32_t *first_step)
{
    inst_t I;
    int rc = inst_init(&I, n, m, row_ptr, lit_var, lit_sign, type, param, fixed, 1);
    if (rc) return rc;
#pragma omp parallel
    {
        real *g = (real *)malloc(sizeof(real) * (size_t)n);
#pragma omp for schedule(dynamic, 1)
        for (int32_t b = 0; b < B; ++b) {
            double *x = X + b;
            int solved = resume ? (is_solution[b] != 0) : 0;
            int32_t first = resume ? first_step[b] : -1;
            for (int32_t t = 1; t <= n_steps && !solved; ++t) {
                eval_candidate(&I, x, ldb, g);
                for (int32_t v = 0; v < n; ++v) {
                    if (fixed && fixed[v] != 0) continue;
                    real nx = (real)x[(int64_t)v * ldb] - (real)eta * g[v];
                    if (nx > 1.0L) nx = 1.0L;
                    if (nx < -1.0L) nx = -1.0L;
                    x[(int64_t)v * ldb] = (double)nx;
                }
                if (check_candidate(&I, x, ldb) == m) { solved = 1; first = step_base + t; }
            }
            int32_t s = check_candidate(&I, x, ldb);
            sat_count[b] = s;
            is_solution[b] = (uint8_t)solved;
            first_step[b] = first;
            if (F) F[b] = (double)eval_candidate(&I, x, ldb, NULL);
        }
        free(g);
    }
    inst_free(&I);
    return 0;
}

/*
 * O11 -- Alg. 1 WITH line search and convergence test ("eta <- lineSearch(FE, grad FE, s)",
 * :120-122 step and projection, :125 "if eta < delta").  Reading B5 (the paper gives no method):
 * per candidate, backtracking with the Armijo rule along the projection arc,
 *     eta = s_max;  repeat at most max_trials times:
 *         X' = clamp(X - eta G) on free variables;  D = <G, X - X'>;
 *         if F(X') <= F(X) - c1 D: accept;  else eta <- beta eta;  if eta < delta: converged.
 * An accepted candidate moves to X'; a converged one keeps X and is frozen (like a solved one);
 * one that exhausts max_trials keeps X for this step.  margin[b] (may be NULL) = the smallest
 * |F(X') - (F(X) - c1 D)| met in the LAST iteration: how close the accept/reject decisions were
 * to a tie (the parity tests compare decisions only where it exceeds the kernel's rounding).
 */
int oracle_step_ls(int32_t n, int32_t m, const int64_t *row_ptr, const int32_t *lit_var,
                   const int8_t *lit_sign, const uint8_t *type, const int32_t *param,
                   const int8_t *fixed, int32_t B, int64_t ldb, double *X /* in/out */,
                   double s_max, double beta, double c1, double delta, int32_t max_trials,
                   int32_t n_steps, int32_t step_base, int32_t resume,
                   double *F /* [B] or NULL */, double *eta_out /* [B] or NULL */, int32_t *sat_count,
                   uint8_t *is_solution, int32_t *first_step, uint8_t *converged,
                   double *margin /* [B] or NULL */)
{
    inst_t I;
    int rc = inst_init(&I, n, m, row_ptr, lit_var, lit_sign, type, param, fixed, 1);
    if (rc) return rc;
    if (!(s_max > 0) || !(beta > 0 && beta < 1) || !(c1 >= 0 && c1 < 1) || !(delta >= 0) || max_trials < 1) {
        inst_free(&I);
        return -1;
    }
#pragma omp parallel
    {
        real *g = (real *)malloc(sizeof(real) * (size_t)n);
        double *xt = (double *)malloc(sizeof(double) * (size_t)n);   /* trial point, one column, stride 1 */
        double *x0 = (double *)malloc(sizeof(double) * (size_t)n);
#pragma omp for schedule(dynamic, 1)
        for (int32_t b = 0; b < B; ++b) {
            double *x = X + b;
            int solved = resume ? (is_solution[b] != 0) : 0;
            int conv = resume ? (converged[b] != 0) : 0;
            int32_t first = resume ? first_step[b] : -1;
            real eta = (real)s_max, mg = INFINITY;
            for (int32_t t = 1; t <= n_steps && !solved && !conv; ++t) {
                real F0 = eval_candidate(&I, x, ldb, g);
                int accepted = 0;
                eta = (real)s_max; mg = INFINITY;
                for (int32_t v = 0; v < n; ++v) x0[v] = x[(int64_t)v * ldb];
                for (int32_t j = 0; j < max_trials && !accepted && !conv; ++j) {
                    real D = 0.0L;
                    for (int32_t v = 0; v < n; ++v) {
                        real nx = (real)x0[v];
                        if (!(fixed && fixed[v] != 0)) {
                            nx = (real)x0[v] - eta * g[v];
                            if (nx > 1.0L) nx = 1.0L;
                            if (nx < -1.0L) nx = -1.0L;
                            D += g[v] * ((real)x0[v] - nx);
                        }
                        xt[v] = (double)nx;
                    }
                    real F1 = eval_candidate(&I, xt, 1, NULL);
                    real gap = fabsl(F1 - (F0 - (real)c1 * D));
                    if (gap < mg) mg = gap;
                    if (F1 <= F0 - (real)c1 * D) accepted = 1;
                    else { eta *= (real)beta; if (eta < (real)delta) conv = 1; }
                }
                if (accepted) for (int32_t v = 0; v < n; ++v) x[(int64_t)v * ldb] = xt[v];
                if (check_candidate(&I, x, ldb) == m) { solved = 1; first = step_base + t; }
            }
            sat_count[b] = check_candidate(&I, x, ldb);
            is_solution[b] = (uint8_t)solved;
            converged[b] = (uint8_t)conv;
            first_step[b] = first;
            if (eta_out) eta_out[b] = (double)eta;
            if (margin) margin[b] = (double)mg;
            if (F) F[b] = (double)eval_candidate(&I, x, ldb, NULL);
        }
        free(g); free(xt); free(x0);
    }
    inst_free(&I);
    return 0;
}

/*
 * O12 -- restart initialisation ("executed repeatedly with different random initialisations";
 * :105-107 fixed variables keep their value in every candidate).  The generator is the one the C ABI
 * documents (a method-level random draw must be the same numbers on both sides): for candidate b,
 * variable v, 64-bit seed (lo, hi) and round r, all arithmetic mod 2^32,
 *     h1 = fmix(lo ^ b*0x9E3779B9);  h2 = fmix((h1 + v*0x85EBCA6B) ^ hi);  h = fmix(h2 + r*0xC2B2AE35);
 *     x = (h >> 8) * 2^-23 - 1  in [-1, 1)
 * with fmix the 32-bit avalanche  h ^= h>>16; h *= 0x85EBCA6B; h ^= h>>13; h *= 0xC2B2AE35; h ^= h>>16.
 * Candidates with keep[b] != 0 are left untouched.
 */
static uint32_t avalanche32(uint32_t h)
{
    h ^= h >> 16; h *= 0x85EBCA6BU; h ^= h >> 13; h *= 0xC2B2AE35U; h ^= h >> 16;
    return h;
}

int oracle_restart(int32_t n, const int8_t *fixed, int32_t B, int64_t ldb, double *X,
                   const uint8_t *keep, uint64_t seed, uint32_t round)
{
    if (n < 1 || B < 0 || ldb < B) return -1;
    const uint32_t lo = (uint32_t)(seed & 0xFFFFFFFFULL), hi = (uint32_t)(seed >> 32);
    for (int32_t b = 0; b < B; ++b) {
        if (keep && keep[b]) continue;
        for (int32_t v = 0; v < n; ++v) {
            double val;
            if (fixed && fixed[v] != 0) val = (double)fixed[v];
            else {
                uint32_t h1 = avalanche32(lo ^ ((uint32_t)b * 0x9E3779B9U));
                uint32_t h2 = avalanche32((h1 + (uint32_t)v * 0x85EBCA6BU) ^ hi);
                uint32_t h = avalanche32(h2 + round * 0xC2B2AE35U);
                val = (double)(h >> 8) / 8388608.0 - 1.0;
            }
            X[(int64_t)v * ldb + b] = val;
        }
    }
    return 0;
}
