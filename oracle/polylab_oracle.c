/*
 * polylab_oracle.c -- plain, slow CPU implementation of Polylab's simplify and
 * product.  TEST INFRASTRUCTURE (see polylab_oracle.h); shares nothing with the
 * CUDA path.  Build: gcc -O2 -ffp-contract=off -fPIC -shared (oracle/oracle.py).
 *
 * Every function cites the passage of /root/reference/PAPER.md it follows.
 */
#include "polylab_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------- exponents */

/* element (t, v) of a row-major unsigned exponent matrix (alpha in N^n) */
static inline uint32_t exp_at(const void* exps, int32_t exp_bytes, int32_t nvars, int64_t t, int32_t v)
{
    const int64_t idx = t * (int64_t)nvars + v;
    switch (exp_bytes) {
    case 1: return ((const uint8_t*)exps)[idx];
    case 2: return ((const uint16_t*)exps)[idx];
    default: return ((const uint32_t*)exps)[idx];
    }
}

/* lexicographic comparison of two rows, variable 0 most significant (reading A1:
 * the order of the transcripts at PAPER.md:195-201 and PAPER.md:134) */
static int row_cmp(const void* exps, int32_t exp_bytes, int32_t nvars, int64_t ta, int64_t tb)
{
    for (int32_t v = 0; v < nvars; ++v) {
        const uint32_t ea = exp_at(exps, exp_bytes, nvars, ta, v);
        const uint32_t eb = exp_at(exps, exp_bytes, nvars, tb, v);
        if (ea < eb) return -1;
        if (ea > eb) return 1;
    }
    return 0;
}

/* ------------------------------------------------- compensated accumulation */

/* Neumaier's compensated sum: s + c tracks the real-number sum of the inputs
 * to within one rounding of the result (reading A6). */
typedef struct {
    double s;       /* running sum                         */
    double c;       /* running compensation                */
    double a;       /* sum of absolute values, A_m         */
    int64_t n;      /* number of contributions, |I_m|      */
    int64_t first;  /* index of the first term of the run  */
} acc_t;

static inline void acc_init(acc_t* q, int64_t first)
{
    q->s = 0.0; q->c = 0.0; q->a = 0.0; q->n = 0; q->first = first;
}

static inline void acc_add(acc_t* q, double x)
{
    const double t = q->s + x;
    /* reading A12: non-finite values propagate as in a plain sum -- once the running sum is +-inf or NaN
     * the compensation (which would compute inf - inf) is left alone, so the value stays +-inf / NaN */
    if (isfinite(t)) {
        if (fabs(q->s) >= fabs(x)) q->c += (q->s - t) + x;
        else                       q->c += (x - t) + q->s;
    }
    q->s = t;
    q->a += fabs(x);
    q->n += 1;
}

static inline double acc_value(const acc_t* q) { return q->s + q->c; }

/* ---------------------------------------------------------- qsort contexts */

static const void* g_exps;
static int32_t g_exp_bytes;
static int32_t g_nvars;

static int cmp_term_index(const void* pa, const void* pb)
{
    const int64_t ta = *(const int64_t*)pa, tb = *(const int64_t*)pb;
    const int r = row_cmp(g_exps, g_exp_bytes, g_nvars, ta, tb);
    if (r) return r;
    return (ta > tb) - (ta < tb);     /* ties by input position: a total order */
}

/* write the U distinct monomials, given as accumulators already in ascending
 * row order, to the caller's arrays; apply the prune predicate of reading A2. */
static void emit(const acc_t* accs, const int64_t* order, int64_t U,
                 const void* exps, int32_t exp_bytes, int32_t nvars, double tol,
                 uint32_t* out_rows, double* out_sum, double* out_abs,
                 int64_t* out_count, uint8_t* out_keep)
{
    for (int64_t k = 0; k < U; ++k) {
        const acc_t* q = &accs[order ? order[k] : k];
        for (int32_t v = 0; v < nvars; ++v)
            out_rows[k * (int64_t)nvars + v] = exp_at(exps, exp_bytes, nvars, q->first, v);
        const double s = acc_value(q);
        out_sum[k] = s;
        out_abs[k] = q->a;
        out_count[k] = q->n;
        /* "removes coefficients below a user-chosen tolerance":
         * keep iff |s_m| > tol; NaN compares false and is dropped (reading A12). */
        out_keep[k] = (fabs(s) > tol) ? 1 : 0;
    }
}

static int args_ok(const double* coef, const void* exps, int32_t exp_bytes, int64_t nterms, int32_t nvars)
{
    if (nterms < 0 || nvars < 1) return 0;
    if (exp_bytes != 1 && exp_bytes != 2 && exp_bytes != 4) return 0;
    if (nterms > 0 && (!coef || !exps)) return 0;
    return 1;
}

/* --------------------------------------------- simplify: hash map + sort */

static uint64_t row_hash(const void* exps, int32_t exp_bytes, int32_t nvars, int64_t t)
{
    /* FNV-1a over the exponent values of the row */
    uint64_t h = 1469598103934665603ULL;
    for (int32_t v = 0; v < nvars; ++v) {
        uint32_t e = exp_at(exps, exp_bytes, nvars, t, v);
        for (int b = 0; b < 4; ++b) { h ^= (e & 0xffu); h *= 1099511628211ULL; e >>= 8; }
    }
    h ^= h >> 29; h *= 0xbf58476d1ce4e5b9ULL; h ^= h >> 32;
    return h;
}

static const acc_t* g_accs;
static int cmp_acc_index(const void* pa, const void* pb)
{
    const int64_t ia = *(const int64_t*)pa, ib = *(const int64_t*)pb;
    return row_cmp(g_exps, g_exp_bytes, g_nvars, g_accs[ia].first, g_accs[ib].first);
}

/* "merges repeated monomials": M = distinct rows, I_m = terms with
 * row m, s_m = sum over I_m of coef; then the distinct rows in ascending order. */
int64_t oracle_simplify(const double* coef, const void* exps, int32_t exp_bytes,
                        int64_t nterms, int32_t nvars, double tol,
                        uint32_t* out_rows, double* out_sum, double* out_abs,
                        int64_t* out_count, uint8_t* out_keep)
{
    if (!args_ok(coef, exps, exp_bytes, nterms, nvars)) return -1;
    if (nterms == 0) return 0;

    int64_t cap = 1024;                 /* slots, power of two */
    int64_t* slots = (int64_t*)malloc((size_t)cap * sizeof(int64_t));   /* acc id or -1 */
    int64_t acc_cap = 512, U = 0;
    acc_t* accs = (acc_t*)malloc((size_t)acc_cap * sizeof(acc_t));
    if (!slots || !accs) { free(slots); free(accs); return -1; }
    for (int64_t i = 0; i < cap; ++i) slots[i] = -1;

    for (int64_t t = 0; t < nterms; ++t) {
        if (2 * (U + 1) > cap) {        /* keep the load factor under one half */
            const int64_t ncap = cap * 2;
            int64_t* ns = (int64_t*)malloc((size_t)ncap * sizeof(int64_t));
            if (!ns) { free(slots); free(accs); return -1; }
            for (int64_t i = 0; i < ncap; ++i) ns[i] = -1;
            for (int64_t k = 0; k < U; ++k) {
                uint64_t p = row_hash(exps, exp_bytes, nvars, accs[k].first) & (uint64_t)(ncap - 1);
                while (ns[p] >= 0) p = (p + 1) & (uint64_t)(ncap - 1);
                ns[p] = k;
            }
            free(slots); slots = ns; cap = ncap;
        }
        uint64_t p = row_hash(exps, exp_bytes, nvars, t) & (uint64_t)(cap - 1);
        int64_t id = -1;
        while (slots[p] >= 0) {
            if (row_cmp(exps, exp_bytes, nvars, accs[slots[p]].first, t) == 0) { id = slots[p]; break; }
            p = (p + 1) & (uint64_t)(cap - 1);
        }
        if (id < 0) {                   /* a monomial not seen before */
            if (U == acc_cap) {
                acc_cap *= 2;
                acc_t* na = (acc_t*)realloc(accs, (size_t)acc_cap * sizeof(acc_t));
                if (!na) { free(slots); free(accs); return -1; }
                accs = na;
            }
            id = U++;
            acc_init(&accs[id], t);
            slots[p] = id;
        }
        acc_add(&accs[id], coef[t]);
    }
    free(slots);

    int64_t* order = (int64_t*)malloc((size_t)U * sizeof(int64_t));
    if (!order) { free(accs); return -1; }
    for (int64_t k = 0; k < U; ++k) order[k] = k;
    g_exps = exps; g_exp_bytes = exp_bytes; g_nvars = nvars; g_accs = accs;
    qsort(order, (size_t)U, sizeof(int64_t), cmp_acc_index);

    emit(accs, order, U, exps, exp_bytes, nvars, tol, out_rows, out_sum, out_abs, out_count, out_keep);
    free(order); free(accs);
    return U;
}

/* ---------------------------------------- simplify: sort, then sequential sum */

int64_t oracle_simplify_sortscan(const double* coef, const void* exps, int32_t exp_bytes,
                                 int64_t nterms, int32_t nvars, double tol,
                                 uint32_t* out_rows, double* out_sum, double* out_abs,
                                 int64_t* out_count, uint8_t* out_keep)
{
    if (!args_ok(coef, exps, exp_bytes, nterms, nvars)) return -1;
    if (nterms == 0) return 0;
    int64_t* idx = (int64_t*)malloc((size_t)nterms * sizeof(int64_t));
    acc_t* accs = (acc_t*)malloc((size_t)nterms * sizeof(acc_t));
    if (!idx || !accs) { free(idx); free(accs); return -1; }
    for (int64_t t = 0; t < nterms; ++t) idx[t] = t;
    g_exps = exps; g_exp_bytes = exp_bytes; g_nvars = nvars;
    qsort(idx, (size_t)nterms, sizeof(int64_t), cmp_term_index);

    int64_t U = 0;
    for (int64_t k = 0; k < nterms; ++k) {
        const int64_t t = idx[k];
        if (k == 0 || row_cmp(exps, exp_bytes, nvars, idx[k - 1], t) != 0) {
            acc_init(&accs[U], t);      /* a new run of equal rows starts here */
            ++U;
        }
        acc_add(&accs[U - 1], coef[t]);
    }
    emit(accs, NULL, U, exps, exp_bytes, nvars, tol, out_rows, out_sum, out_abs, out_count, out_keep);
    free(idx); free(accs);
    return U;
}

/* ------------------------------------------------------------------ product */

/* (sum_i ca_i x^a_i)(sum_j cb_j x^b_j) = sum_{i,j} (ca_i cb_j) x^(a_i+b_j)
 * (mtimes/times on scalar polynomials). */
int64_t oracle_expand(const double* ca, const void* ea, int64_t na,
                      const double* cb, const void* eb, int64_t nb,
                      int32_t exp_bytes, int32_t nvars,
                      double* out_coef, uint32_t* out_rows)
{
    if (!args_ok(ca, ea, exp_bytes, na, nvars) || !args_ok(cb, eb, exp_bytes, nb, nvars)) return -1;
    for (int64_t i = 0; i < na; ++i) {
        for (int64_t j = 0; j < nb; ++j) {
            const int64_t k = i * nb + j;
            volatile double prod = ca[i] * cb[j];      /* one rounded multiplication */
            out_coef[k] = prod;
            for (int32_t v = 0; v < nvars; ++v)
                out_rows[k * (int64_t)nvars + v] =
                    exp_at(ea, exp_bytes, nvars, i, v) + exp_at(eb, exp_bytes, nvars, j, v);
        }
    }
    return na * nb;
}

int64_t oracle_mul_simplify(const double* ca, const void* ea, int64_t na,
                            const double* cb, const void* eb, int64_t nb,
                            int32_t exp_bytes, int32_t nvars, double tol,
                            uint32_t* out_rows, double* out_sum, double* out_abs,
                            int64_t* out_count, uint8_t* out_keep)
{
    if (!args_ok(ca, ea, exp_bytes, na, nvars) || !args_ok(cb, eb, exp_bytes, nb, nvars)) return -1;
    const int64_t N = na * nb;
    if (N == 0) return 0;
    double* pc = (double*)malloc((size_t)N * sizeof(double));
    uint32_t* pr = (uint32_t*)malloc((size_t)N * (size_t)nvars * sizeof(uint32_t));
    if (!pc || !pr) { free(pc); free(pr); return -1; }
    oracle_expand(ca, ea, na, cb, eb, nb, exp_bytes, nvars, pc, pr);
    const int64_t U = oracle_simplify(pc, pr, 4, N, nvars, tol, out_rows, out_sum, out_abs, out_count, out_keep);
    free(pc); free(pr);
    return U;
}

/* --------------------------------------------------------------- evaluation */

/* p(x0) = sum_t c_t x0^alpha_t ("evaluate at a numeric point") */
int oracle_eval(const double* coef, const void* exps, int32_t exp_bytes,
                int64_t nterms, int32_t nvars, const double* x,
                double* out_value, double* out_abs)
{
    if (!args_ok(coef, exps, exp_bytes, nterms, nvars) || !x) return -1;
    long double total = 0.0L, total_abs = 0.0L;
    for (int64_t t = 0; t < nterms; ++t) {
        long double m = (long double)coef[t];
        for (int32_t v = 0; v < nvars; ++v) {
            const uint32_t e = exp_at(exps, exp_bytes, nvars, t, v);
            for (uint32_t k = 0; k < e; ++k) m *= (long double)x[v];
        }
        total += m;
        total_abs += fabsl(m);
    }
    if (out_value) *out_value = (double)total;
    if (out_abs) *out_abs = (double)total_abs;
    return 0;
}
