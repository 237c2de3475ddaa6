/*
 * polylab_oracle.h -- CPU oracle for Polylab `simplify` and polynomial products.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, link or call
 * anything in oracle/.  It shares no code, header, table or constant with the
 * CUDA path under paper_2604_06575_b200/csrc/ and never packs monomial keys.
 *
 * What it computes is the paper's definition, executed slowly:
 *   - a polynomial is "coefficient vector and exponent matrix with matching
 *     monomial count" (Table 3, constructor MPOLY(n,coef,pow);
 *     PAPER.md:97, section 3.1);
 *   - simplify(p,zeroprec) returns a "polynomial with merged monomials and small
 *     terms removed" (Table 3); it "merges repeated monomials and
 *     removes coefficients below a user-chosen tolerance" (Table 4);
 *   - a product multiplies every term of one operand with every term of the
 *     other (mtimes/times, Table 4; the merged cross term of
 *     quadprod; simplify(p_d^3), section 6.3).
 *
 * Readings of points the paper leaves open:
 *   A1 output order = ascending lexicographic on the exponent row, variable 0
 *      (column 0) most significant -- the order of the paper's machine-printed
 *      transcripts;
 *   A2 keep a merged monomial iff |s_m| > tol (absolute, strict);
 *   A4 pruning applies to merged sums only, never to input terms;
 *   A6 s_m is the real-number sum rounded (nearly) once: Neumaier compensated
 *      summation in fp64.
 *
 * Parity pins: tests/test_oracle_*.py (worked examples of the paper, closed
 * forms, brute force, exact rational / math.fsum sums).  No function here is
 * "parity unpinned".
 *
 * Exponent matrices are row-major, one row per term, `exp_bytes` in {1,2,4}
 * (unsigned little-endian integers).  Not thread-safe (qsort context is static).
 */
#ifndef POLYLAB_ORACLE_H
#define POLYLAB_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/*
 * simplify by hash map: group equal rows, sum coefficients, sort the distinct
 * rows lexicographically.  Outputs (caller-allocated, capacity `nterms` rows):
 *   out_rows  [U x nvars] uint32, ascending lexicographic, no duplicates
 *   out_sum   [U] s_m   = compensated sum of the coefficients of monomial m
 *   out_abs   [U] A_m   = sum of |coefficients| of monomial m
 *   out_count [U] |I_m| = number of input terms of monomial m
 *   out_keep  [U] 1 iff |s_m| > tol (reading A2), else 0
 * Returns U (the number of distinct monomials, UNPRUNED), or -1 on bad
 * arguments / allocation failure.  nterms == 0 returns 0.
 */
int64_t oracle_simplify(const double* coef, const void* exps, int32_t exp_bytes,
                        int64_t nterms, int32_t nvars, double tol,
                        uint32_t* out_rows, double* out_sum, double* out_abs,
                        int64_t* out_count, uint8_t* out_keep);

/*
 * The same result by a structurally different route (no hashing): sort the
 * term indices by row (ties by index), then one sequential pass that sums
 * each run.  O(N log N) row comparisons -- for small and medium inputs.
 */
int64_t oracle_simplify_sortscan(const double* coef, const void* exps, int32_t exp_bytes,
                                 int64_t nterms, int32_t nvars, double tol,
                                 uint32_t* out_rows, double* out_sum, double* out_abs,
                                 int64_t* out_count, uint8_t* out_keep);

/*
 * Raw product a*b: na*nb terms, term (i,j) at index i*nb+j has coefficient
 * fl(ca_i * cb_j) (one IEEE multiplication) and exponent row a_i + b_j.
 * Outputs: out_coef [na*nb], out_rows [na*nb x nvars] uint32.  Returns na*nb.
 */
int64_t oracle_expand(const double* ca, const void* ea, int64_t na,
                      const double* cb, const void* eb, int64_t nb,
                      int32_t exp_bytes, int32_t nvars,
                      double* out_coef, uint32_t* out_rows);

/*
 * simplify(a*b): oracle_expand followed by oracle_simplify.  Output arrays need
 * capacity na*nb.  A_m is the sum of |fl(ca_i*cb_j)|.  Returns U or -1.
 */
int64_t oracle_mul_simplify(const double* ca, const void* ea, int64_t na,
                            const double* cb, const void* eb, int64_t nb,
                            int32_t exp_bytes, int32_t nvars, double tol,
                            uint32_t* out_rows, double* out_sum, double* out_abs,
                            int64_t* out_count, uint8_t* out_keep);

/*
 * p(x) = sum_t coef[t] * prod_v x[v]^exps[t][v]  (the paper's eval),
 * by repeated multiplication in long double.  *out_value = p(x),
 * *out_abs = sum_t |coef[t] * x^alpha_t| (the scale for comparisons).
 */
int oracle_eval(const double* coef, const void* exps, int32_t exp_bytes,
                int64_t nterms, int32_t nvars, const double* x,
                double* out_value, double* out_abs);

#ifdef __cplusplus
}
#endif
#endif /* POLYLAB_ORACLE_H */
