/*
 * zippel_ref.h -- CPU ORACLE for one Zippel lifting step over Z/pZ.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may load it.  It shares no code, header,
 * table or constant with the CUDA path under paper_2505_24256_b200/csrc/ and include/.
 *
 * Everything here is the plain, single-threaded, literal form of what the paper's method
 * computes (PAPER.md = /root/reference/PAPER.md, arXiv 2505.24256):
 *   - modular multiplication is the paper's "variant 1", (unsigned __int128)a*b % n
 *     (section 2.1); no Montgomery form, no deferred reduction, no tables;
 *   - the transposed Vandermonde solve is the master-polynomial / synthetic-division /
 *     Horner route of section 2.2, cross-checked by the generic O(t^3)
 *     elimination the paper mentions in section 1;
 *   - Newton interpolation is eq. (1);
 *   - the balanced variant is eq. (4).
 * Readings of garbled / silent passages are listed in DESIGN.md ("Readings").
 *
 * Parity pins: every function below is pinned by tests/test_oracle_pins.py against something
 * other than itself (Python big integers, exact rational Lagrange interpolation, Vieta,
 * Gauss-Jordan, closed forms, planted recovery, the golden worked example).  No function
 * here is "parity unpinned".
 *
 * All pointers are HOST pointers.  All residues are canonical, in [0, p).  3 <= p < 2^63, p odd
 * (primality is the caller's business; tests use p = 2^63 - 25 and small primes).
 *
 * Layout (same as the product's C-ABI so tests can feed both):
 *   exps    uint16 [T_tot x nv] row-major, row i = exponents of skeleton term i
 *   offsets int64  [F+1], terms of function f are [offsets[f], offsets[f+1]); T_tot = offsets[F]
 *   vals    uint64 [B x T_tot], vals[b*T_tot + offsets[f] + s] = v_{b,s} of function f
 *   coefs / out  same layout as vals
 *   status  int32  [F]: 0 ok, else (index << 8) | code, see REF_ST_*
 */
#ifndef ZIPPEL_REF_H
#define ZIPPEL_REF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define REF_OK 0
#define REF_ERR_ARG 1

#define REF_ST_DUPLICATE_NODE 16   /* den_i == 0 (two terms map to one node) or m_i == 0 with s0 = 1 */
#define REF_ST_DUPLICATE_SAMPLE 17 /* c_j == c_j' in Newton */
#define REF_ST_ZERO_PIVOT 18       /* u_{0,s} == 0 in balancing */
#define REF_ST_NO_RATIONAL 21 /* rational reconstruction: no a/b within the bounds (or gcd(a, b) != 1) */
#define REF_ST_THIELE_DEGENERATE 20 /* an inverse difference of eq. (2) has a zero denominator at some but not all points */

/* ---- arithmetic in Z/pZ (variant 1 is the definition) ---- */
uint64_t ref_mulmod(uint64_t a, uint64_t b, uint64_t p);
uint64_t ref_addmod(uint64_t a, uint64_t b, uint64_t p);
uint64_t ref_submod(uint64_t a, uint64_t b, uint64_t p);
uint64_t ref_powmod(uint64_t a, uint64_t e, uint64_t p);
uint64_t ref_invmod(uint64_t a, uint64_t p); /* a^(p-2); a != 0, p prime */

/* ---- the prime (north_star: deterministic Miller-Rabin fixes p) ---- */
int ref_is_prime_u64(uint64_t n);
uint64_t ref_largest_prime_below(uint64_t n); /* largest prime < n, n > 2 */

/* ---- (a1) nodes m_i = prod_j y_j^{e_ij}  (eq. (3)) ---- */
int ref_zippel_eval_nodes(const uint16_t* exps, int64_t T_tot, int nv, const uint64_t* anchors,
                          uint64_t p, uint64_t* nodes);

/* ---- (a2) master polynomial M(z) = prod_i (z - m_i), M[0..t], M[t] = 1 ---- */
void ref_master_poly(const uint64_t* m, int64_t t, uint64_t p, uint64_t* M);

/* ---- (a3)+(a4) per node: synthetic division, Horner denominator, B dot products, scale
 *      (PAPER.md L193-197).  Also exported piecewise so tests can compare intermediates:
 *      den[i] = Q_i(m_i), num[b*t + i] = sum_s q_{i,s} v_{b,s}  (single function, ld = t). ---- */
void ref_node_quotient(const uint64_t* M, int64_t t, uint64_t m_i, uint64_t p, uint64_t* q /* [t] */);
void ref_node_solve(const uint64_t* m, const uint64_t* M, int64_t t, const uint64_t* vals, int64_t ld,
                    int B, uint64_t p, uint64_t* den /* [t] */, uint64_t* num /* [B x t], ld = t */);

/* the same per-node routine for n node values x[] chosen by the caller; den [n], num [B x n] */
void ref_node_solve_at(const uint64_t* x, int64_t n, const uint64_t* M, int64_t t, const uint64_t* vals, int64_t ld,
                       int B, uint64_t p, uint64_t* den, uint64_t* num);

int ref_vandermonde_solve_batch(const uint64_t* nodes, const int64_t* offsets, int F,
                                const uint64_t* vals, int B, int s0, uint64_t p, uint64_t* coefs,
                                int32_t* status);

/* ---- brute-force cross-check: A[s][i] = m_i^(s+s0), solve A c = v by Gauss-Jordan, O(t^3)
 *      ("complexity O(t^3)").  Returns 0, or 1 if singular. ---- */
int ref_gauss_solve(const uint64_t* m, int64_t t, const uint64_t* v, int s0, uint64_t p, uint64_t* c);

/* ---- (a5) Newton interpolation in x_k, eq. (1), 0-based.
 *      basis 0: a_0..a_D with f(x) = a_0 + (x-c_0)[a_1 + (x-c_1)[a_2 + ...]];
 *      basis 1: monomial coefficients P_0..P_D in x_k. ---- */
int ref_newton_interp_batch(const uint64_t* samples, int B, const uint64_t* vals, int64_t n, int64_t ld,
                            uint64_t p, int basis, uint64_t* out, int32_t* status);

/* ---- one lifting step = (a1) .. (a5) ---- */
int ref_zippel_lift_step(const uint16_t* exps, const int64_t* offsets, int F, int nv,
                         const uint64_t* anchors, const uint64_t* samples, int B, int s0,
                         const uint64_t* vals, uint64_t p, int basis, uint64_t* out,
                         uint64_t* nodes_out /* may be NULL */, int32_t* status);

/* ---- (a6) power sums R_{b,s} = sum_i a_{b,i} m_i^(s+s0), s = 0..t_f-1: the skeleton evaluated
 *      at the Zippel probe points.  coef and out in the vals layout. ---- */
int ref_power_sums(const uint64_t* nodes, const int64_t* offsets, int F, const uint64_t* coef, int B,
                   int s0, uint64_t p, uint64_t* out);

/* ---- (a6) balanced lifting step for one part (numerator or denominator), eq. (4)
 *      (PAPER.md L215-217):  V_{j,s} = u_{j,s} * R_s / u_{0,s},  then (a2)..(a5) on V. ---- */
typedef struct {
  const uint16_t* exps;     /* [T_tot x nv] */
  const int64_t* offsets;   /* [F+1] */
  const uint64_t* skel;     /* [T_tot] skeleton coefficients a'_i */
  const uint64_t* uvals;    /* [B x T_tot] normalised univariate values u_{j,s} */
  uint64_t* out;            /* [B x T_tot] */
} ref_part;

int ref_balanced_zippel_lift_step(const ref_part* num, const ref_part* den, int F, int nv,
                                  const uint64_t* anchors, const uint64_t* samples, int B, int s0,
                                  uint64_t p, int basis, int32_t* status /* [2F]: num then den */);

/* ---- values of the coefficient polynomials in x_k at the samples (the inverse of basis-1 Newton):
 *      out[j*ld + i] = sum_d P[d*ld + i] * c_j^d, d = 0..B-1 ("similar reconstructed
 *      polynomials for other values of x_k").  Used by tests to make probe values of a planted function. ---- */
int ref_poly_rows_eval(const uint64_t* samples, int B, const uint64_t* P, int64_t n, int64_t ld,
                       uint64_t p, uint64_t* out);

/* ---- fresh probes: value of a sparse polynomial sum_i coef_i prod_j z_j^{e_ij} ---- */
uint64_t ref_eval_sparse(const uint16_t* exps, const uint64_t* coef, int64_t t, int nv,
                         const uint64_t* point, uint64_t p);

/* ---- (f2) univariate Thiele reconstruction, eq. (2), one column of values at a time:
 *   f(x) = b_0 + (x - x_0) / ( b_1 + (x - x_1) / ( b_2 + ... + (x - x_{K-2}) / b_{K-1} ) )      (0-based)
 * with the inverse differences  phi_0(x_i) = f(x_i),  phi_k(x_i) = (x_i - x_{k-1}) / (phi_{k-1}(x_i) - phi_{k-1}(x_{k-1})),
 * i >= k, and b_k = phi_k(x_k).  The fraction ends at K = k terms when every phi_{k-1}(x_i), i >= k, equals
 * phi_{k-1}(x_{k-1}) (the function is reproduced at all remaining points); K = T if that never happens.  If
 * only some of them are equal the column gets status (k << 8) | REF_ST_THIELE_DEGENERATE and zero output.
 * The fraction is then expanded from the tail, (N, D) <- (b_k N + (x - x_k) D, N), starting at (b_{K-1}, 1),
 * trimmed to its true degrees and scaled so that D is monic.
 *   points [T] pairwise distinct; vals [T x n] (row j = values at x_j, leading dimension ld)
 *   num, den [T x n]: row d = coefficient of x^d (zero above the degree); degs [2 x n]: deg N, deg D (deg N = -1
 *   for the zero function); cf [T x n]: b_0..b_{K-1} (zero above K), may be NULL; status [n].
 * A duplicate point: every status = (j << 8) | REF_ST_DUPLICATE_SAMPLE. ---- */
int ref_thiele_reconstruct_batch(const uint64_t* points, int T, const uint64_t* vals, int64_t n, int64_t ld,
                                 uint64_t p, uint64_t* num, uint64_t* den, int32_t* degs, uint64_t* cf,
                                 int32_t* status);

/* ---- (f1) skeleton extension between two lifting steps (the polynomial in k variables
 *      reconstructed by one step is the skeleton of the next): from the monomial-in-x_k coefficients
 *      coefs[d*T_tot + off_f + i] of every skeleton term i of function f, the terms of the new skeleton are the
 *      pairs (i, d) with a non-zero coefficient, in the order i ascending, then d ascending:
 *        new_exps row = (exps row of i, d)   [nv + 1 columns],   new_coefs = that coefficient,
 *        new_offsets [F+1] term ranges,   degs[f] = largest d with a non-zero coefficient in f (-1: none;
 *        the early-termination test: degs[f] < B-1 means fewer samples of x_k would have sufficed).
 *      Returns the total number of new terms through new_offsets[F]; writes at most cap terms. ---- */
int ref_extend_skeleton(const uint16_t* exps, const int64_t* offsets, int F, int nv, const uint64_t* coefs, int B,
                        uint64_t p, uint16_t* new_exps, uint64_t* new_coefs, int64_t cap, int64_t* new_offsets,
                        int32_t* degs);

/* ---- (f4) second prime + CRT + rational reconstruction (the reduction is run over several large
 *      primes "fitting into 2^64" and "the final reconstruction to rational numbers is performed as a final step").
 *      For every coefficient i with residues r1[i] mod p1 and r2[i] mod p2 (p1 != p2 odd primes < 2^63):
 *        x = r1 + p1 * ((r2 - r1) * p1^-1 mod p2)  in [0, m),  m = p1 p2           (Chinese remainder theorem)
 *        extended Euclid on (m, x):  (r, t) sequences with r_j = t_j x (mod m), stopped at the first r_j <= N,
 *        N = D = floor(sqrt((m - 1) / 2))  (Wang's bounds: 2 N D < m makes the answer unique);
 *        a = r_j, b = t_j, sign moved to a so that b > 0; valid iff b <= D and gcd(|a|, b) = 1.
 *      num [n] int64 (signed), den [n] int64 (> 0), status [n]: 0 or REF_ST_NO_RATIONAL (num = den = 0). ---- */
int ref_crt_rational_batch(const uint64_t* r1, const uint64_t* r2, int64_t n, uint64_t p1, uint64_t p2, int64_t* num,
                           int64_t* den, int32_t* status);

#ifdef __cplusplus
}
#endif
#endif
