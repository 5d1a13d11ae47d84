/*
 * zippel_ref.c -- CPU ORACLE (test infrastructure, not the product; see zippel_ref.h).
 *
 * Plain C, single-threaded, one mulmod definition, no shared code with the CUDA path.
 * Each function cites the passage of /root/reference/PAPER.md (arXiv 2505.24256) it follows.
 * Where the paper's text is garbled the reading is the one listed in DESIGN.md ("Readings",
 * G1..G25, taken from SURVEY.md 8(c).2).
 */
#include "zippel_ref.h"

#include <stdlib.h>
#include <string.h>

typedef unsigned __int128 u128;

/* ------------------------------------------------------------------------------------------
 * Arithmetic in Z/pZ.  PAPER.md L88-100 (section 2.1, variant 1): "return
 * (static_cast<__uint128_t>(a) * b) % n".  On the CPU this is simply the definition.
 * ---------------------------------------------------------------------------------------- */
uint64_t ref_mulmod(uint64_t a, uint64_t b, uint64_t p) { return (uint64_t)(((u128)a * b) % p); }

uint64_t ref_addmod(uint64_t a, uint64_t b, uint64_t p) { return (uint64_t)(((u128)a + b) % p); }

uint64_t ref_submod(uint64_t a, uint64_t b, uint64_t p) { return (uint64_t)(((u128)a + p - (b % p)) % p); }

/* square-and-multiply, right-to-left */
uint64_t ref_powmod(uint64_t a, uint64_t e, uint64_t p) {
  uint64_t r = 1 % p;
  a %= p;
  while (e) {
    if (e & 1) r = ref_mulmod(r, a, p);
    a = ref_mulmod(a, a, p);
    e >>= 1;
  }
  return r;
}

/* Fermat: a^(p-2) (p prime, a != 0 mod p) */
uint64_t ref_invmod(uint64_t a, uint64_t p) { return ref_powmod(a, p - 2, p); }

/* ------------------------------------------------------------------------------------------
 * Deterministic Miller-Rabin.  The bases {2,...,37} are a proven deterministic set for every
 * n < 3.3e24, hence for all 64-bit n.  north_star: "a deterministic Miller-Rabin test that fixes
 * p as the largest prime below 2^63".
 * ---------------------------------------------------------------------------------------- */
int ref_is_prime_u64(uint64_t n) {
  static const uint64_t bases[12] = {2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37};
  if (n < 2) return 0;
  for (int i = 0; i < 12; ++i) {
    if (n == bases[i]) return 1;
    if (n % bases[i] == 0) return 0;
  }
  uint64_t d = n - 1;
  int r = 0;
  while ((d & 1) == 0) {
    d >>= 1;
    ++r;
  }
  for (int i = 0; i < 12; ++i) {
    uint64_t x = ref_powmod(bases[i], d, n);
    if (x == 1 || x == n - 1) continue;
    int composite = 1;
    for (int k = 1; k < r; ++k) {
      x = ref_mulmod(x, x, n);
      if (x == n - 1) {
        composite = 0;
        break;
      }
    }
    if (composite) return 0;
  }
  return 1;
}

uint64_t ref_largest_prime_below(uint64_t n) {
  for (uint64_t c = n - 1; c >= 2; --c)
    if (ref_is_prime_u64(c)) return c;
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * (a1) Nodes.  PAPER.md L55 eq. (3): term i of the skeleton is x_1^{p_1,i} ... x_{k-1}^{p_{k-1},i};
 * L60 (reading G1): the s-th Zippel probe is (y_1^s, ..., y_{k-1}^s), so the term takes the value
 * m_i^s with m_i = prod_j y_j^{e_ij}.
 * ---------------------------------------------------------------------------------------- */
int ref_zippel_eval_nodes(const uint16_t* exps, int64_t T_tot, int nv, const uint64_t* anchors,
                          uint64_t p, uint64_t* nodes) {
  if (!exps || !anchors || !nodes || T_tot <= 0 || nv <= 0) return REF_ERR_ARG;
  for (int64_t i = 0; i < T_tot; ++i) {
    uint64_t m = 1 % p;
    for (int j = 0; j < nv; ++j) m = ref_mulmod(m, ref_powmod(anchors[j], exps[i * nv + j], p), p);
    nodes[i] = m;
  }
  return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * (a2) Master polynomial M(z) = prod_i (z - m_i) = sum_l M_l z^l ("Lagrange
 * interpolation").  Start M = [1]; for each node: M <- M * (z - m).
 * ---------------------------------------------------------------------------------------- */
void ref_master_poly(const uint64_t* m, int64_t t, uint64_t p, uint64_t* M) {
  M[0] = 1 % p;
  for (int64_t n = 0; n < t; ++n) {
    /* M currently has degree n (coefficients M[0..n]); multiply by (z - m[n]) */
    M[n + 1] = M[n];
    for (int64_t l = n; l >= 1; --l) M[l] = ref_submod(M[l - 1], ref_mulmod(m[n], M[l], p), p);
    M[0] = ref_submod(0, ref_mulmod(m[n], M[0], p), p);
  }
}

/* ------------------------------------------------------------------------------------------
 * (a3) Synthetic division of M by (z - m_i): Q_i(z) = M(z)/(z - m_i) = sum_{l<t} q_l z^l with
 * q_{t-1} = 1, q_{l-1} = M_l + m_i q_l  ("Horner's scheme", L194 "vector of powers").
 * ---------------------------------------------------------------------------------------- */
void ref_node_quotient(const uint64_t* M, int64_t t, uint64_t m_i, uint64_t p, uint64_t* q) {
  q[t - 1] = 1 % p;
  for (int64_t l = t - 1; l >= 1; --l) q[l - 1] = ref_addmod(M[l], ref_mulmod(m_i, q[l], p), p);
}

/* Per node i:
 *   q <- 1 (= q_{t-1}); d <- 1; acc_b <- v_{b,t-1};
 *   for l = t-1 .. 1:  q <- M_l + m_i q  (= q_{l-1});  d <- d m_i + q;  acc_b <- acc_b + q v_{b,l-1}.
 * Then d = Q_i(m_i) = prod_{j != i} (m_i - m_j)  (reading G15) and acc_b = sum_s q_{i,s} v_{b,s}.
 */
void ref_node_solve(const uint64_t* m, const uint64_t* M, int64_t t, const uint64_t* vals, int64_t ld,
                    int B, uint64_t p, uint64_t* den, uint64_t* num) {
  for (int64_t i = 0; i < t; ++i) {
    uint64_t q = 1 % p, d = 1 % p;
    for (int b = 0; b < B; ++b) num[(int64_t)b * t + i] = vals[(int64_t)b * ld + (t - 1)] % p;
    for (int64_t l = t - 1; l >= 1; --l) {
      q = ref_addmod(M[l], ref_mulmod(m[i], q, p), p);
      d = ref_addmod(ref_mulmod(d, m[i], p), q, p);
      for (int b = 0; b < B; ++b)
        num[(int64_t)b * t + i] =
            ref_addmod(num[(int64_t)b * t + i], ref_mulmod(q, vals[(int64_t)b * ld + (l - 1)], p), p);
    }
    den[i] = d;
  }
}

/* The same per-node routine for n node values picked by the caller (the full-size parity check of SURVEY.md 8(c).3:
 * "the oracle's per-node routine on 256 random node indices"): M has degree t, x[] are n of its roots (or any
 * residues: then d = Q_x(x) with Q_x = the quotient of M by (z - x), remainder dropped).  den [n], num [B x n].
 */
void ref_node_solve_at(const uint64_t* x, int64_t n, const uint64_t* M, int64_t t, const uint64_t* vals, int64_t ld,
                       int B, uint64_t p, uint64_t* den, uint64_t* num) {
  for (int64_t i = 0; i < n; ++i) {
    uint64_t q = 1 % p, d = 1 % p;
    for (int b = 0; b < B; ++b) num[(int64_t)b * n + i] = vals[(int64_t)b * ld + (t - 1)] % p;
    for (int64_t l = t - 1; l >= 1; --l) {
      q = ref_addmod(M[l], ref_mulmod(x[i], q, p), p);
      d = ref_addmod(ref_mulmod(d, x[i], p), q, p);
      for (int b = 0; b < B; ++b)
        num[(int64_t)b * n + i] =
            ref_addmod(num[(int64_t)b * n + i], ref_mulmod(q, vals[(int64_t)b * ld + (l - 1)], p), p);
    }
    den[i] = d;
  }
}

/* ------------------------------------------------------------------------------------------
 * (a2)-(a4) Transposed Vandermonde solve, all functions, all right-hand sides.
 * System (reading G1):  sum_i c_i m_i^(s+s0) = v_s,  s = 0..t-1.
 * With Q_i as above:  sum_s q_{i,s} v_s = sum_j c_j m_j^s0 Q_i(m_j) = c_i m_i^s0 Q_i(m_i), so
 *   c_i = (sum_s q_{i,s} v_s) / Q_i(m_i)  [ / m_i if s0 = 1 ].
 * ---------------------------------------------------------------------------------------- */
int ref_vandermonde_solve_batch(const uint64_t* nodes, const int64_t* offsets, int F,
                                const uint64_t* vals, int B, int s0, uint64_t p, uint64_t* coefs,
                                int32_t* status) {
  if (!nodes || !offsets || !vals || !coefs || !status || F <= 0 || B <= 0 || (s0 != 0 && s0 != 1))
    return REF_ERR_ARG;
  const int64_t T_tot = offsets[F];
  for (int f = 0; f < F; ++f) {
    const int64_t off = offsets[f], t = offsets[f + 1] - offsets[f];
    if (t <= 0) return REF_ERR_ARG;
    const uint64_t* m = nodes + off;
    uint64_t* M = (uint64_t*)malloc((size_t)(t + 1) * sizeof(uint64_t));
    uint64_t* den = (uint64_t*)malloc((size_t)t * sizeof(uint64_t));
    uint64_t* num = (uint64_t*)malloc((size_t)t * (size_t)B * sizeof(uint64_t));
    ref_master_poly(m, t, p, M);
    ref_node_solve(m, M, t, vals + off, T_tot, B, p, den, num);
    status[f] = 0;
    for (int64_t i = 0; i < t; ++i) {
      if (den[i] == 0 || (s0 == 1 && m[i] == 0)) {
        status[f] = (int32_t)(((uint32_t)i << 8) | REF_ST_DUPLICATE_NODE);
        break;
      }
    }
    if (status[f] == 0) {
      for (int64_t i = 0; i < t; ++i) {
        uint64_t scale = ref_invmod(den[i], p);
        if (s0 == 1) scale = ref_mulmod(scale, ref_invmod(m[i], p), p);
        for (int b = 0; b < B; ++b)
          coefs[(int64_t)b * T_tot + off + i] = ref_mulmod(num[(int64_t)b * t + i], scale, p);
      }
    }
    free(M);
    free(den);
    free(num);
  }
  return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * Brute force (the generic solve "has a complexity O(t^3)"): A[s][i] = m_i^(s+s0),
 * Gauss-Jordan with the first non-zero pivot in each column.
 * ---------------------------------------------------------------------------------------- */
int ref_gauss_solve(const uint64_t* m, int64_t t, const uint64_t* v, int s0, uint64_t p, uint64_t* c) {
  const int64_t w = t + 1;
  uint64_t* A = (uint64_t*)malloc((size_t)t * (size_t)w * sizeof(uint64_t));
  for (int64_t s = 0; s < t; ++s) {
    for (int64_t i = 0; i < t; ++i) A[s * w + i] = ref_powmod(m[i], (uint64_t)(s + s0), p);
    A[s * w + t] = v[s] % p;
  }
  for (int64_t col = 0; col < t; ++col) {
    int64_t piv = -1;
    for (int64_t r = col; r < t; ++r)
      if (A[r * w + col] != 0) {
        piv = r;
        break;
      }
    if (piv < 0) {
      free(A);
      return 1;
    }
    if (piv != col)
      for (int64_t k = 0; k < w; ++k) {
        uint64_t tmp = A[col * w + k];
        A[col * w + k] = A[piv * w + k];
        A[piv * w + k] = tmp;
      }
    const uint64_t inv = ref_invmod(A[col * w + col], p);
    for (int64_t k = 0; k < w; ++k) A[col * w + k] = ref_mulmod(A[col * w + k], inv, p);
    for (int64_t r = 0; r < t; ++r) {
      if (r == col) continue;
      const uint64_t fct = A[r * w + col];
      if (fct == 0) continue;
      for (int64_t k = 0; k < w; ++k)
        A[r * w + k] = ref_submod(A[r * w + k], ref_mulmod(fct, A[col * w + k], p), p);
    }
  }
  for (int64_t i = 0; i < t; ++i) c[i] = A[i * w + t];
  free(A);
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * (a5) Newton interpolation, eq. (1), 0-based (reading G16):
 *   f(x) = a_0 + (x - c_0)[a_1 + (x - c_1)[a_2 + ...]].
 * Divided differences in place: for l = 1..D: for j = D down to l:
 *   a_j <- (a_j - a_{j-1}) / (c_j - c_{j-l}).
 * basis 1 expands to monomials: P <- [a_D]; for j = D-1..0: P <- P (x - c_j) + a_j.
 * The B(B-1)/2 inverse differences depend only on the samples and are computed once.
 * status[0]: smallest j with c_j == c_j' for some j' < j  -> (j << 8) | DUPLICATE_SAMPLE.
 * ---------------------------------------------------------------------------------------- */
int ref_newton_interp_batch(const uint64_t* samples, int B, const uint64_t* vals, int64_t n, int64_t ld,
                            uint64_t p, int basis, uint64_t* out, int32_t* status) {
  if (!samples || !vals || !out || !status || B <= 0 || n <= 0 || ld < n || (basis != 0 && basis != 1))
    return REF_ERR_ARG;
  const int D = B - 1;
  status[0] = 0;
  for (int j = 0; j < B && status[0] == 0; ++j)
    for (int jj = 0; jj < j; ++jj)
      if (samples[j] % p == samples[jj] % p) {
        status[0] = (int32_t)(((uint32_t)j << 8) | REF_ST_DUPLICATE_SAMPLE);
        break;
      }
  if (status[0] != 0) return REF_OK;

  uint64_t* invdiff = (uint64_t*)malloc((size_t)B * (size_t)B * sizeof(uint64_t));
  for (int j = 0; j < B; ++j)
    for (int jj = 0; jj < j; ++jj) invdiff[j * B + jj] = ref_invmod(ref_submod(samples[j], samples[jj], p), p);
  uint64_t* a = (uint64_t*)malloc((size_t)B * sizeof(uint64_t));
  uint64_t* P = (uint64_t*)malloc((size_t)B * sizeof(uint64_t));

  for (int64_t i = 0; i < n; ++i) {
    for (int j = 0; j < B; ++j) a[j] = vals[(int64_t)j * ld + i] % p;
    for (int l = 1; l <= D; ++l)
      for (int j = D; j >= l; --j) a[j] = ref_mulmod(ref_submod(a[j], a[j - 1], p), invdiff[j * B + (j - l)], p);
    if (basis == 0) {
      for (int j = 0; j < B; ++j) out[(int64_t)j * ld + i] = a[j];
    } else {
      /* P has degree deg; P <- P (x - c_j) + a_j */
      int deg = 0;
      P[0] = a[D];
      for (int j = D - 1; j >= 0; --j) {
        const uint64_t cj = samples[j] % p;
        P[deg + 1] = P[deg];
        for (int k = deg; k >= 1; --k) P[k] = ref_submod(P[k - 1], ref_mulmod(cj, P[k], p), p);
        P[0] = ref_submod(a[j], ref_mulmod(cj, P[0], p), p);
        ++deg;
      }
      for (int j = 0; j < B; ++j) out[(int64_t)j * ld + i] = P[j];
    }
  }
  free(invdiff);
  free(a);
  free(P);
  return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * One lifting step k-1 -> k: nodes, the B = D+1 Vandermonde solves, Newton in x_k
 * on every coefficient.  A function whose solve failed keeps its solve status; otherwise a duplicate
 * sample marks every function.
 * ---------------------------------------------------------------------------------------- */
int ref_zippel_lift_step(const uint16_t* exps, const int64_t* offsets, int F, int nv,
                         const uint64_t* anchors, const uint64_t* samples, int B, int s0,
                         const uint64_t* vals, uint64_t p, int basis, uint64_t* out, uint64_t* nodes_out,
                         int32_t* status) {
  if (!exps || !offsets || !anchors || !samples || !vals || !out || !status || F <= 0) return REF_ERR_ARG;
  const int64_t T_tot = offsets[F];
  if (T_tot <= 0) return REF_ERR_ARG;
  uint64_t* nodes = (uint64_t*)malloc((size_t)T_tot * sizeof(uint64_t));
  uint64_t* coefs = (uint64_t*)calloc((size_t)T_tot * (size_t)B, sizeof(uint64_t));
  int rc = ref_zippel_eval_nodes(exps, T_tot, nv, anchors, p, nodes);
  if (rc == REF_OK) rc = ref_vandermonde_solve_batch(nodes, offsets, F, vals, B, s0, p, coefs, status);
  int32_t nst = 0;
  if (rc == REF_OK) rc = ref_newton_interp_batch(samples, B, coefs, T_tot, T_tot, p, basis, out, &nst);
  if (rc == REF_OK && nst != 0)
    for (int f = 0; f < F; ++f)
      if (status[f] == 0) status[f] = nst;
  if (rc == REF_OK && nodes_out) memcpy(nodes_out, nodes, (size_t)T_tot * sizeof(uint64_t));
  free(nodes);
  free(coefs);
  return rc;
}

/* ------------------------------------------------------------------------------------------
 * (a6) Power sums: the skeleton (with coefficient row b) evaluated at the Zippel probe points,
 *   R_{b,s} = sum_i a_{b,i} m_i^(s+s0)   (L219 "raise base variable values to various
 *   powers and substitute them into the polynomial").
 * ---------------------------------------------------------------------------------------- */
int ref_power_sums(const uint64_t* nodes, const int64_t* offsets, int F, const uint64_t* coef, int B,
                   int s0, uint64_t p, uint64_t* out) {
  if (!nodes || !offsets || !coef || !out || F <= 0 || B <= 0 || (s0 != 0 && s0 != 1)) return REF_ERR_ARG;
  const int64_t T_tot = offsets[F];
  for (int f = 0; f < F; ++f) {
    const int64_t off = offsets[f], t = offsets[f + 1] - offsets[f];
    for (int b = 0; b < B; ++b)
      for (int64_t s = 0; s < t; ++s) {
        uint64_t r = 0;
        for (int64_t i = 0; i < t; ++i)
          r = ref_addmod(r, ref_mulmod(coef[(int64_t)b * T_tot + off + i],
                                       ref_powmod(nodes[off + i], (uint64_t)(s + s0), p), p), p);
        out[(int64_t)b * T_tot + off + s] = r;
      }
  }
  return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * (a6) Balanced lifting step for one part.  PAPER.md L215-217 eq. (4), reading G3: with u_{j,s} the
 * normalised univariate value at probe s and sample c_j (true value times an unknown h_s), and the
 * skeleton a' (true coefficients at c_0 times an unknown C):
 *   V_{j,s} = u_{j,s} * R_s / u_{0,s},   R_s = sum_i a'_i m_i^(s+s0)  = skeleton value at probe s,
 * equals C * n(y^s, c_j); the numerator and the denominator are then lifted independently.
 * status: ZERO_PIVOT (smallest s with u_{0,s} = 0), else the solve's, else Newton's.
 * ---------------------------------------------------------------------------------------- */
static int ref_balanced_part(const ref_part* part, int F, int nv, const uint64_t* anchors,
                             const uint64_t* samples, int B, int s0, uint64_t p, int basis, int32_t* status) {
  const int64_t T_tot = part->offsets[F];
  if (T_tot <= 0) return REF_ERR_ARG;
  uint64_t* nodes = (uint64_t*)malloc((size_t)T_tot * sizeof(uint64_t));
  uint64_t* R = (uint64_t*)malloc((size_t)T_tot * sizeof(uint64_t));
  uint64_t* V = (uint64_t*)calloc((size_t)T_tot * (size_t)B, sizeof(uint64_t));
  uint64_t* coefs = (uint64_t*)calloc((size_t)T_tot * (size_t)B, sizeof(uint64_t));
  int32_t* pst = (int32_t*)calloc((size_t)F, sizeof(int32_t));
  int rc = ref_zippel_eval_nodes(part->exps, T_tot, nv, anchors, p, nodes);
  if (rc == REF_OK) rc = ref_power_sums(nodes, part->offsets, F, part->skel, 1, s0, p, R);
  if (rc == REF_OK) {
    for (int f = 0; f < F; ++f) {
      const int64_t off = part->offsets[f], t = part->offsets[f + 1] - off;
      for (int64_t s = 0; s < t; ++s) {
        const uint64_t u0 = part->uvals[off + s] % p;
        if (u0 == 0) {
          pst[f] = (int32_t)(((uint32_t)s << 8) | REF_ST_ZERO_PIVOT);
          break;
        }
      }
      if (pst[f] != 0) { /* keep the solve well defined; outputs of a failed function are unspecified */
        for (int j = 0; j < B; ++j)
          for (int64_t s = 0; s < t; ++s) V[(int64_t)j * T_tot + off + s] = (j == 0) ? R[off + s] : 0;
        continue;
      }
      for (int64_t s = 0; s < t; ++s) {
        const uint64_t scale = ref_mulmod(R[off + s], ref_invmod(part->uvals[off + s] % p, p), p);
        for (int j = 0; j < B; ++j)
          V[(int64_t)j * T_tot + off + s] = ref_mulmod(part->uvals[(int64_t)j * T_tot + off + s] % p, scale, p);
      }
    }
    rc = ref_vandermonde_solve_batch(nodes, part->offsets, F, V, B, s0, p, coefs, status);
  }
  int32_t nst = 0;
  if (rc == REF_OK) rc = ref_newton_interp_batch(samples, B, coefs, T_tot, T_tot, p, basis, part->out, &nst);
  if (rc == REF_OK)
    for (int f = 0; f < F; ++f) {
      if (pst[f] != 0) status[f] = pst[f];
      else if (status[f] == 0 && nst != 0) status[f] = nst;
    }
  free(nodes);
  free(R);
  free(V);
  free(coefs);
  free(pst);
  return rc;
}

int ref_balanced_zippel_lift_step(const ref_part* num, const ref_part* den, int F, int nv,
                                  const uint64_t* anchors, const uint64_t* samples, int B, int s0,
                                  uint64_t p, int basis, int32_t* status) {
  if (!num || !den || !anchors || !samples || !status || F <= 0 || B <= 0) return REF_ERR_ARG;
  int rc = ref_balanced_part(num, F, nv, anchors, samples, B, s0, p, basis, status);
  if (rc == REF_OK) rc = ref_balanced_part(den, F, nv, anchors, samples, B, s0, p, basis, status + F);
  return rc;
}

/* Values at x_k = c_j of polynomials given by monomial coefficients (row d = coefficient of x_k^d):
 * plain sum of powers, term by term. */
int ref_poly_rows_eval(const uint64_t* samples, int B, const uint64_t* P, int64_t n, int64_t ld,
                       uint64_t p, uint64_t* out) {
  if (!samples || !P || !out || B <= 0 || n <= 0 || ld < n) return REF_ERR_ARG;
  for (int j = 0; j < B; ++j)
    for (int64_t i = 0; i < n; ++i) {
      uint64_t r = 0;
      for (int d = 0; d < B; ++d)
        r = ref_addmod(r, ref_mulmod(P[(int64_t)d * ld + i] % p, ref_powmod(samples[j], (uint64_t)d, p), p), p);
      out[(int64_t)j * ld + i] = r;
    }
  return REF_OK;
}

/* Fresh probes ("the following probes ... also match the guessed function"). */
uint64_t ref_eval_sparse(const uint16_t* exps, const uint64_t* coef, int64_t t, int nv,
                         const uint64_t* point, uint64_t p) {
  uint64_t r = 0;
  for (int64_t i = 0; i < t; ++i) {
    uint64_t term = coef[i] % p;
    for (int j = 0; j < nv; ++j) term = ref_mulmod(term, ref_powmod(point[j], exps[i * nv + j], p), p);
    r = ref_addmod(r, term, p);
  }
  return r;
}

/* ------------------------------------------------------------------------------------------
 * (f2) Thiele reconstruction, eq. (2); see zippel_ref.h for the statement.
 * Literal form: one modular inverse per inverse difference, no batching.
 * ---------------------------------------------------------------------------------------- */
int ref_thiele_reconstruct_batch(const uint64_t* points, int T, const uint64_t* vals, int64_t n, int64_t ld,
                                 uint64_t p, uint64_t* num, uint64_t* den, int32_t* degs, uint64_t* cf,
                                 int32_t* status) {
  if (!points || !vals || !num || !den || !degs || !status || T <= 0 || n <= 0 || ld < n) return REF_ERR_ARG;
  int32_t dup = 0;
  for (int j = 0; j < T && !dup; ++j)
    for (int jj = 0; jj < j; ++jj)
      if (points[j] % p == points[jj] % p) {
        dup = (int32_t)(((uint32_t)j << 8) | REF_ST_DUPLICATE_SAMPLE);
        break;
      }
  uint64_t* phi = (uint64_t*)malloc((size_t)T * sizeof(uint64_t));
  uint64_t* b = (uint64_t*)malloc((size_t)T * sizeof(uint64_t));
  uint64_t* N = (uint64_t*)calloc((size_t)T + 1, sizeof(uint64_t));
  uint64_t* D = (uint64_t*)calloc((size_t)T + 1, sizeof(uint64_t));
  uint64_t* Nn = (uint64_t*)calloc((size_t)T + 1, sizeof(uint64_t));
  for (int64_t i = 0; i < n; ++i) {
    for (int d = 0; d < T; ++d) {
      num[(int64_t)d * ld + i] = 0;
      den[(int64_t)d * ld + i] = 0;
      if (cf) cf[(int64_t)d * ld + i] = 0;
    }
    degs[i] = -1;
    degs[ld + i] = -1;
    status[i] = dup;
    if (dup) continue;
    /* inverse differences */
    for (int j = 0; j < T; ++j) phi[j] = vals[(int64_t)j * ld + i] % p;
    int K = T, bad = 0;
    b[0] = phi[0];
    for (int k = 1; k < T; ++k) {
      int zeros = 0;
      for (int j = k; j < T; ++j) zeros += (phi[j] == phi[k - 1]);
      if (zeros == T - k) {
        K = k;
        break;
      }
      if (zeros != 0) {
        bad = k;
        break;
      }
      for (int j = T - 1; j >= k; --j)
        phi[j] = ref_mulmod(ref_submod(points[j] % p, points[k - 1] % p, p),
                            ref_invmod(ref_submod(phi[j], phi[k - 1], p), p), p);
      b[k] = phi[k];
    }
    if (bad) {
      status[i] = (int32_t)(((uint32_t)bad << 8) | REF_ST_THIELE_DEGENERATE);
      continue;
    }
    if (cf)
      for (int k = 0; k < K; ++k) cf[(int64_t)k * ld + i] = b[k];
    /* expansion from the tail: (N, D) <- (b_k N + (x - x_k) D, N) */
    for (int d = 0; d <= T; ++d) N[d] = D[d] = 0;
    N[0] = b[K - 1];
    D[0] = 1 % p;
    for (int k = K - 2; k >= 0; --k) {
      const uint64_t xk = points[k] % p;
      for (int d = 0; d <= T; ++d) {
        uint64_t v = ref_mulmod(b[k], N[d], p);                       /* b_k N        */
        if (d >= 1) v = ref_addmod(v, D[d - 1], p);                   /* + x D        */
        v = ref_submod(v, ref_mulmod(xk, D[d], p), p);                /* - x_k D      */
        Nn[d] = v;
      }
      for (int d = 0; d <= T; ++d) {
        D[d] = N[d];
        N[d] = Nn[d];
      }
    }
    int dn = T, dd = T;
    while (dn >= 0 && N[dn] == 0) --dn;
    while (dd >= 0 && D[dd] == 0) --dd;
    /* D = previous N is never the zero polynomial unless f has a pole at every point: treat as degenerate */
    if (dd < 0) {
      status[i] = (int32_t)(((uint32_t)0 << 8) | REF_ST_THIELE_DEGENERATE);
      continue;
    }
    const uint64_t sc = ref_invmod(D[dd], p);
    for (int d = 0; d <= dn; ++d) num[(int64_t)d * ld + i] = ref_mulmod(N[d], sc, p);
    for (int d = 0; d <= dd; ++d) den[(int64_t)d * ld + i] = ref_mulmod(D[d], sc, p);
    degs[i] = dn;
    degs[ld + i] = dd;
  }
  free(phi);
  free(b);
  free(N);
  free(D);
  free(Nn);
  return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * (f1) skeleton extension; see zippel_ref.h.
 * ---------------------------------------------------------------------------------------- */
int ref_extend_skeleton(const uint16_t* exps, const int64_t* offsets, int F, int nv, const uint64_t* coefs, int B,
                        uint64_t p, uint16_t* new_exps, uint64_t* new_coefs, int64_t cap, int64_t* new_offsets,
                        int32_t* degs) {
  if (!exps || !offsets || !coefs || !new_exps || !new_coefs || !new_offsets || !degs || F <= 0 || nv <= 0 || B <= 0 ||
      cap < 0)
    return REF_ERR_ARG;
  const int64_t T_tot = offsets[F];
  int64_t pos = 0;
  for (int f = 0; f < F; ++f) {
    new_offsets[f] = pos;
    degs[f] = -1;
    for (int64_t i = offsets[f]; i < offsets[f + 1]; ++i)
      for (int d = 0; d < B; ++d) {
        const uint64_t v = coefs[(int64_t)d * T_tot + i] % p;
        if (v == 0) continue;
        if (pos < cap) {
          for (int j = 0; j < nv; ++j) new_exps[pos * (nv + 1) + j] = exps[i * nv + j];
          new_exps[pos * (nv + 1) + nv] = (uint16_t)d;
          new_coefs[pos] = v;
        }
        if (d > degs[f]) degs[f] = d;
        ++pos;
      }
  }
  new_offsets[F] = pos;
  return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * (f4) CRT of two primes and rational reconstruction; see zippel_ref.h.  Plain unsigned __int128.
 * ---------------------------------------------------------------------------------------- */
typedef unsigned __int128 ref_u128;
typedef __int128 ref_i128;

static ref_u128 ref_isqrt128(ref_u128 v) { /* floor(sqrt(v)) by bisection on the bits */
  ref_u128 r = 0;
  for (int b = 63; b >= 0; --b) {
    const ref_u128 c = r | ((ref_u128)1 << b);
    if (c * c <= v) r = c;
  }
  return r;
}

int ref_crt_rational_batch(const uint64_t* r1, const uint64_t* r2, int64_t n, uint64_t p1, uint64_t p2, int64_t* num,
                           int64_t* den, int32_t* status) {
  if (!r1 || !r2 || !num || !den || !status || n <= 0 || p1 == p2 || p1 < 3 || p2 < 3 || (p1 >> 63) || (p2 >> 63))
    return REF_ERR_ARG;
  const ref_u128 m = (ref_u128)p1 * p2;
  const ref_u128 N = ref_isqrt128((m - 1) / 2);
  const uint64_t p1inv = ref_invmod(p1 % p2, p2);
  for (int64_t i = 0; i < n; ++i) {
    const uint64_t a1 = r1[i] % p1, a2 = r2[i] % p2;
    const uint64_t h = ref_mulmod(ref_submod(a2, a1 % p2, p2), p1inv, p2);
    const ref_u128 x = (ref_u128)a1 + (ref_u128)p1 * h;
    ref_u128 ra = m, rb = x;
    ref_i128 ta = 0, tb = 1;
    while (rb > N) {
      const ref_u128 q = ra / rb;
      const ref_u128 rn = ra - q * rb;
      const ref_i128 tn = ta - (ref_i128)q * tb;
      ra = rb;
      rb = rn;
      ta = tb;
      tb = tn;
    }
    ref_i128 a = (ref_i128)rb, b = tb;
    if (b < 0) {
      a = -a;
      b = -b;
    }
    int ok = (b > 0) && ((ref_u128)b <= N);
    if (ok) { /* gcd(|a|, b) */
      uint64_t g0 = (uint64_t)(a < 0 ? -a : a), g1 = (uint64_t)b;
      while (g1) {
        const uint64_t tmp = g0 % g1;
        g0 = g1;
        g1 = tmp;
      }
      ok = (g0 == 1);
    }
    num[i] = ok ? (int64_t)a : 0;
    den[i] = ok ? (int64_t)b : 0;
    status[i] = ok ? 0 : REF_ST_NO_RATIONAL;
  }
  return REF_OK;
}
