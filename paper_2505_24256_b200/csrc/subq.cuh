// subq.cuh -- sub-quadratic transposed Vandermonde solve for long skeletons (PAPER.md L37, L250-254,
// Table 3: 125k .. 4.8m monomials).  Same answer as the quadratic route of section 2.2 (the solution is unique,
// reading G21); the operations are reorganised around products of polynomials (ntt.cuh):
//
//   sum_s v_s z^-(s+1) = sum_i c_i / (z - m_i) = N(z) / M(z),  N(m_i) = c_i M'(m_i)   (G15),
//
// so the right-hand side v IS the tail of N / M at infinity.  For a block S of nodes with master polynomial M_S write
// tail_S(P) = the first |S| coefficients of z^-1, z^-2, .. in P / M_S.  Then
//   (up)    M_{L u R} = M_L M_R                                        -- product tree above the 1024-node leaves
//   (down)  tail_L(P)_k = sum_j (M_R)_j tail_{L u R}(P)_{k+j}          -- a correlation with the SIBLING's polynomial
//           (because P / M_L = M_R * P / M_{L u R}, and the polynomial part contributes nothing to the tail)
//   (leaf)  sum_l q_{i,l} tail_S(P)_l = (P mod M_S)(m_i)               -- the synthetic-division dot of (a3), unscaled
// For P = N the root tail is v itself; for P = M' it is the power sums of the nodes, rev(M') / rev(M) mod x^t, which
// needs one power-series inverse of rev(M) (Newton iteration).  Finally c_i = N(m_i) / M'(m_i) [/ m_i if s0 = 1].
// Every product is a cyclic convolution of length 2a at block size a (ntt.cuh); the leaf step runs the existing
// k_node_solve on the leaves as if they were functions, with B + 1 right-hand sides (the values and the M' tail).
//
// Storage: a monic polynomial of degree n is kept WITHOUT its leading 1, as n Montgomery coefficients in the slots of
// the nodes it covers (as in k_tree_leaf); level l holds the polynomials of the blocks of LEAF 2^l nodes.  Tails are
// plain residues in the same slots.  All indices below are local to a "run" of consecutive long functions.
#pragma once
#include "ntt.cuh"

struct SqTask {
  int64_t base;  // first slot of the left block
  int32_t a;     // left block length (pairs: the level's block size; copies: the length to copy)
  int32_t b;     // right block length (>= 1); 0 marks a copy task
};

// ---- (up) ---------------------------------------------------------------------------------------------------------------
// The product of a pair is taken on the REVERSED children (k_sq_down_prepx below fills X: rev(A') rev(B') = rev(A' B'),
// degree a + b - 2), because their transforms are what the down-tree needs again: O[t][i] = (A' B')_{a+b-2-i}.
// C' = A' B' + z^a B' + z^b A'  (Montgomery in, Montgomery out: co carries K = 2^-64)
__global__ void __launch_bounds__(256)
k_sq_up_fin(const uint64_t* __restrict__ lev, const SqTask* __restrict__ tasks, int64_t P, int logn,
            const uint64_t* __restrict__ O, int64_t EO, NttCtx cx, CrtOut co, ZpMod kp, uint64_t* __restrict__ nxt) {
  zp_grid_dep_wait();
  const int64_t n = (int64_t)1 << logn;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EO; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t c = e & (n - 1);
    const SqTask t = tasks[e >> logn];
    if (c >= t.a + t.b) continue;
    uint64_t r = 0;
    if (c <= t.a + t.b - 2) {
      const int64_t src = e - c + (t.a + t.b - 2 - c);
      r = ntt_crt(O[src], O[EO + src], O[2 * EO + src], cx, co, kp);
    }
    if (c >= t.a) r = mod_add(r, lev[t.base + t.a + (c - t.a)], kp.p);
    if (c >= t.b) r = mod_add(r, lev[t.base + (c - t.b)], kp.p);
    nxt[t.base + c] = r;
  }
}
// blocks without a sibling pass through: dst[v ld + slot] = src[v ld + slot]
__global__ void __launch_bounds__(256)
k_sq_copy(const SqTask* __restrict__ tasks, int ntasks, const uint64_t* __restrict__ src, uint64_t* __restrict__ dst, int V,
          int64_t ld) {
  zp_grid_dep_wait();
  for (int x = blockIdx.y; x < ntasks * V; x += gridDim.y) {
    const SqTask t = tasks[x % ntasks];
    const int64_t o = (int64_t)(x / ntasks) * ld + t.base;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < t.a; i += gridDim.x * blockDim.x) dst[o + i] = src[o + i];
  }
}

// ---- (down) -------------------------------------------------------------------------------------------------------------
// X[j][2t][i] = A'_{a-1-i}, X[j][2t+1][i] = B'_{b-1-i}  (the reversed children), n = 2a
__global__ void __launch_bounds__(256)
k_sq_down_prepx(const uint64_t* __restrict__ lev, const SqTask* __restrict__ tasks, int64_t P, int logn,
                uint64_t* __restrict__ X, int64_t EX) {
  zp_grid_dep_wait();
  const int64_t n = (int64_t)1 << logn;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EX; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t seg = e >> logn, i = e & (n - 1);
    const SqTask t = tasks[seg >> 1];
    uint64_t v = 0;
    if (seg & 1) {
      if (i < t.b) v = lev[t.base + t.a + t.b - 1 - i];
    } else {
      if (i < t.a) v = lev[t.base + t.a - 1 - i];
    }
    X[e] = v;
    X[EX + e] = v;
    X[2 * EX + e] = v;
  }
}
// Y[j][v P + t][i] = tail_{L u R}(P_v)_i, i < a + b  (copies = 1: one copy serves the three primes, n <= 4096)
__global__ void __launch_bounds__(256)
k_sq_down_prepy(const uint64_t* __restrict__ cur, int64_t ld, const SqTask* __restrict__ tasks, int64_t P, int logn,
                uint64_t* __restrict__ Y, int64_t EY, int copies) {
  zp_grid_dep_wait();
  const int64_t n = (int64_t)1 << logn;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EY; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t seg = e >> logn, i = e & (n - 1);
    const int64_t v = (int64_t)((uint32_t)seg / (uint32_t)P);  // (segments of a launch: < 2^31)
    const SqTask t = tasks[seg - v * P];
    const uint64_t x = (i < t.a + t.b) ? cur[v * ld + t.base + i] : 0;
    Y[e] = x;
    if (copies == 3) {  // the strided passes of a long transform work in place, per prime
      Y[EY + e] = x;
      Y[2 * EY + e] = x;
    }
  }
}
// O segment o = (v P + t) 2 + side.  side 0: tail_L_k = c_{k+b} + (rev(B') * c)_{k+b-1}, k < a;
//                                    side 1: tail_R_k = c_{k+a} + (rev(A') * c)_{k+a-1}, k < b.
__global__ void __launch_bounds__(256)
k_sq_down_fin(const uint64_t* __restrict__ cur, int64_t ld, const SqTask* __restrict__ tasks, int64_t P, int logn,
              const uint64_t* __restrict__ O, int64_t EO, NttCtx cx, CrtOut co, ZpMod kp, uint64_t* __restrict__ nxt) {
  zp_grid_dep_wait();
  const int64_t h = (int64_t)1 << (logn - 1);  // a tail is at most half a segment long (b <= a = n / 2): lanes over (o, k < n / 2)
  for (int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; x < EO / 2; x += (int64_t)gridDim.x * blockDim.x) {
    const int64_t o = x >> (logn - 1), k = x & (h - 1);
    const int side = (int)(o & 1);
    const int64_t vt = o >> 1, v = (int64_t)((uint32_t)vt / (uint32_t)P);
    const SqTask t = tasks[vt - v * P];
    const int64_t len = side ? t.b : t.a, sh = side ? t.a : t.b;  // own length, sibling's length
    if (k >= len) continue;
    const int64_t src = (o << logn) + (k + sh - 1);
    const uint64_t r = ntt_crt(O[src], O[EO + src], O[2 * EO + src], cx, co, kp);
    const uint64_t* c = cur + v * ld + t.base;
    nxt[v * ld + t.base + (side ? t.a : 0) + k] = mod_add(r, c[k + sh], kp.p);
  }
}

// ---- power-series inverse of f = rev(M):  f_0 = 1, f_i = M_{t-i} (i <= t), 0 beyond -------------------------------------
// All the functions of a run go through the iteration together (one segment, or pair of segments, per function and
// step).  SqFn describes a function; the host sorts the array by t, longest first, so that the functions still
// iterating at precision k (t > k) are a prefix of it.
struct SqFn {
  int64_t moff;  // slot of the function's first node in the run: its top-level polynomial and its tails start there
  int64_t aoff;  // first word of its inverse series alpha in the alpha buffer (room for its final precision)
  int64_t t;
};
ZP_DEV uint64_t sq_f(const uint64_t* __restrict__ Mtop, int64_t t, int64_t i, const ZpMod& kp) {  // Montgomery
  return i == 0 ? kp.r1 : (i <= t ? Mtop[t - i] : 0);
}
// base case: alpha = 1 / f mod x^KB by Newton steps with schoolbook products in shared memory, one CTA per function
#define ZP_SQ_KB 1024
__global__ void __launch_bounds__(512)
k_sq_inv_base(const uint64_t* __restrict__ top, const SqFn* __restrict__ fns, ZpMod kp, uint64_t* __restrict__ alphas) {
  __shared__ uint64_t f[ZP_SQ_KB], g[ZP_SQ_KB], ev[ZP_SQ_KB / 2];
  const SqFn fn = fns[blockIdx.x];
  const uint64_t* Mtop = top + fn.moff;
  uint64_t* alpha = alphas + fn.aoff;
  for (int i = threadIdx.x; i < ZP_SQ_KB; i += blockDim.x) {
    f[i] = sq_f(Mtop, fn.t, i, kp);
    g[i] = 0;
  }
  __syncthreads();
  if (threadIdx.x == 0) g[0] = kp.r1;
  __syncthreads();
  for (int k = 1; k < ZP_SQ_KB; k <<= 1) {
    // e_i = (f g)_{k+i} = sum_{j<k} f_{k+i-j} g_j,  i < k
    for (int i = threadIdx.x; i < k; i += blockDim.x) {
      Acc acc;
      acc_zero(acc);
      for (int j = 0; j < k; ++j) acc_mac(acc, f[k + i - j], g[j]);
      ev[i] = mont_mul(acc_redc160(acc, kp), kp.c160, kp);
    }
    __syncthreads();
    // g_{k+i} = -(g e)_i = -sum_{j<=i} g_j e_{i-j}
    for (int i = threadIdx.x; i < k; i += blockDim.x) {
      Acc acc;
      acc_zero(acc);
      for (int j = 0; j <= i; ++j) acc_mac(acc, g[j], ev[i - j]);
      g[k + i] = mod_neg(mont_mul(acc_redc160(acc, kp), kp.c160, kp), kp.p);
    }
    __syncthreads();
  }
  for (int i = threadIdx.x; i < ZP_SQ_KB; i += blockDim.x) alpha[i] = g[i];
}
// Newton step k -> 2k (n = 2k) for the first nact functions, first product: X[2s] = f_s mod x^2k, X[2s+1] = alpha_s mod x^k
__global__ void __launch_bounds__(256)
k_sq_newton_prep1(const uint64_t* __restrict__ top, const SqFn* __restrict__ fns, int64_t nact, const uint64_t* __restrict__ alphas,
                  int logn, ZpMod kp, uint64_t* __restrict__ X) {
  zp_grid_dep_wait();
  const int64_t n = (int64_t)1 << logn, EX = 2 * nact * n, k = n >> 1;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EX; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t seg = e >> logn, i = e & (n - 1);
    const SqFn fn = fns[seg >> 1];
    const uint64_t v = (seg & 1) ? (i < k ? alphas[fn.aoff + i] : 0) : sq_f(top + fn.moff, fn.t, i, kp);
    X[e] = v;
    X[EX + e] = v;
    X[2 * EX + e] = v;
  }
}
// second product of the step: X[2s][i] = e_i = (f alpha)_{k+i}, i < k (O = inverse transforms of the first products),
// X[2s+1][i] = alpha_i, i < k, both zero-padded to n
__global__ void __launch_bounds__(256)
k_sq_newton_mid(const uint64_t* __restrict__ O, const SqFn* __restrict__ fns, int64_t nact, int logn, NttCtx cx, CrtOut co,
                ZpMod kp, const uint64_t* __restrict__ alphas, uint64_t* __restrict__ X) {
  zp_grid_dep_wait();
  const int64_t n = (int64_t)1 << logn, k = n >> 1, EX = 2 * nact * n, EO = nact * n;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EX; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t seg = e >> logn, i = e & (n - 1), s = seg >> 1;
    uint64_t v = 0;
    if (i < k) {
      const int64_t o = s * n + k + i;
      v = (seg & 1) ? alphas[fns[s].aoff + i] : ntt_crt(O[o], O[EO + o], O[2 * EO + o], cx, co, kp);
    }
    X[e] = v;
    X[EX + e] = v;
    X[2 * EX + e] = v;
  }
}
// alpha_{k+i} = -(alpha e)_i, i < k
__global__ void __launch_bounds__(256)
k_sq_newton_fin(const uint64_t* __restrict__ O, const SqFn* __restrict__ fns, int64_t nact, int logn, NttCtx cx, CrtOut co,
                ZpMod kp, uint64_t* __restrict__ alphas) {
  zp_grid_dep_wait();
  const int64_t n = (int64_t)1 << logn, k = n >> 1, EO = nact * n;
  for (int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; x < nact * k; x += (int64_t)gridDim.x * blockDim.x) {
    const int64_t s = x >> (logn - 1), i = x - s * k, o = s * n + i;
    alphas[fns[s].aoff + k + i] = mod_neg(ntt_crt(O[o], O[EO + o], O[2 * EO + o], cx, co, kp), kp.p);
  }
}
// root tails of M' for the functions fns[g0 .. g0 + ng), which share the product length n >= 2t:
// X[2s][i] = rev(M')_i = (t - i) f_i, X[2s+1][i] = alpha_i, i < t, zero-padded to n
__global__ void __launch_bounds__(256)
k_sq_root_prep(const uint64_t* __restrict__ top, const SqFn* __restrict__ fns, int64_t ng, const uint64_t* __restrict__ alphas,
               int logn, ZpMod kp, uint64_t* __restrict__ X) {
  zp_grid_dep_wait();
  const int64_t n = (int64_t)1 << logn, EX = 2 * ng * n;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EX; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t seg = e >> logn, i = e & (n - 1);
    const SqFn fn = fns[seg >> 1];
    uint64_t v = 0;
    if (i < fn.t)
      v = (seg & 1) ? alphas[fn.aoff + i]
                    : mont_mul(sq_f(top + fn.moff, fn.t, i, kp), to_mont(zp_canon((uint64_t)(fn.t - i), kp.p), kp), kp);
    X[e] = v;
    X[EX + e] = v;
    X[2 * EX + e] = v;
  }
}
// tail_k = (rev(M') alpha)_k, k < t: the power sums of the nodes, plain (co carries K = 2^-128); tails: the M' row of the run
__global__ void __launch_bounds__(256)
k_sq_root_fin(const uint64_t* __restrict__ O, const SqFn* __restrict__ fns, int64_t ng, int logn, NttCtx cx, CrtOut co, ZpMod kp,
              uint64_t* __restrict__ tails) {
  zp_grid_dep_wait();
  const int64_t n = (int64_t)1 << logn, EO = ng * n;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EO; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t s = e >> logn, i = e & (n - 1);
    const SqFn fn = fns[s];
    if (i < fn.t) tails[fn.moff + i] = ntt_crt(O[e], O[EO + e], O[2 * EO + e], cx, co, kp);
  }
}
// root tails of the right-hand sides: the values themselves (canonicalised, reading G22)
__global__ void __launch_bounds__(256)
k_sq_load_vals(const uint64_t* __restrict__ vals, int64_t ldv, int B, int64_t T, ZpMod kp, uint64_t* __restrict__ tails,
               int64_t ld) {
  for (int b = blockIdx.y; b < B; b += gridDim.y)
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < T; i += (int64_t)gridDim.x * blockDim.x)
      tails[b * ld + i] = zp_canon(vals[b * ldv + i], kp.p);
}
__global__ void k_fill_u64(uint64_t* x, int64_t n, uint64_t v) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) x[i] = v;
}
