// small.cuh -- one lifting step of a SMALL batch in a single launch (BASELINE.json configs[0]: one function of t = 50
// terms, B = 11 samples, where the thirteen launches of the general path cost 100 us of launch and dependency latency
// for 20 ns of arithmetic).  One CTA per function, one lane per node, the whole of PAPER.md section 1-2.2 in order:
//   (a1) m_i = prod_j y_j^e_ij                                   (L55 eq. (3))
//   (a2) M(z) = prod_i (z - m_i), product tree in shared memory   (L191)
//   (a3) q_{l-1} = M_l + m_i q_l;  d = Q_i(m_i);  num_b = sum_l q_l v_{b,l}   (L193-195; deferred sums, L205-209)
//   (a4) c_{b,i} = num_b / (d [m_i])                              (L196)
//   (a5) Newton divided differences in x_k, optional monomial expansion   (L17-22 eq. (1))
// The same exact arithmetic as the general path, so the same (unique) results bit for bit; the host takes this path
// when F <= ZP_SMALL_MAXF, every t <= ZP_SMALL_MAXT and t B is small enough for one lane per node to be the fast way
// (zippel_capi.cu: small_ok).
#pragma once
#include "kernels.cuh"

#define ZP_SMALL_MAXF 32
#define ZP_SMALL_MAXT 128
#define ZP_SMALL_NB 4    // right-hand sides per pass over the quotient chain (accumulators in registers)
#define ZP_SMALL_MAXG 3  // groups of lanes that share the right-hand sides of a function; one more group builds tables
#define ZP_SMALL_MAXB 25  // Newton's steps per level and lane: (B - 1) / LPC <= ZP_SMALL_OPS (LPC = 4 from B = 9 on, else 2)
#define ZP_SMALL_OPS 6
#define ZP_SMALL_LB 16   // Newton as a matrix (below): B <= 16 samples and t <= 64 terms
#define ZP_SMALL_LS 17   // row stride of that matrix in shared memory (odd: the four rows a warp reads lie in different banks)

struct SmallOffs {
  int64_t o[ZP_SMALL_MAXF + 1];
};

// Newton's recurrence in x_k (and the expansion to monomials, basis = 1) on ONE column of B plain values, shared by LPC
// = 2 or 4 neighbouring lanes of a warp (sub = this lane's place among them; every lane of the warp calls, `on` says
// whether the column exists): element j of the column is col[j * stride].  The steps of one level (or of one pass of
// the expansion) read the previous level only: a lane loads the operands of its (at most ZP_SMALL_OPS) steps, the warp
// meets, the lane multiplies and stores, the warp meets again -- the latency of one Montgomery product per level.
ZP_DEV void small_newton_column(uint64_t* col, int stride, int LPC, int sub, bool on, int B, int basis, const uint64_t* sInv,
                                const uint64_t* sC, const ZpMod& k) {
  const uint64_t p = k.p;
  const int D = B - 1;
  for (int l = 1; l <= D; ++l) {  // level l: c_j <- (c_j - c_{j-1}) / (x_j - x_{j-l}),  j = D .. l
    uint64_t a[ZP_SMALL_OPS], bb[ZP_SMALL_OPS];
#pragma unroll
    for (int x = 0; x < ZP_SMALL_OPS; ++x) {
      const int j = D - sub - LPC * x;
      if (on && j >= l) a[x] = col[j * stride], bb[x] = col[(j - 1) * stride];
    }
    __syncwarp();
#pragma unroll
    for (int x = 0; x < ZP_SMALL_OPS; ++x) {
      const int j = D - sub - LPC * x;
      if (on && j >= l) col[j * stride] = mont_mul(mod_sub(a[x], bb[x], p), sInv[j * B + (j - l)], k);
    }
    __syncwarp();
  }
  if (basis == 1)
    for (int j = D - 1; j >= 0; --j) {  // pass j: a_x <- a_x - c_j a_{x+1},  x = j .. D - 1
      const uint64_t cj = sC[j];
      uint64_t a[ZP_SMALL_OPS], bb[ZP_SMALL_OPS];
#pragma unroll
      for (int x = 0; x < ZP_SMALL_OPS; ++x) {
        const int e = j + sub + LPC * x;
        if (on && e < D) a[x] = col[e * stride], bb[x] = col[(e + 1) * stride];
      }
      __syncwarp();
#pragma unroll
      for (int x = 0; x < ZP_SMALL_OPS; ++x) {
        const int e = j + sub + LPC * x;
        if (on && e < D) col[e * stride] = mod_sub(a[x], mont_mul(bb[x], cj, k), p);
      }
      __syncwarp();
    }
}

// CTA = (G + 1) groups of MAXT lanes.  Lane i of group g < G owns node i and the right-hand sides [g per, (g + 1) per):
// every group runs the quotient chain of its node itself (one modular multiply-add per stage; the chain is the
// critical path, the dot products ride on it), so the B dot products of a node proceed in G lanes at once.  Group G
// meanwhile inverts Newton's sample differences and, running the chain once more without dot products, computes the
// denominators Q_i(m_i) and their inverses, which nothing needs before the columns go out.
__global__ void __launch_bounds__(ZP_SMALL_MAXT*(ZP_SMALL_MAXG + 1))
k_lift_small(const uint16_t* __restrict__ exps, SmallOffs offs, int nv, const uint64_t* __restrict__ anchors,
             const uint64_t* __restrict__ samples, int B, int G, int s0, const uint64_t* __restrict__ vals, int64_t T_tot,
             ZpMod k, int basis, uint64_t* __restrict__ out, uint64_t* __restrict__ nodes_out, int32_t* __restrict__ status) {
  __shared__ uint64_t Y[32 * 16];                  // (y_j^(2^b))~
  __shared__ uint64_t buf[2][ZP_SMALL_MAXT];       // product tree; then M~_0 .. M~_{t-1}
  __shared__ uint64_t sInv[64 * 64];               // (1 / (c_j - c_jj))~, jj < j
  __shared__ uint64_t sC[64];                      // c_j~
  __shared__ ulonglong2 sMt[ZP_SMALL_MAXT];        // {M_l, its Shoup companion}, l < t (plain residues)
  __shared__ uint64_t sDinv[ZP_SMALL_MAXT];        // (1 / (Q_i(m_i) [m_i]))~
  __shared__ uint64_t sL[ZP_SMALL_LB * ZP_SMALL_LS];  // Newton's matrix L[r][e] (plain) at sL[r LS + e]
  __shared__ int32_t s_solve, s_newton;
  extern __shared__ __align__(16) uint64_t cols[];  // [B x MAXT]: column c_{.,i} at cols[b MAXT + i]; then sv
  constexpr int S = ZP_SMALL_MAXT;
  zp_grid_dep_wait();  // (launched with programmatic stream serialization: lift_small)
  const int f = blockIdx.x;
  const int64_t off = offs.o[f];
  const int t = (int)(offs.o[f + 1] - off);
  // warp w serves group g = w div 4 and the nodes 32 q .. 32 q + 31 with q = (w + rev(g)) mod 4, rev = the two bits of g
  // swapped: the four warps of a group sit on the four schedulers (warp w runs on scheduler w mod 4), and the warps
  // with live lanes (q small when t is) of DIFFERENT groups on different ones (with q = w mod 4 a function of 50 terms
  // kept its six solving warps on two schedulers)
  const int g = threadIdx.x / S, i = 32 * (((threadIdx.x >> 5) + ((g & 1) << 1 | (g >> 1 & 1))) & 3) + (threadIdx.x & 31);
  const bool live = i < t;
  const uint64_t p = k.p;
  if (threadIdx.x == 0) s_solve = s_newton = ZP_ST_NONE;
  // ---- the function's values -> shared memory (unit-stride loads), the anchors' power table
  uint64_t* sv = cols + B * S;  // [B x MAXT]: v_{b,l} at sv[b MAXT + l]
  for (int b = g; b < B; b += G + 1)
    if (live) sv[b * S + i] = zp_canon(vals[(int64_t)b * T_tot + off + i], p);
  if (threadIdx.x < nv) {
    uint64_t y = to_mont(zp_canon(anchors[threadIdx.x], p), k);
    for (int b = 0; b < 16; ++b) {
      Y[threadIdx.x * 16 + b] = y;
      y = mont_mul(y, y, k);
    }
  }
  __syncthreads();
  if (g == G) {  // ---- the table group: Newton's inverse differences
    for (int x = i; x < B * B; x += S) {
      const int j = x / B, jj = x % B;
      const uint64_t cj = zp_canon(samples[j], p);
      if (jj == 0) sC[j] = to_mont(cj, k);
      if (jj < j) {
        const uint64_t diff = mod_sub(cj, zp_canon(samples[jj], p), p);
        if (diff == 0) atomicMin(&s_newton, (int32_t)(((uint32_t)j << 8) | ZP_ST_DUPLICATE_SAMPLE));
        sInv[x] = mont_inv(to_mont(diff, k), k);
      }
    }
  }
  // ---- (a1) node of this lane (every group computes it: no hand-over)
  uint64_t mm = 0;  // m_i~
  if (live) {
    const uint16_t* e = exps + (off + i) * nv;
    mm = k.r1;
    for (int j = 0; j < nv; ++j) {
      uint32_t ej = e[j];
      for (int b = 0; ej; ++b, ej >>= 1)
        if (ej & 1) mm = mont_mul(mm, Y[j * 16 + b], k);
    }
    if (g == 0) {
      if (nodes_out) nodes_out[off + i] = from_mont(mm, k);
      buf[0][i] = mod_neg(mm, p);  // (z - m_i)' = -m_i~
    }
  }
  // ---- (a2) product tree (as k_tree_leaf), by group 0; the barriers are the CTA's
  int cur = 0;
  for (int a = 1; a < t; a <<= 1) {
    __syncthreads();
    if (live && g == 0) {
      const int base = i & ~(2 * a - 1);
      const int b = (t - base - a) < a ? (t - base - a) : a;
      buf[cur ^ 1][i] = (b <= 0) ? buf[cur][i] : tree_merge_coef(buf[cur] + base, a, b, i - base, k);
    }
    cur ^= 1;
  }
  __syncthreads();
  if (live && g == 0) {  // M_l as a plain residue with its Shoup companion: the addend of the chain's Horner step
    const uint64_t Mm = buf[cur][i];
    sMt[i] = make_ulonglong2(from_mont(Mm, k), shoup_companion(Mm, k));
  }
  __syncthreads();
  // ---- (a3): the right-hand sides of this group, NB per pass over the chain q_{t-1} = 1, q_{l-1} = M_l + m q_l.
  // One warp or two per scheduler run this, so it is the number of instructions on the dependent path that counts:
  // the chain runs on plain residues with Shoup steps (modarith.cuh: horner_step, lazy in [0, 2p)) and the dot products
  // take the lazy q as it is (deferred sums, L205-209).  The columns are stored UNSCALED; the division (a4) by
  // d = Q(m) [m] commutes with Newton's recurrence (linear in the column) and is applied on the way out.  d and its
  // inverse are the table group's: the chain once more, without dot products, beside the solving groups.
  if (live) {
    const uint64_t m = from_mont(mm, k), mc = shoup_companion(mm, k);
    if (g < G) {
      const int per = (B + G - 1) / G, bA = g * per, bB = (bA + per < B) ? bA + per : B;
      for (int b0 = bA; b0 < bB; b0 += ZP_SMALL_NB) {
        const int nb = (bB - b0 < ZP_SMALL_NB) ? bB - b0 : ZP_SMALL_NB;
        Acc acc[ZP_SMALL_NB];
#pragma unroll
        for (int b = 0; b < ZP_SMALL_NB; ++b) acc_zero(acc[b]);
        uint64_t q = 1 % p;              // plain, lazy in [0, 2p)
        const uint64_t* v[ZP_SMALL_NB];  // rows beyond nb repeat the last one (their sums are dropped): no branch in the loop
#pragma unroll
        for (int b = 0; b < ZP_SMALL_NB; ++b) v[b] = sv + (b0 + (b < nb ? b : nb - 1)) * S;
        for (int l = t - 1; l >= 1; --l) {
#pragma unroll
          for (int b = 0; b < ZP_SMALL_NB; ++b) acc_mac(acc[b], q, v[b][l]);
          const ulonglong2 Ml = sMt[l];
          q = horner_step(q, m, mc, Ml.x, Ml.y, k);
        }
#pragma unroll
        for (int b = 0; b < ZP_SMALL_NB; ++b) acc_mac(acc[b], q, v[b][0]);
#pragma unroll
        for (int b = 0; b < ZP_SMALL_NB; ++b)
          if (b < nb)  // sum of plain x plain: redc160, then c224, give the plain sum
            cols[(b0 + b) * S + i] = mont_mul(acc_redc160(acc[b], k), k.c224, k);
      }
    } else {  // d = Q(m) = sum_l q_l m^l by Horner beside the chain: d <- d m + q
      uint64_t q = 1 % p, d = q;
      for (int l = t - 1; l >= 1; --l) {
        const ulonglong2 Ml = sMt[l];
        q = horner_step(q, m, mc, Ml.x, Ml.y, k);
        d = lazy_canon(shoup_mul_lazy(d, m, mc, k), p) + lazy_canon(q, p);
      }
      uint64_t dd = to_mont(lazy_canon(d, p), k);
      if (s0) dd = mont_mul(dd, mm, k);
      if (dd == 0) atomicMin(&s_solve, (int32_t)(((uint32_t)i << 8) | ZP_ST_DUPLICATE_NODE));
      sDinv[i] = mont_inv(dd, k);  // (1 / (d [m]))~
    }
  }
  // Newton's recurrence is linear in a column: out = L col with the B x B matrix L = Newton(identity), which depends on
  // the samples only.  Where the table group has idle warps (t <= 64: its lanes i >= 64) and the matrix is small
  // (B <= 16) they compute L beside the solve, four lanes per column of the identity, and the columns of the solve
  // then take one deferred dot product per output instead of 2 (B - 1) dependent levels.
  const bool use_L = B <= ZP_SMALL_LB && t <= 64;
  if (use_L && g == G && i >= 64) {  // (whole warps: i = 32 q + lane)
    const int ce = (i - 64) >> 2, sub = i & 3;
    const bool on = ce < B;
    for (int rr = sub; rr < B; rr += 4)
      if (on) sL[rr * ZP_SMALL_LS + ce] = (rr == ce) ? 1 % p : 0;
    __syncwarp();
    small_newton_column(sL + (on ? ce : 0), ZP_SMALL_LS, 4, sub, on, B, basis, sInv, sC, k);
  }
  __syncthreads();  // the columns, sDinv, sInv, sC, s_newton (and L) are complete
  // ---- (a5) Newton in x_k on the columns (shared memory), then the columns go out
  if (use_L) {  // out_r = sum_e L[r][e] col[e]: four lanes per column, rows r = sub (mod 4); plain x plain sums (c224)
    const int ci = threadIdx.x >> 2, sub = threadIdx.x & 3;
    const bool on = ci < t;  // 32 (G + 1) >= 64 >= t columns
    uint64_t v[ZP_SMALL_LB];
#pragma unroll
    for (int e = 0; e < ZP_SMALL_LB; ++e) v[e] = (on && e < B) ? cols[e * S + ci] : 0;
    __syncwarp();  // (the four lanes of a column have read it before any of them writes)
    Acc acc[ZP_SMALL_LB / 4];
#pragma unroll
    for (int x = 0; x < ZP_SMALL_LB / 4; ++x) acc_zero(acc[x]);
#pragma unroll
    for (int e = 0; e < ZP_SMALL_LB; ++e)
      if (e < B) {  // (uniform)
#pragma unroll
        for (int x = 0; x < ZP_SMALL_LB / 4; ++x)
          if (sub + 4 * x < B) acc_mac(acc[x], sL[(sub + 4 * x) * ZP_SMALL_LS + e], v[e]);
      }
#pragma unroll
    for (int x = 0; x < ZP_SMALL_LB / 4; ++x)
      if (on && sub + 4 * x < B) cols[(sub + 4 * x) * S + ci] = mont_mul(acc_redc160(acc[x], k), k.c224, k);
  } else {  // the recurrence itself, shared among LPC lanes per column (all the CTA's lanes work: 128 (G + 1) >= 128 LPC)
    const int LPC = (G + 1 >= 4) ? 4 : 2;  // G >= 1
    const int ci = threadIdx.x / LPC, sub = threadIdx.x % LPC;
    const bool on = ci < t;
    small_newton_column(cols + (on ? ci : 0), S, LPC, sub, on, B, basis, sInv, sC, k);
  }
  __syncthreads();
  for (int b = g; b < B; b += G + 1)
    if (live) out[(int64_t)b * T_tot + off + i] = mont_mul(cols[b * S + i], sDinv[i], k);  // (a4): plain x Montgomery
  if (threadIdx.x == 0) {
    const int32_t s = (s_solve != ZP_ST_NONE) ? s_solve : s_newton;
    status[f] = (s == ZP_ST_NONE) ? 0 : s;
  }
}
