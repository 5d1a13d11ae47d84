// ntt.cuh -- exact polynomial products over Z/pZ for a 63-bit p (skeletons
// "measured in millions" of terms, where the t^2 master polynomial and per-node division of section 2.2 stop being
// affordable).  p - 1 = 2 * 3^4 * 17 * 23 * ... has no power-of-two factor, so there is no NTT modulo p itself: a
// product of two polynomials with coefficients in [0, p) is computed as an INTEGER cyclic convolution modulo three
// NTT-friendly primes q1 > q2 > q3 just below 2^62 (q = c 2^26 + 1), recombined by Garner's CRT and reduced
// modulo p.  Bound: a coefficient of the integer product is < 2^23 * p^2 < 2^149 < q1 q2 q3 ~ 2^186 (transform lengths
// up to 2^24, at most 2^23 non-zero terms per operand).
//
// Transform (per prime, length n = 2^k <= 2^24), "modulus splitting" Cooley-Tukey: stage M = 1, 2, .., n/2 splits
// each of the M residue blocks  a mod (x^(n/M) - rho_i)  into  mod (x^(n/2M) -/+ sqrt(rho_i)):
//     (u, v) -> (u + r_i v, u - r_i v),   r_i = U[M + i] = w_{2M}^{brev(i)}      (natural order in, bit-reversed out),
// so a stage reads ONE contiguous slice U[M .. 2M) of a table that does not depend on n, and all butterflies of a
// block share their twiddle (warp-uniform or unit-stride reads).  The inverse runs the stages backwards with
// Gentleman-Sande butterflies (u + v, (u - v) r_i^-1); the factor 1/n is folded into the pointwise product.
// Values stay lazy (Harvey): forward in [0, 4q), inverse in [0, 2q); every twiddle product is a Shoup multiply-add
// with a zero addend (modarith.cuh horner_step: any 64-bit x in, [0, 2q) out), which needs q < 2^62.
//
// Lengths above 4096 take two or three passes over the buffer (L2 / HBM): strided passes do the first stages on
// columns of an [R x L] view (a CTA owns G consecutive columns: coalesced rows of G words), then every row c is an
// independent cyclic transform of length L once its elements j are twisted by w_n^(brev(c) j) (the substitution
// x -> theta_c x that turns  mod (x^L - rho_c)  into  mod (x^L - 1)); the twist rides on the next pass's load
// (forward) or store (inverse) and takes its factor from two 4096-entry tables: w^E = Thi[E >> 12] * Tlo[E & 4095].
#pragma once
#include "modarith.cuh"

#define ZP_NTT_LOGMAX 24   // longest transform 2^24; the root w has order 2^24
#define ZP_NTT_TAB 4096    // entries per table
#define ZP_NTT_LOGC 12     // a CTA transforms chunks of 4096 words in shared memory
#define ZP_NTT_C (1 << ZP_NTT_LOGC)
#define ZP_NTT_THREADS 256      // lanes per CTA for full grids
#define ZP_NTT_THREADS_SMALL 512  // for grids that leave SMs idle: one group per lane and round, half the latency

struct NttCtx {
  ZpMod q[3];
  const ulonglong2* U[3];    // [4096] U[M + i] = { r, r' }, r = w_{2M}^{brev_{log M}(i)} plain, r' its Shoup companion
  const ulonglong2* Ui[3];   // [4096] the inverses r^-1
  const ulonglong2* Tlo[3];  // [4096] w^i            (w of order 2^24)
  const ulonglong2* Thi[3];  // [4096] w^(4096 i)
  uint64_t g2;               // Garner: (q1^-1 mod q2) 2^64 mod q2
  uint64_t g3a;              //         (q1 mod q3) 2^64 mod q3
  uint64_t g3b;              //         ((q1 q2)^-1 mod q3) 2^64 mod q3
};
// c K mod p for the integer c recovered by the CRT:  mont_mul_p(k1, C1) + mont_mul_p(k2, C2) + mont_mul_p(k3, C3)
struct CrtOut {
  uint64_t C1, C2, C3;  // K 2^64, q1 K 2^64, q1 q2 K 2^64  (mod p)
};

#if defined(__CUDACC__)
// x * w mod q, lazily: any 64-bit x in, [0, 2q) out (w = {w, w'} with its Shoup companion; modarith.cuh)
ZP_DEV uint64_t ntt_mul(uint64_t x, ulonglong2 w, const ZpMod& q) { return shoup_mul_lazy(x, w.x, w.y, q); }
ZP_DEV uint32_t brev_bits(uint32_t x, int bits) { return bits ? (__brev(x) >> (32 - bits)) : 0u; }

// x * w^E (forward) or x * w^-E (inverse), E < 2^24, from the two-level tables
template <bool INV>
ZP_DEV uint64_t ntt_twist(uint64_t x, uint32_t E, const ulonglong2* __restrict__ Tlo, const ulonglong2* __restrict__ Thi,
                          const ZpMod& q) {
  if (INV) E = ((1u << ZP_NTT_LOGMAX) - E) & ((1u << ZP_NTT_LOGMAX) - 1);
  x = ntt_mul(x, __ldg(Thi + (E >> 12)), q);
  return ntt_mul(x, __ldg(Tlo + (E & 4095)), q);
}

// ---- tables: one thread per entry ------------------------------------------------------------------------------
// which = 0: U, 1: Ui, 2: Tlo, 3: Thi.  wroot = the 2^24-th root of unity of this prime in Montgomery form.
__global__ void k_ntt_tables(ZpMod q, uint64_t wroot_mont, ulonglong2* U, ulonglong2* Ui, ulonglong2* Tlo, ulonglong2* Thi) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 4 * ZP_NTT_TAB) return;
  const int which = idx / ZP_NTT_TAB, i = idx % ZP_NTT_TAB;
  uint64_t e;  // exponent of w
  if (which <= 1) {
    if (i == 0) {
      e = 0;
    } else {
      const int lm = 31 - __clz(i);  // M = 2^lm, block i - M
      const uint32_t b = brev_bits((uint32_t)(i - (1 << lm)), lm);
      e = (uint64_t)b << (ZP_NTT_LOGMAX - 1 - lm);  // w_{2M} = w^(2^24 / 2M)
      if (which == 1) e = ((1ull << ZP_NTT_LOGMAX) - e) & ((1ull << ZP_NTT_LOGMAX) - 1);
    }
  } else {
    e = (which == 2) ? (uint64_t)i : (uint64_t)i << 12;
  }
  const uint64_t wm = mont_pow(wroot_mont, e, q);
  const ulonglong2 r = make_ulonglong2(from_mont(wm, q), shoup_companion(wm, q));
  (which == 0 ? U : which == 1 ? Ui : which == 2 ? Tlo : Thi)[i] = r;
}

// ---- the CTA-level transform: a tile of 4096 words in shared memory, radix-8 rounds in registers ---------------------
// A CTA works on a tile of 4096 words e (12 bits).  A pass runs the stages that act on the bits hi .. lo of e (hi >= lo;
// forward from hi down, inverse from lo up); the stage on bit b pairs e with e + 2^b and uses the twiddle U[2^ls + i],
// ls = hi - b, i = the bits hi .. b+1 of e (the block the pair lies in).  The stages are taken three at a time: in the
// round of field f (bits 3f+2 .. 3f) a lane loads the 8 words of a group that differ in that field only, runs up to three
// stages on them in registers and writes them back -- one load and one store of shared memory per word and round
// instead of one per word and stage, in a loop over the rounds (the code stays small: the butterfly is ~30
// instructions that fill the multiplier pipe and the issue slots alike, so instruction fetch and every extra instruction
// count).  512 groups per round, two per lane.  Shared memory holds word e at e ^ ((e >> 3) & 15): conflict-free for
// 64-bit accesses in all four rounds and for unit-stride staging.
#define ZP_NTT_SMEM ZP_NTT_C
ZP_DEV int ntt_pad(int e) { return e ^ ((e >> 3) & 15); }
// first word of group gidx (9 bits) in the round whose field starts at bit sh: the field bits are zero
ZP_DEV int ntt_gbase(int gidx, int sh) { return ((gidx >> sh) << (sh + 3)) | (gidx & ((1 << sh) - 1)); }

// the twiddles of the (up to three) stages of the field at bit sh for the group whose first word is eb: slot 4 >> bb ..
// of stage bb holds its 4 >> bb entries (w[1]: stage 2; w[2..3]: stage 1; w[4..7]: stage 0); stages outside [lo, hi] load
// nothing.  Issued before the words of the group are read, so that the two latencies overlap.
ZP_DEV void ntt_group_twiddles(ulonglong2 (&w)[8], int eb, int sh, int hi, int bmax, int lo, const ulonglong2* __restrict__ tab) {
#pragma unroll
  for (int bb = 2; bb >= 0; --bb) {
    const int b = sh + bb;
    if (b > bmax || b < lo) continue;  // uniform
    const int ls = hi - b, mask = (1 << ls) - 1;
    const int ihi = (eb >> (sh + 3)) << (2 - bb);  // the block bits above the field; j's bits above bb fill the rest
#pragma unroll
    for (int k = 0; k < (4 >> bb); ++k) w[(4 >> bb) + k] = __ldg(tab + (1 << ls) + ((ihi | k) & mask));
  }
}
// the forward stages of one field on one group (values in [0, 4q), Harvey butterflies)
ZP_DEV void ntt_group_fwd(uint64_t (&x)[8], const ulonglong2 (&w)[8], int sh, int bmax, int lo, const ZpMod& q) {
  const uint64_t q2 = 2 * q.p;
#pragma unroll
  for (int bb = 2; bb >= 0; --bb) {
    const int b = sh + bb;
    if (b > bmax || b < lo) continue;  // uniform
#pragma unroll
    for (int j0 = 0; j0 < 8; ++j0) {
      if (j0 >> bb & 1) continue;
      const int j1 = j0 | (1 << bb);
      uint64_t u = x[j0];
      u = (u >= q2) ? u - q2 : u;
      const uint64_t v = ntt_mul(x[j1], w[(4 >> bb) + (j0 >> (bb + 1))], q);
      x[j0] = u + v;
      x[j1] = u - v + q2;
    }
  }
}
// inverse: values in [0, 2q), Gentleman-Sande butterflies with the inverse twiddles
ZP_DEV void ntt_group_inv(uint64_t (&x)[8], const ulonglong2 (&w)[8], int sh, int bmax, int lo, const ZpMod& q) {
  const uint64_t q2 = 2 * q.p;
#pragma unroll
  for (int bb = 0; bb < 3; ++bb) {
    const int b = sh + bb;
    if (b > bmax || b < lo) continue;  // uniform
#pragma unroll
    for (int j0 = 0; j0 < 8; ++j0) {
      if (j0 >> bb & 1) continue;
      const int j1 = j0 | (1 << bb);
      const uint64_t u = x[j0], v = x[j1];
      const uint64_t sum = u + v;
      x[j0] = (sum >= q2) ? sum - q2 : sum;
      x[j1] = ntt_mul(u - v + q2, w[(4 >> bb) + (j0 >> (bb + 1))], q);
    }
  }
}
// The stages on the top three bits 11 .. 9 of the tile index run in the registers of the lane that loads (forward) or
// stores (inverse) the words: lane T moves the words e = T + TH m, so with TH <= 512 those bits are bits of m, the pairs
// of such a stage are pairs of the lane's own words, and the twiddle depends on m only (the same for every lane).  A
// lane takes its words eight at a time (those that differ in the bits 11 .. 9 only: e = T + TH h + 512 mm, mm = 0 .. 7,
// h < 512 / TH).  One round trip through shared memory and one barrier less per tile transform than four rounds there.
#define ZP_NTT_TOPBIT 9
template <int TH>
ZP_DEV int ntt_top_word(int h, int mm) { return threadIdx.x + TH * h + 512 * mm; }
ZP_DEV void ntt_top_fwd(uint64_t (&x)[8], int hi, int lo, const ulonglong2* __restrict__ U, const ZpMod& q) {
  const uint64_t q2 = 2 * q.p;
#pragma unroll
  for (int bb = 2; bb >= 0; --bb) {
    const int b = ZP_NTT_TOPBIT + bb;
    if (b > hi || b < lo) continue;  // uniform
    const int ls = hi - b, mask = (1 << ls) - 1;
#pragma unroll
    for (int k = 0; k < (4 >> bb); ++k) {  // the blocks of this stage among the lane's words
      const ulonglong2 w = __ldg(U + (1 << ls) + (k & mask));
#pragma unroll
      for (int jl = 0; jl < (1 << bb); ++jl) {
        const int m0 = (k << (bb + 1)) | jl, m1 = m0 | (1 << bb);
        uint64_t u = x[m0];
        u = (u >= q2) ? u - q2 : u;
        const uint64_t v = ntt_mul(x[m1], w, q);
        x[m0] = u + v;
        x[m1] = u - v + q2;
      }
    }
  }
}
ZP_DEV void ntt_top_inv(uint64_t (&x)[8], int hi, int lo, const ulonglong2* __restrict__ Ui, const ZpMod& q) {
  const uint64_t q2 = 2 * q.p;
#pragma unroll
  for (int bb = 0; bb < 3; ++bb) {
    const int b = ZP_NTT_TOPBIT + bb;
    if (b > hi || b < lo) continue;  // uniform
    const int ls = hi - b, mask = (1 << ls) - 1;
#pragma unroll
    for (int k = 0; k < (4 >> bb); ++k) {
      const ulonglong2 w = __ldg(Ui + (1 << ls) + (k & mask));
#pragma unroll
      for (int jl = 0; jl < (1 << bb); ++jl) {
        const int m0 = (k << (bb + 1)) | jl, m1 = m0 | (1 << bb);
        const uint64_t u = x[m0], v = x[m1];
        const uint64_t sum = u + v;
        x[m0] = (sum >= q2) ? sum - q2 : sum;
        x[m1] = ntt_mul(u - v + q2, w, q);
      }
    }
  }
}
// the stages of [lo, hi] BELOW bit 9 on the tile in shared memory, three per round (the tile is complete and
// visible on entry and on exit); hi is still the pass's top bit: it fixes the twiddle level of every stage
template <bool INV, int TH>
ZP_DEV void ntt_tile(uint64_t* sm, int hi, int lo, const ulonglong2* __restrict__ tab, const ZpMod& q) {
  const int bmax = hi < ZP_NTT_TOPBIT - 1 ? hi : ZP_NTT_TOPBIT - 1;
#pragma unroll 1
  for (int r = 0; r < 3; ++r) {
    const int f = INV ? r : 2 - r, sh = 3 * f;
    if (sh > bmax || sh + 2 < lo) continue;  // no stage in this field
#pragma unroll 1
    for (int g = 0; g < ZP_NTT_C / 8 / TH; ++g) {
      const int eb = ntt_gbase(threadIdx.x + TH * g, sh);
      ulonglong2 w[8];
      ntt_group_twiddles(w, eb, sh, hi, bmax, lo, tab);
      uint64_t x[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) x[j] = sm[ntt_pad(eb + (j << sh))];
      if (INV) ntt_group_inv(x, w, sh, bmax, lo, q);
      else ntt_group_fwd(x, w, sh, bmax, lo, q);
#pragma unroll
      for (int j = 0; j < 8; ++j) sm[ntt_pad(eb + (j << sh))] = x[j];
    }
    __syncthreads();
  }
}

// ---- one pass over a buffer: every CTA transforms one tile of 4096 words of one prime ---------------------------
// buf: [3][E] words (prime-major), E = words per prime.  Two kinds of tile:
//   chunk (logR = 0):  4096 consecutive words = 4096 / ln complete transforms of length ln = 2^logn <= 4096 (a whole
//                      transform, or the rows of the last pass of a longer one): the stages on the bits logn-1 .. 0;
//   strided (logR > 0): the first logR stages of a transform of length n = 2^logn on its [R x L] view (L = n / R): the
//                      tile is R rows x G = 4096 / R consecutive columns, word e = r G + c: the stages on the bits
//                      11 .. 12 - logR.  R <= 512 (rows of G >= 8 words).
// logRp > 0: the transforms are the rows of parents of length 2^(logn + logRp); row c's element j is twisted by
// w_parent^(brev(c) j) on load (forward) / by its inverse on store (inverse).
template <bool INV, int TH>
__global__ void __launch_bounds__(TH, 1024 / TH)
k_ntt_pass(uint64_t* __restrict__ buf, int64_t E, int logn, int logR, int logRp, NttCtx cx) {
  zp_grid_dep_wait();
  __shared__ uint64_t sm[ZP_NTT_SMEM];
  const int jp = blockIdx.y;
  const ZpMod q = cx.q[jp];
  const int T = threadIdx.x;
  uint64_t* g = buf + (int64_t)jp * E;
  const int lpar = logn + logRp;
  // word e of the tile <-> offset into g: base + ((e >> logG) << rowshift) + (e & (G - 1))
  int64_t base;
  int logG, rowshift;
  if (logR == 0) {
    base = (int64_t)blockIdx.x * ZP_NTT_C;
    logG = ZP_NTT_LOGC;
    rowshift = 0;
  } else {
    const int logL = logn - logR;
    logG = ZP_NTT_LOGC - logR;
    const int tiles_log = logL - logG;  // column tiles per transform
    const int64_t tr = (int64_t)blockIdx.x >> tiles_log;
    const int col0 = (int)(blockIdx.x & ((1 << tiles_log) - 1)) << logG;
    base = (tr << logn) + col0;
    rowshift = logL;
    if ((tr << logn) >= E) return;
  }
  const int G1 = (1 << logG) - 1;
  const int ln1 = (1 << logn) - 1;
  const int hi = logR ? 11 : logn - 1, lo = logR ? 12 - logR : 0;
  uint64_t x[8];
  if (!INV) {
#pragma unroll 1
    for (int h = 0; h < 512 / TH; ++h) {
#pragma unroll
      for (int mm = 0; mm < 8; ++mm) {
        const int e = ntt_top_word<TH>(h, mm);
        const int64_t off = base + ((int64_t)(e >> logG) << rowshift) + (e & G1);
        uint64_t v = 0;
        if (off < E) {
          v = g[off];
          if (logRp) {
            const uint32_t c = (uint32_t)((off >> logn) & ((1 << logRp) - 1)), pos = (uint32_t)(off & ln1);
            v = ntt_twist<false>(v, (brev_bits(c, logRp) * pos) << (ZP_NTT_LOGMAX - lpar), cx.Tlo[jp], cx.Thi[jp], q);
          }
        }
        x[mm] = v;
      }
      ntt_top_fwd(x, hi, lo, cx.U[jp], q);
#pragma unroll
      for (int mm = 0; mm < 8; ++mm) sm[ntt_pad(ntt_top_word<TH>(h, mm))] = x[mm];
    }
    __syncthreads();
    ntt_tile<false, TH>(sm, hi, lo, cx.U[jp], q);
#pragma unroll 4
    for (int m = 0; m < ZP_NTT_C / TH; ++m) {
      const int e = T + TH * m;
      const int64_t off = base + ((int64_t)(e >> logG) << rowshift) + (e & G1);
      if (off < E) g[off] = sm[ntt_pad(e)];
    }
  } else {
#pragma unroll 4
    for (int m = 0; m < ZP_NTT_C / TH; ++m) {
      const int e = T + TH * m;
      const int64_t off = base + ((int64_t)(e >> logG) << rowshift) + (e & G1);
      sm[ntt_pad(e)] = (off < E) ? g[off] : 0;
    }
    __syncthreads();
    ntt_tile<true, TH>(sm, hi, lo, cx.Ui[jp], q);
#pragma unroll 1
    for (int h = 0; h < 512 / TH; ++h) {
#pragma unroll
      for (int mm = 0; mm < 8; ++mm) x[mm] = sm[ntt_pad(ntt_top_word<TH>(h, mm))];
      ntt_top_inv(x, hi, lo, cx.Ui[jp], q);
#pragma unroll
      for (int mm = 0; mm < 8; ++mm) {
        const int e = ntt_top_word<TH>(h, mm);
        const int64_t off = base + ((int64_t)(e >> logG) << rowshift) + (e & G1);
        if (off < E) {
          uint64_t v = x[mm];
          if (logRp) {
            const uint32_t c = (uint32_t)((off >> logn) & ((1 << logRp) - 1)), pos = (uint32_t)(off & ln1);
            v = ntt_twist<true>(v, (brev_bits(c, logRp) * pos) << (ZP_NTT_LOGMAX - lpar), cx.Tlo[jp], cx.Thi[jp], q);
          }
          g[off] = v;
        }
      }
    }
  }
}

// ---- products: forward chunk stages, pointwise product, inverse chunk stages in ONE kernel ----------------------------
// Segments are n = 2^logseg words; the last logn <= 12 stages of their transforms (all of them when logseg <= 12; else
// the strided passes have run on A and B before, and run on O after, this kernel; logRp as in k_ntt_pass) act inside
// chunks of 4096 consecutive words, and the pointwise product is position-wise, so a CTA can take the chunk of the two
// operands through the forward stages, multiply, and take the product back through the inverse stages without the
// transformed operands ever leaving the SM.  The factor 1/n rides on the product (Kq[j] = 2^128 / n mod q_j:
// mont_mul(mont_mul(a, b), Kq) = a b / n).  A CTA = one chunk of one prime.
//   MODE 0 (pairs): O segment o = A segment 2o * A segment 2o + 1               (up-tree; Newton; root); B != null (= A):
//                   the complete transforms of the operands, times 2^64 / n (canonical), are written back over them --
//                   kept for MODE 1 later, whose pointwise product is then ONE Montgomery product per word
//   MODE 1 (down) : O segments 2 vt + side = A segment vt * B segment 2 (vt mod P) + 1 - side, side = 0, 1, where B holds
//                   the COMPLETE forward transforms times 2^64 / n that MODE 0 kept: tails x reversed siblings, the siblings' transforms are
//                   shared by all the vectors of a level.  EA, EB, EO: words per prime of the three buffers; SA: the
//                   distance between the primes' copies of A.
ZP_DEV uint64_t ntt_canon4(uint64_t b, const ZpMod& q) {  // [0, 4q) -> [0, q)
  b = (b >= 2 * q.p) ? b - 2 * q.p : b;
  return (b >= q.p) ? b - q.p : b;
}
template <int MODE, int TH>
__global__ void __launch_bounds__(TH, 768 / TH)
k_ntt_mul(const uint64_t* A, int64_t EA, int64_t SA, const uint64_t* B, int64_t EB, uint64_t* __restrict__ O,
          int64_t EO, int logn, int logRp, int logseg, int64_t P, NttCtx cx, uint64_t Kq0, uint64_t Kq1, uint64_t Kq2) {
  zp_grid_dep_wait();
  extern __shared__ __align__(16) uint64_t ntt_mul_smem[];  // 2 x 32 KB (dynamic: above the 48 KB static limit)
  uint64_t *sm = ntt_mul_smem, *smA = ntt_mul_smem + ZP_NTT_SMEM;  // the working tile; the first operand's transform
  const int jp = blockIdx.y;
  const ZpMod q = cx.q[jp];
  const uint64_t Kq = jp == 0 ? Kq0 : jp == 1 ? Kq1 : Kq2;
  const int T = threadIdx.x;
  const int64_t c0 = (int64_t)blockIdx.x * ZP_NTT_C;  // first word of the chunk in the driving buffer (O / A)
  const int64_t Edrv = MODE == 0 ? EO : EA;
  const uint32_t segmask = (1u << logseg) - 1;
  const ulonglong2 *Tlo = cx.Tlo[jp], *Thi = cx.Thi[jp];
  A += (int64_t)jp * SA;  // SA = EA, or 0 when the three primes read ONE copy of the operand (residues mod p, MODE 1)
  B += (int64_t)jp * EB;
  O += (int64_t)jp * EO;
  // Segments of at least a chunk (logseg >= 12): the chunk lies in ONE segment, seg0, at the positions pos0 + e, and
  // (transforms longer than a chunk, logRp > 0, have logn = 12) in one row of its parent: word e is twisted by
  // w^((bc e) << tsh).  Shorter segments: several per chunk, no twist; the segment of word e is seg0 + ((pos0 + e) >> logseg).
  const uint32_t seg0 = (uint32_t)(c0 >> logseg), pos0 = (uint32_t)c0 & segmask;
  const uint32_t bc = logRp ? brev_bits((pos0 >> logn) & ((1u << logRp) - 1), logRp) : 0;
  const int tsh = ZP_NTT_LOGMAX - logn - logRp;
  const uint32_t Pu = (uint32_t)P, t0 = seg0 % Pu;
  // the first (and in MODE 0 the second) operand's chunk -> forward stages; the first one's transform is parked in smA
#pragma unroll 1
  for (int which = 0; which < (MODE == 0 ? 2 : 1); ++which) {
#pragma unroll 1
    for (int h = 0; h < 512 / TH; ++h) {
      uint64_t x[8];
#pragma unroll
      for (int mm = 0; mm < 8; ++mm) {
        const int e = ntt_top_word<TH>(h, mm);
        uint64_t v = 0;
        if (c0 + e < Edrv) {
          if (MODE == 0) {
            const uint32_t seg = seg0 + ((pos0 + e) >> logseg), pos = (pos0 + e) & segmask;
            v = A[((int64_t)(2 * seg + which) << logseg) | pos];
          } else {
            v = A[c0 + e];
          }
          if (logRp) v = ntt_twist<false>(v, (bc * (uint32_t)e) << tsh, Tlo, Thi, q);
        }
        x[mm] = v;
      }
      ntt_top_fwd(x, logn - 1, 0, cx.U[jp], q);  // the stages on the bits 11 .. 9, in registers
#pragma unroll
      for (int mm = 0; mm < 8; ++mm) sm[ntt_pad(ntt_top_word<TH>(h, mm))] = x[mm];
    }
    __syncthreads();
    ntt_tile<false, TH>(sm, logn - 1, 0, cx.U[jp], q);
    if (MODE == 0 && B != nullptr) {  // keep: the operand's complete transform goes back to where it came from (B = A)
#pragma unroll 4
      for (int m = 0; m < ZP_NTT_C / TH; ++m) {
        const int e = T + TH * m;
        if (c0 + e < Edrv) {
          const uint32_t seg = seg0 + ((pos0 + e) >> logseg), pos = (pos0 + e) & segmask;
          const_cast<uint64_t*>(A)[((int64_t)(2 * seg + which) << logseg) | pos] = mont_mul(sm[ntt_pad(e)], Kq, q);  // x 2^64 / n
        }
      }
    }
    if (which == 0) {
#pragma unroll 4
      for (int m = 0; m < ZP_NTT_C / TH; ++m) smA[T + TH * m] = sm[T + TH * m];  // same swizzle
      __syncthreads();  // the working tile is reused
    }
  }
#pragma unroll 1
  for (int side = 0; side < (MODE == 0 ? 1 : 2); ++side) {
    if (MODE == 0) {  // the second operand's transform is in the working tile
#pragma unroll 4
      for (int m = 0; m < ZP_NTT_C / TH; ++m) {
        const int se = T + TH * m;  // any order: the product is position-wise
        sm[se] = mont_mul(mont_mul(smA[se], ntt_canon4(sm[se], q), q), Kq, q);
      }
    } else {  // the sibling's transform at the same positions of its segment: all 16 loads of a lane in flight together
      uint64_t b[ZP_NTT_C / TH];
#pragma unroll
      for (int m = 0; m < ZP_NTT_C / TH; ++m) {
        const int e = T + TH * m;
        const uint32_t seg = seg0 + ((pos0 + e) >> logseg), pos = (pos0 + e) & segmask;
        const uint32_t tsk = (logseg >= ZP_NTT_LOGC) ? t0 : seg % Pu;  // uniform branch: the division only for short segments
        b[m] = (c0 + e < Edrv) ? __ldg(B + (((int64_t)(2 * tsk + 1 - side) << logseg) | pos)) : 0;
      }
#pragma unroll
      for (int m = 0; m < ZP_NTT_C / TH; ++m) {
        const int se = ntt_pad(T + TH * m);
        sm[se] = mont_mul(smA[se], b[m], q);  // (the kept transform carries 2^64 / n and is canonical)
      }
    }
    __syncthreads();
    ntt_tile<true, TH>(sm, logn - 1, 0, cx.Ui[jp], q);
#pragma unroll 1
    for (int h = 0; h < 512 / TH; ++h) {
      uint64_t x[8];
#pragma unroll
      for (int mm = 0; mm < 8; ++mm) x[mm] = sm[ntt_pad(ntt_top_word<TH>(h, mm))];
      ntt_top_inv(x, logn - 1, 0, cx.Ui[jp], q);
#pragma unroll
      for (int mm = 0; mm < 8; ++mm) {
        const int e = ntt_top_word<TH>(h, mm);
        if (c0 + e >= Edrv) continue;
        uint64_t v = x[mm];
        if (logRp) v = ntt_twist<true>(v, (bc * (uint32_t)e) << tsh, Tlo, Thi, q);
        if (MODE == 0) {
          O[c0 + e] = v;
        } else {
          const uint32_t seg = seg0 + ((pos0 + e) >> logseg), pos = (pos0 + e) & segmask;
          O[((int64_t)(2 * seg + side) << logseg) | pos] = v;
        }
      }
    }
    __syncthreads();  // MODE 1: the tile is reused by the other side
  }
}

// ---- Garner's CRT of one coefficient, then c K mod p ---------------------------------------------------------------------
// r1, r2, r3: the residues of the integer c modulo q1, q2, q3, lazy in [0, 2q).  c = k1 + q1 k2 + q1 q2 k3.
ZP_DEV uint64_t ntt_crt(uint64_t r1, uint64_t r2, uint64_t r3, const NttCtx& cx, const CrtOut& co, const ZpMod& kp) {
  const ZpMod &q1 = cx.q[0], &q2 = cx.q[1], &q3 = cx.q[2];
  const uint64_t k1 = lazy_canon(r1, q1.p);
  r2 = lazy_canon(r2, q2.p);
  r3 = lazy_canon(r3, q3.p);
  const uint64_t k1_2 = lazy_canon(k1, q2.p);  // k1 < q1 < 2 q2
  const uint64_t k2 = mont_mul(mod_sub(r2, k1_2, q2.p), cx.g2, q2);
  const uint64_t k1_3 = lazy_canon(k1, q3.p), k2_3 = lazy_canon(k2, q3.p);
  const uint64_t t3 = mod_sub(mod_sub(r3, k1_3, q3.p), mont_mul(k2_3, cx.g3a, q3), q3.p);
  const uint64_t k3 = mont_mul(t3, cx.g3b, q3);
  uint64_t r = mod_add(mont_mul(k1, co.C1, kp), mont_mul(k2, co.C2, kp), kp.p);
  return mod_add(r, mont_mul(k3, co.C3, kp), kp.p);
}
#endif  // __CUDACC__
