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
#define ZP_NTT_THREADS 256

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
// x * w mod q, lazily: any 64-bit x in, [0, 2q) out (w = {w, w'} with its Shoup companion)
ZP_DEV uint64_t ntt_mul(uint64_t x, ulonglong2 w, const ZpMod& q) { return horner_step(x, w.x, w.y, 0, 0, q); }
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

// ---- chunk pass: every CTA transforms 4096 consecutive words of one prime in shared memory -----------------------
// The chunk holds 4096 / ln complete transforms of length ln = 2^logn <= 4096 (the whole transform, or the rows of the
// last pass of a longer one).  logRp > 0: the transforms are the rows of parents of length ln 2^logRp; row c's
// element j is twisted by w_parent^(brev(c) j) on load (forward) / by its inverse on store (inverse).
// buf: [3][E] words (prime-major), E = words per prime (a multiple of ln).
template <bool INV>
__global__ void __launch_bounds__(ZP_NTT_THREADS)
k_ntt_chunk(uint64_t* __restrict__ buf, int64_t E, int logn, int logRp, NttCtx cx) {
  __shared__ uint64_t x[ZP_NTT_C];
  const int j = blockIdx.y;
  const ZpMod q = cx.q[j];
  const uint64_t q2 = 2 * q.p;
  uint64_t* g = buf + (int64_t)j * E;
  const int64_t c0 = (int64_t)blockIdx.x * ZP_NTT_C;
  const int ln = 1 << logn;
  const ulonglong2* __restrict__ U = INV ? cx.Ui[j] : cx.U[j];
  const int lpar = logn + logRp;  // log2 of the parent length
  for (int e = threadIdx.x; e < ZP_NTT_C; e += ZP_NTT_THREADS) {
    uint64_t v = 0;
    if (c0 + e < E) {
      v = g[c0 + e];
      if (!INV && logRp) {
        const int64_t tr = (c0 + e) >> logn;  // transform index; row c = tr mod R
        const uint32_t c = (uint32_t)(tr & ((1 << logRp) - 1)), jj = (uint32_t)((c0 + e) & (ln - 1));
        const uint32_t Ex = (brev_bits(c, logRp) * jj) << (ZP_NTT_LOGMAX - lpar);
        v = ntt_twist<false>(v, Ex, cx.Tlo[j], cx.Thi[j], q);
      }
    }
    x[e] = v;
  }
  __syncthreads();
  if (!INV) {
    for (int lm = 0; lm < logn; ++lm) {  // stage M = 2^lm, half = ln / 2M
      const int lh = logn - 1 - lm, half = 1 << lh;
      for (int bf = threadIdx.x; bf < ZP_NTT_C / 2; bf += ZP_NTT_THREADS) {
        const int s = bf >> (logn - 1), r = bf & ((ln >> 1) - 1);
        const int i = r >> lh, jj = r & (half - 1);
        const int pos = (s << logn) + (i << (lh + 1)) + jj;
        const ulonglong2 w = __ldg(U + (1 << lm) + i);
        uint64_t u = x[pos];
        u = (u >= q2) ? u - q2 : u;
        const uint64_t v = ntt_mul(x[pos + half], w, q);
        x[pos] = u + v;
        x[pos + half] = u - v + q2;
      }
      __syncthreads();
    }
  } else {
    for (int lm = logn - 1; lm >= 0; --lm) {
      const int lh = logn - 1 - lm, half = 1 << lh;
      for (int bf = threadIdx.x; bf < ZP_NTT_C / 2; bf += ZP_NTT_THREADS) {
        const int s = bf >> (logn - 1), r = bf & ((ln >> 1) - 1);
        const int i = r >> lh, jj = r & (half - 1);
        const int pos = (s << logn) + (i << (lh + 1)) + jj;
        const ulonglong2 w = __ldg(U + (1 << lm) + i);
        const uint64_t u = x[pos], v = x[pos + half];  // [0, 2q)
        const uint64_t sum = u + v;
        x[pos] = (sum >= q2) ? sum - q2 : sum;
        x[pos + half] = ntt_mul(u - v + q2, w, q);
      }
      __syncthreads();
    }
  }
  for (int e = threadIdx.x; e < ZP_NTT_C; e += ZP_NTT_THREADS) {
    if (c0 + e < E) {
      uint64_t v = x[e];
      if (INV && logRp) {
        const int64_t tr = (c0 + e) >> logn;
        const uint32_t c = (uint32_t)(tr & ((1 << logRp) - 1)), jj = (uint32_t)((c0 + e) & (ln - 1));
        const uint32_t Ex = (brev_bits(c, logRp) * jj) << (ZP_NTT_LOGMAX - lpar);
        v = ntt_twist<true>(v, Ex, cx.Tlo[j], cx.Thi[j], q);
      }
      g[c0 + e] = v;
    }
  }
}

// ---- strided pass: the first logR stages of transforms of length n = 2^logn on the [R x L] view (L = n / R) ------
// CTA = (transform, tile of G = 4096 / R consecutive columns); R <= 512.  logRp as above (these transforms are rows of
// a longer parent: the middle pass of a three-pass plan).
template <bool INV>
__global__ void __launch_bounds__(ZP_NTT_THREADS)
k_ntt_strided(uint64_t* __restrict__ buf, int64_t E, int logn, int logR, int logRp, NttCtx cx) {
  __shared__ uint64_t x[ZP_NTT_C];
  const int j = blockIdx.y;
  const ZpMod q = cx.q[j];
  const uint64_t q2 = 2 * q.p;
  const int logG = ZP_NTT_LOGC - logR, G = 1 << logG, R = 1 << logR;
  const int logL = logn - logR;
  const int tiles_log = logL - logG;  // column tiles per transform
  const int64_t tr = (int64_t)blockIdx.x >> tiles_log;
  const int col0 = (int)(blockIdx.x & ((1 << tiles_log) - 1)) << logG;
  uint64_t* g = buf + (int64_t)j * E + (tr << logn) + col0;
  if ((tr << logn) >= E) return;
  const ulonglong2* __restrict__ U = INV ? cx.Ui[j] : cx.U[j];
  const int lpar = logn + logRp;
  const uint32_t crow = (uint32_t)(tr & ((1 << logRp) - 1));  // this transform's row in its parent
  const uint32_t cb = brev_bits(crow, logRp);
  for (int e = threadIdx.x; e < ZP_NTT_C; e += ZP_NTT_THREADS) {
    const int r = e >> logG, c = e & (G - 1);
    uint64_t v = g[((int64_t)r << logL) + c];
    if (!INV && logRp) {
      const uint32_t jj = ((uint32_t)r << logL) + col0 + c;  // position inside this transform
      v = ntt_twist<false>(v, (cb * jj) << (ZP_NTT_LOGMAX - lpar), cx.Tlo[j], cx.Thi[j], q);
    }
    x[e] = v;
  }
  __syncthreads();
  if (!INV) {
    for (int lm = 0; lm < logR; ++lm) {
      const int lh = logR - 1 - lm, half = 1 << lh;
      for (int bf = threadIdx.x; bf < ZP_NTT_C / 2; bf += ZP_NTT_THREADS) {
        const int c = bf & (G - 1), rb = bf >> logG;
        const int i = rb >> lh, jj = rb & (half - 1);
        const int pos = (((i << (lh + 1)) + jj) << logG) + c;
        const ulonglong2 w = __ldg(U + (1 << lm) + i);
        uint64_t u = x[pos];
        u = (u >= q2) ? u - q2 : u;
        const uint64_t v = ntt_mul(x[pos + (half << logG)], w, q);
        x[pos] = u + v;
        x[pos + (half << logG)] = u - v + q2;
      }
      __syncthreads();
    }
  } else {
    for (int lm = logR - 1; lm >= 0; --lm) {
      const int lh = logR - 1 - lm, half = 1 << lh;
      for (int bf = threadIdx.x; bf < ZP_NTT_C / 2; bf += ZP_NTT_THREADS) {
        const int c = bf & (G - 1), rb = bf >> logG;
        const int i = rb >> lh, jj = rb & (half - 1);
        const int pos = (((i << (lh + 1)) + jj) << logG) + c;
        const ulonglong2 w = __ldg(U + (1 << lm) + i);
        const uint64_t u = x[pos], v = x[pos + (half << logG)];
        const uint64_t sum = u + v;
        x[pos] = (sum >= q2) ? sum - q2 : sum;
        x[pos + (half << logG)] = ntt_mul(u - v + q2, w, q);
      }
      __syncthreads();
    }
  }
  for (int e = threadIdx.x; e < ZP_NTT_C; e += ZP_NTT_THREADS) {
    const int r = e >> logG, c = e & (G - 1);
    uint64_t v = x[e];
    if (INV && logRp) {
      const uint32_t jj = ((uint32_t)r << logL) + col0 + c;
      v = ntt_twist<true>(v, (cb * jj) << (ZP_NTT_LOGMAX - lpar), cx.Tlo[j], cx.Thi[j], q);
    }
    g[((int64_t)r << logL) + c] = v;
  }
}

// ---- pointwise products in the transformed domain -------------------------------------------------------------------
// out segment o = A segment ia(o) * B segment ib(o) * (1/n), per prime; segments are n = 2^logn words.
//   mode 0 (pairs)  : A = B = X,  ia = 2o, ib = 2o + 1                          (up-tree; Newton; root)
//   mode 1 (down)   : A = Y, ia = o / 2;  B = X, ib = 2 ((o / 2) mod P) + 1 - (o & 1)   (tails x reversed siblings)
//   mode 2 (against): A = Y, ia = o;  B = X, ib = 1                             (Newton's second product)
// Kq[j] = 2^128 / n mod q_j: mont_mul(mont_mul(a, b), Kq) = a b / n.  EA, EB, EO: words per prime of the three buffers.
__global__ void __launch_bounds__(256)
k_ntt_pointwise(const uint64_t* __restrict__ A, int64_t EA, const uint64_t* __restrict__ B, int64_t EB,
                uint64_t* __restrict__ O, int64_t EO, int logn, int mode, int64_t P, NttCtx cx, uint64_t Kq0, uint64_t Kq1,
                uint64_t Kq2) {
  const int j = blockIdx.y;
  const ZpMod q = cx.q[j];
  const uint64_t Kq = j == 0 ? Kq0 : j == 1 ? Kq1 : Kq2;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EO; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t o = e >> logn, i = e & (((int64_t)1 << logn) - 1);
    int64_t ia, ib;
    if (mode == 0) {
      ia = 2 * o;
      ib = 2 * o + 1;
    } else if (mode == 1) {
      ia = o >> 1;
      ib = 2 * ((o >> 1) % P) + 1 - (o & 1);
    } else {
      ia = o;
      ib = 1;
    }
    const uint64_t a = A[(int64_t)j * EA + (ia << logn) + i];
    uint64_t b = B[(int64_t)j * EB + (ib << logn) + i];  // lazy, < 4q
    b = (b >= 2 * q.p) ? b - 2 * q.p : b;
    b = (b >= q.p) ? b - q.p : b;
    O[(int64_t)j * EO + e] = mont_mul(mont_mul(a, b, q), Kq, q);
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
