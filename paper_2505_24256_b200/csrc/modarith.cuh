// modarith.cuh -- (a0) arithmetic substrate: 63-bit Montgomery arithmetic on the sm_100a integer pipes.
//
// What the paper does here (section 2.1): 64-bit a*b mod n on the GPU; the FLINT
// port (precomputed inverse, no division) won.  What this build does instead: Montgomery form with
// R = 2^64 in 32-bit limbs.  Measured on B200 (profiles/r01_baseline.md): IMAD (32-bit low
// multiply-add) issues at 63.5 lanes/clk/SM, IMAD.WIDE.U32 (32x32+64->64) at 31.8 and IMAD.HI at 30.8, on the
// same fma-heavy pipe; IADD3/LOP3 run on the alu pipe and co-issue -- so everything is built from
// mul.wide/mad.wide (one wide product instead of a lo + hi pair) and the carries ride on predicates
// (ptxas turns add.cc/addc on mad.wide results into IMAD.WIDE[.X]).
//
// Forms:  plain x in [0,p);  Montgomery x~ = x * 2^64 mod p in [0,p).
//   mont_mul(a,b) = a*b*2^-64 mod p            (10 multiplier instructions: 8 IMAD.WIDE + 2 IMAD.LO)
//   horner_step   = m*x + a mod p, lazily, for a fixed m with its Shoup companion (6 IMAD.WIDE + 4 IMAD)
//   Acc           = deferred 160-bit accumulator of 64x64 products ("emulating a
//                   192-bit integer"; 160 bits suffice: < 2^31 products of < 2^128)   4 IMAD.WIDE / MAC
//   acc_redc160   = T * 2^-160 mod p for a 160-bit T, any odd p < 2^63 (five 32-bit REDC rounds)
#pragma once
#include <cstdint>

struct ZpMod {
  uint64_t p;
  uint32_t p0, p1;  // p = p1:p0
  uint32_t pinv;    // -p^{-1} mod 2^32
  uint64_t r1;      // 2^64  mod p : Montgomery form of 1
  uint64_t r2;      // 2^128 mod p : to_mont multiplier
  uint64_t c96;     // 2^96  mod p : mont_mul(acc_redc160(sum of mont*mont), c96)  -> plain
  uint64_t c160;    // 2^160 mod p : mont_mul(acc_redc160(sum of mont*mont), c160) -> Montgomery
                    //               mont_mul(acc_redc160(sum of mont*plain), c160) -> plain
  uint64_t c224;    // 2^224 mod p : mont_mul(acc_redc160(sum of mont*plain), c224) -> Montgomery
  uint64_t np;      // 2^64 - p          : x + q*np = x - q*p  (mod 2^64)
  uint64_t ninv64;  // -p^{-1} mod 2^64  : shoup_companion
};

#if defined(__CUDACC__)
#define ZP_DEV __device__ __forceinline__

ZP_DEV uint64_t zp_mulw(uint32_t a, uint32_t b) {
  uint64_t r;
  asm("mul.wide.u32 %0, %1, %2;" : "=l"(r) : "r"(a), "r"(b));
  return r;
}
ZP_DEV uint64_t zp_madw(uint32_t a, uint32_t b, uint64_t c) {
  uint64_t r;
  asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(r) : "r"(a), "r"(b), "l"(c));
  return r;
}

ZP_DEV uint32_t zp_madlo(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t r;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}

ZP_DEV uint64_t mod_add(uint64_t a, uint64_t b, uint64_t p) {  // a, b < p < 2^63: no overflow
  uint64_t r = a + b, s = r - p;
  return (r >= p) ? s : r;
}
ZP_DEV uint64_t mod_sub(uint64_t a, uint64_t b, uint64_t p) {
  uint64_t r = a - b;
  return (a >= b) ? r : r + p;
}
ZP_DEV uint64_t mod_neg(uint64_t a, uint64_t p) { return a ? p - a : 0; }
// input residue -> canonical.  Callers pass canonical residues (reading G22), so the 64-bit division (about a
// hundred instructions) sits behind a branch that is practically never taken.
// Programmatic dependent launch (sm_90+): a kernel launched with the "programmatic stream serialization" attribute may
// become resident while its predecessor in the stream drains; it must not touch global memory before this wait, which
// returns when the predecessor grid has completed and its writes are visible.  A no-op under a plain launch.
ZP_DEV void zp_grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
ZP_DEV uint64_t zp_canon(uint64_t x, uint64_t p) { return x < p ? x : x % p; }

// Montgomery product (54 pipe cycles against 62.5 and 59.7 for the two 32-bit-round forms kept in ubench.cuh,
// zippel_ubench kinds 20 / 8 / 21, profiles/r01_final.md): one 64-bit REDC round, written with 64-bit operations
// (the compiler expands them).  Requires a*b < p*2^64 (true for any a < 2^64 and b < p):
//     m = lo(T) * (-p^-1 mod 2^64);  (T + m p) / 2^64 = hi(T) + hi(m p) + (lo(T) != 0)  < 2p.
ZP_DEV uint64_t mont_mul(uint64_t a, uint64_t b, const ZpMod& k) {
  const uint64_t lo = a * b, hi = __umul64hi(a, b);
  const uint64_t m = lo * k.ninv64;
  const uint64_t r = hi + __umul64hi(m, k.p) + (lo != 0);
  const uint64_t s = r - k.p;
  return (r >= k.p) ? s : r;
}
ZP_DEV uint64_t to_mont(uint64_t x, const ZpMod& k) { return mont_mul(x, k.r2, k); }
ZP_DEV uint64_t from_mont(uint64_t x, const ZpMod& k) { return mont_mul(x, 1, k); }

// x~^e (Montgomery in, Montgomery out), right-to-left square and multiply.
ZP_DEV uint64_t mont_pow(uint64_t x, uint64_t e, const ZpMod& k) {
  uint64_t r = k.r1;
  while (e) {
    if (e & 1) r = mont_mul(r, x, k);
    x = mont_mul(x, x, k);
    e >>= 1;
  }
  return r;
}
// a^-1 2^k mod p for a in [1, p), p odd, gcd(a, p) = 1 -- the first phase of Kaliski's "almost Montgomery inverse", with
// the runs of halvings taken at once (count of trailing zeros) and no branch in the loop, so that lanes with different
// arguments run the same instructions.  Plain 64-bit integers, no multiplication: a Montgomery product is about 160
// cycles of latency on sm_100a and a Fermat power is 125 of them in a chain; this loop is ~45 iterations (at most
// 126) of ~30 instructions.  Invariants (u, v odd):  p = u s + v r  (so r + s <= p: nothing overflows),
// a s = v 2^k,  a r = -u 2^k (mod p).  The loop ends with u = v = gcd(a, p); then a s = 2^k.  62 <= ... k <= 126 for
// p near 2^63, k >= log2 p in general.  0 or a common factor (p not prime) -> 0; callers flag zeros.
ZP_DEV uint64_t zp_almost_inv(uint64_t a, uint64_t p, int& kout) {
  kout = 0;
  if (a == 0) return 0;
  uint64_t u = p, v = a, r = 0, s = 1;
  int k = __ffsll((long long)v) - 1;
  v >>= k;
  while (u != v) {
    const bool gt = u > v;
    const uint64_t d = gt ? u - v : v - u;  // even, non-zero
    const int z = __ffsll((long long)d) - 1;
    const uint64_t dz = d >> z, sum = r + s, sh = (gt ? s : r) << z;
    u = gt ? dz : u;
    v = gt ? v : dz;
    r = gt ? sum : sh;
    s = gt ? sh : sum;
    k += z;
  }
  kout = k;
  return u == 1 ? s : 0;
}
// 2^j mod p, 0 <= j <= 64
ZP_DEV uint64_t zp_pow2_mod(int j, const ZpMod& k) {
  if (j == 64) return k.r1;
  const uint64_t x = 1ull << j;
  if (x < k.p) return x;
  return (x - k.p < k.p) ? x - k.p : x % k.p;  // (the division only for p < 2^62)
}
// Inverse, x~ -> (x^-1)~ ; 0 -> 0 (callers flag it).  p prime is the caller's contract.  With s = (x~)^-1 2^k from above,
// (x^-1)~ = 2^128 / x~ = s 2^(128-k):  mont_mul(s, r2) = s 2^64, times 2^e / 2^64 with e = 128 - k in [2, 128].
ZP_DEV uint64_t mont_inv(uint64_t x, const ZpMod& k) {
  int kk;
  const uint64_t s = zp_almost_inv(x, k.p, kk);
  const int e = 128 - kk;
  const uint64_t c = (e <= 64) ? zp_pow2_mod(e, k) : mont_mul(zp_pow2_mod(e - 64, k), k.r2, k);  // 2^e mod p
  return mont_mul(mont_mul(s, k.r2, k), c, k);
}
// Inverse by Fermat: kept as the cross-check of the one above (zippel_modarith_selftest)
ZP_DEV uint64_t mont_inv_fermat(uint64_t x, const ZpMod& k) { return mont_pow(x, k.p - 2, k); }
// (the argument is uniform across the warp: the one inversion of a batched inversion; same routine)
ZP_DEV uint64_t mont_inv_uniform(uint64_t x, const ZpMod& k) { return mont_inv(x, k); }

// ---- Horner step with Shoup companions (the hot recurrence of (a3): q <- M_l + m q, d <- M'_l + m d) ----
// For w in [0,p) its companion is w' = floor(w 2^64 / p) < 2^64.  Since w 2^64 - w~ = w' p with
// w~ = w 2^64 mod p (the Montgomery form), w' = -w~ p^{-1} mod 2^64: one 64-bit low product.
ZP_DEV uint64_t shoup_companion(uint64_t w_mont, const ZpMod& k) { return w_mont * k.ninv64; }

// x <- m x + a (mod p), lazily: ANY x < 2^64 in, result in [0, 2p) (< 2^64 because p < 2^63).
// With qq = floor((m' x + a') / 2^64):  (m x + a)/p = (m' x + a')/2^64 + (e1 x + e3)/2^64 with
// e1, e3 in [0,1), so  u = m x + a - qq p = p (frac + (e1 x + e3)/2^64)  lies in [0, 2p) and is computed
// exactly modulo 2^64.  No conditional correction and no Montgomery form: 10 multiplier instructions
// (4 wide for the exact high half of m' x + a', 2 wide + 4 low for u) and 3 carry instructions.
ZP_DEV uint64_t horner_step(uint64_t x, uint64_t m, uint64_t mp, uint64_t a, uint64_t ap, const ZpMod& k) {
  const uint32_t w0 = (uint32_t)mp, w1 = (uint32_t)(mp >> 32), x0 = (uint32_t)x, x1 = (uint32_t)(x >> 32);
  const uint32_t m0 = (uint32_t)m, m1 = (uint32_t)(m >> 32);
  const uint32_t np0 = (uint32_t)k.np, np1 = (uint32_t)(k.np >> 32);
  const uint64_t Bm = zp_mulw(w0, x1);
  uint32_t tlo, thi;
  asm("{\n\t"
      ".reg .u64 d, s;\n\t"
      ".reg .u32 dlo, dhi, slo, shi, c0, c1, dummy;\n\t"
      "mul.wide.u32 d, %2, %3;\n\t"
      "add.cc.u64 d, d, %4;\n\t"  // D = w0 x0 + a'            carry c0 (weight 2^64)
      "addc.u32 c0, 0, 0;\n\t"
      "mul.wide.u32 s, %5, %3;\n\t"
      "add.cc.u64 s, s, %6;\n\t"  // S = w1 x0 + w0 x1         carry c1 (weight 2^96)
      "addc.u32 c1, 0, 0;\n\t"
      "mov.b64 {dlo, dhi}, d;\n\t"
      "mov.b64 {slo, shi}, s;\n\t"
      "add.cc.u32 dummy, slo, dhi;\n\t"
      "addc.cc.u32 %0, shi, c0;\n\t"
      "addc.u32 %1, c1, 0;\n\t"
      "}"
      : "=r"(tlo), "=r"(thi)
      : "r"(w0), "r"(x0), "l"(ap), "r"(w1), "l"(Bm));
  const uint64_t qq = zp_madw(w1, x1, ((uint64_t)thi << 32) | tlo);
  const uint32_t q0 = (uint32_t)qq, q1 = (uint32_t)(qq >> 32);
  uint32_t uh = (uint32_t)(a >> 32);  // u = m x + a + qq np  (mod 2^64)
  uh = zp_madlo(m0, x1, uh);
  uh = zp_madlo(m1, x0, uh);
  uh = zp_madlo(q0, np1, uh);
  uh = zp_madlo(q1, np0, uh);
  uint64_t u = ((uint64_t)uh << 32) | (uint32_t)a;
  u = zp_madw(m0, x0, u);
  u = zp_madw(q0, np0, u);
  return u;
}
ZP_DEV uint64_t lazy_canon(uint64_t x, uint64_t p) {  // [0,2p) -> [0,p)
  const uint64_t s = x - p;
  return (x >= p) ? s : x;
}
// x * w mod p, lazily, for a fixed multiplier w in [0, p) with its companion w' = floor(w 2^64 / p): ANY 64-bit x in,
// [0, 2p) out.  horner_step without its addends (whose carry plumbing ptxas keeps even when they are zero):
// qq = floor(w' x / 2^64) exactly (4 wide products, the carries through predicates), then w x - qq p modulo 2^64
// (2 wide + 4 low products): 16 units of the multiplier pipe and 4 instructions on the alu pipe.
ZP_DEV uint64_t shoup_mul_lazy(uint64_t x, uint64_t w, uint64_t wc, const ZpMod& k) {
  const uint32_t x0 = (uint32_t)x, x1 = (uint32_t)(x >> 32), p0 = (uint32_t)wc, p1 = (uint32_t)(wc >> 32);
  const uint32_t w0 = (uint32_t)w, w1 = (uint32_t)(w >> 32);
  const uint32_t np0 = (uint32_t)k.np, np1 = (uint32_t)(k.np >> 32);
  uint64_t qq;
  asm("{\n\t"
      ".reg .u64 a, s, s2, t;\n\t"
      ".reg .u32 alo, ahi, slo, shi, c1, tlo, thi, dummy;\n\t"
      "mul.wide.u32 a, %1, %3;\n\t"   // w'0 x0 (its high word carries into the middle)
      "mul.wide.u32 s, %1, %4;\n\t"   // w'0 x1
      "mul.wide.u32 s2, %2, %3;\n\t"  // w'1 x0
      "add.cc.u64 s, s2, s;\n\t"      // middle sum, carry c1 (weight 2^96)
      "addc.u32 c1, 0, 0;\n\t"
      "mov.b64 {alo, ahi}, a;\n\t"
      "mov.b64 {slo, shi}, s;\n\t"
      "add.cc.u32 dummy, slo, ahi;\n\t"
      "addc.cc.u32 tlo, shi, 0;\n\t"
      "addc.u32 thi, c1, 0;\n\t"
      "mov.b64 t, {tlo, thi};\n\t"
      "mad.wide.u32 %0, %2, %4, t;\n\t"  // w'1 x1 + (middle >> 32)
      "}"
      : "=l"(qq)
      : "r"(p0), "r"(p1), "r"(x0), "r"(x1));
  const uint32_t q0 = (uint32_t)qq, q1 = (uint32_t)(qq >> 32);
  uint32_t uh = zp_madlo(w0, x1, 0);
  uh = zp_madlo(w1, x0, uh);
  uh = zp_madlo(q0, np1, uh);
  uh = zp_madlo(q1, np0, uh);
  uint64_t u = (uint64_t)uh << 32;
  u = zp_madw(w0, x0, u);
  return zp_madw(q0, np0, u);
}
// the same with a canonical result
ZP_DEV uint64_t shoup_mul(uint64_t x, ulonglong2 w, const ZpMod& k) {
  return lazy_canon(shoup_mul_lazy(x, w.x, w.y, k), k.p);
}

// Deferred accumulator.  value = E + O * 2^32 with
//   E = e0 + e1*2^64 + e2*2^128  (takes x0*y0 at bit 0 and x1*y1 at bit 64),
//   O = o0 + o1*2^64             (takes x0*y1 + x1*y0).
// Per MAC: 4 IMAD.WIDE with the accumulate folded in, the carries leave through predicates into the
// two 32-bit counters: 2 IADD3.X.  The split keeps every multiply 64-bit aligned so that no shifted
// add is needed (8 registers instead of 5; the 5-register form costs 4 IADD3 per MAC).
struct Acc {
  uint64_t e0, e1, o0;
  uint32_t e2, o1;
};
ZP_DEV void acc_zero(Acc& a) { a.e0 = a.e1 = a.o0 = 0; a.e2 = a.o1 = 0; }
ZP_DEV void acc_mac(Acc& a, uint64_t x, uint64_t y) {
  const uint32_t x0 = (uint32_t)x, x1 = (uint32_t)(x >> 32), y0 = (uint32_t)y, y1 = (uint32_t)(y >> 32);
  const uint64_t lo = zp_mulw(x0, y0), hi = zp_mulw(x1, y1), m0 = zp_mulw(x0, y1), m1 = zp_mulw(x1, y0);
  asm("add.cc.u64 %0, %0, %3;\n\t"
      "addc.cc.u64 %1, %1, %4;\n\t"
      "addc.u32 %2, %2, 0;"
      : "+l"(a.e0), "+l"(a.e1), "+r"(a.e2)
      : "l"(lo), "l"(hi));
  asm("add.cc.u64 %0, %0, %2;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "add.cc.u64 %0, %0, %3;\n\t"
      "addc.u32 %1, %1, 0;"
      : "+l"(a.o0), "+r"(a.o1)
      : "l"(m0), "l"(m1));
}

// Two MACs into the same accumulator, a += x*y + u*w, written so that carries of equal weight are adjacent:
// ptxas then folds each pair of carries into ONE IADD3.X with two carry-ins (alu pipe) instead of IMAD.X
// (which would take a slot of the multiplier pipe, the bound of the hot loop): 8 IMAD.WIDE + 3 IADD3.X.
ZP_DEV void acc_mac2(Acc& a, uint64_t x, uint64_t y, uint64_t u, uint64_t w) {
  const uint32_t x0 = (uint32_t)x, x1 = (uint32_t)(x >> 32), y0 = (uint32_t)y, y1 = (uint32_t)(y >> 32);
  const uint32_t u0 = (uint32_t)u, u1 = (uint32_t)(u >> 32), w0 = (uint32_t)w, w1 = (uint32_t)(w >> 32);
  const uint64_t lo = zp_mulw(x0, y0), hi = zp_mulw(x1, y1), lo2 = zp_mulw(u0, w0), hi2 = zp_mulw(u1, w1);
  asm("add.cc.u64 %0, %0, %3;\n\t"
      "addc.cc.u64 %1, %1, %4;\n\t"
      "addc.u32 %2, %2, 0;\n\t"
      "add.cc.u64 %0, %0, %5;\n\t"
      "addc.cc.u64 %1, %1, %6;\n\t"
      "addc.u32 %2, %2, 0;"
      : "+l"(a.e0), "+l"(a.e1), "+r"(a.e2)
      : "l"(lo), "l"(hi), "l"(lo2), "l"(hi2));
  const uint64_t m0 = zp_mulw(x0, y1), m1 = zp_mulw(x1, y0), m2 = zp_mulw(u0, w1), m3 = zp_mulw(u1, w0);
  asm("add.cc.u64 %0, %0, %2;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "add.cc.u64 %0, %0, %3;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "add.cc.u64 %0, %0, %4;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "add.cc.u64 %0, %0, %5;\n\t"
      "addc.u32 %1, %1, 0;"
      : "+l"(a.o0), "+r"(a.o1)
      : "l"(m0), "l"(m1), "l"(m2), "l"(m3));
}

// acc_mac2 on limbs: a += (x1:x0)*(y1:y0) + (u1:u0)*(w1:w0), the caller supplies the 32-bit halves (the node-solve
// loop loads the broadcast operands as {y0, w0, y1, w1} so that the two limbs of one operand sit in registers of
// the same parity: profiles/r01_final.md, register banks).
ZP_DEV void acc_mac2_limbs(Acc& a, uint32_t x0, uint32_t x1, uint32_t y0, uint32_t y1, uint32_t u0, uint32_t u1,
                           uint32_t w0, uint32_t w1) {
  const uint64_t lo = zp_mulw(x0, y0), hi = zp_mulw(x1, y1), lo2 = zp_mulw(u0, w0), hi2 = zp_mulw(u1, w1);
  asm("add.cc.u64 %0, %0, %3;\n\t"
      "addc.cc.u64 %1, %1, %4;\n\t"
      "addc.u32 %2, %2, 0;\n\t"
      "add.cc.u64 %0, %0, %5;\n\t"
      "addc.cc.u64 %1, %1, %6;\n\t"
      "addc.u32 %2, %2, 0;"
      : "+l"(a.e0), "+l"(a.e1), "+r"(a.e2)
      : "l"(lo), "l"(hi), "l"(lo2), "l"(hi2));
  const uint64_t m0 = zp_mulw(x0, y1), m1 = zp_mulw(x1, y0), m2 = zp_mulw(u0, w1), m3 = zp_mulw(u1, w0);
  asm("add.cc.u64 %0, %0, %2;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "add.cc.u64 %0, %0, %3;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "add.cc.u64 %0, %0, %4;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "add.cc.u64 %0, %0, %5;\n\t"
      "addc.u32 %1, %1, 0;"
      : "+l"(a.o0), "+r"(a.o1)
      : "l"(m0), "l"(m1), "l"(m2), "l"(m3));
}

// T * 2^-160 mod p, canonical, for the 160-bit T held in the accumulator (five REDC rounds of 32 bits:
// T_{k+1} = (T_k + m p)/2^32 < T_k/2^32 + p, so T_5 < T_0/2^160 + p(1 + 2^-32 + ...) <= p + 1).
ZP_DEV uint64_t acc_redc160(const Acc& a, const ZpMod& k) {
  // fold E + O*2^32 into five words
  uint32_t w0 = (uint32_t)a.e0, w1 = (uint32_t)(a.e0 >> 32), w2 = (uint32_t)a.e1, w3 = (uint32_t)(a.e1 >> 32), w4 = a.e2;
  {
    uint64_t c = (uint64_t)w1 + (uint32_t)a.o0;
    w1 = (uint32_t)c;
    c = (uint64_t)w2 + (uint32_t)(a.o0 >> 32) + (c >> 32);
    w2 = (uint32_t)c;
    c = (uint64_t)w3 + a.o1 + (c >> 32);
    w3 = (uint32_t)c;
    w4 += (uint32_t)(c >> 32);
  }
#pragma unroll
  for (int r = 0; r < 5; ++r) {
    const uint32_t m = w0 * k.pinv;
    uint64_t c = zp_madw(m, k.p0, (uint64_t)w0);      // low word cancels
    c = zp_madw(m, k.p1, (uint64_t)w1 + (c >> 32));   // (2^32-1)(2^31-1) + 2*2^32 < 2^64
    w0 = (uint32_t)c;
    c = (uint64_t)w2 + (c >> 32);
    w1 = (uint32_t)c;
    c = (uint64_t)w3 + (c >> 32);
    w2 = (uint32_t)c;
    c = (uint64_t)w4 + (c >> 32);
    w3 = (uint32_t)c;
    w4 = (uint32_t)(c >> 32);
  }
  const uint64_t r = ((uint64_t)w1 << 32) | w0;  // w2 = w3 = w4 = 0 here
  const uint64_t s = r - k.p;
  return (r >= k.p) ? s : r;
}
#endif  // __CUDACC__
