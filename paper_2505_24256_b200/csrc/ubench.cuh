// ubench.cuh -- roofline micro-benchmarks for the 32-bit integer multiplier (fma-heavy) pipe of sm_100a.
// the denominator of every reported fraction is measured, not assumed.  Each kernel
// keeps CH independent chains per lane in registers, no memory traffic; the host (bench side) divides
// lane-ops by elapsed time.  Kinds (ZP_UB_*):
//   0 mad.lo.u32          IMAD            32x32+32 -> 32
//   1 mad.wide.u32        IMAD.WIDE.U32   32x32+64 -> 64
//   2 mad.hi.u32          IMAD.HI.U32     hi32(32x32)+32
//   3 mad.wide + add.cc / addc chain (IMAD.WIDE with carry-out + IADD3.X): the deferred MAC (4 wide / MAC)
//   4 add + xor           IADD3 + LOP3    (alu pipe; 2 per statement)
//   5 mad.wide.u32 and IADD3 interleaved 1:1 (co-issue check)
//   6 mad.lo.u32 and mad.wide.u32 interleaved 2:1
//   7 the library's Horner step (horner_step, modarith.cuh): modular x <- m x + a with Shoup companions
//   8 the library's Montgomery product (mont_mul)
//   9 fma.rn.f64          DFMA            (fp64 pipe)
//  10 DFMA and IMAD.WIDE interleaved 1:1 (do the fp64 and fma-heavy pipes overlap?)
//  11 mul.wide.u32        IMAD.WIDE.U32 with a zero addend (the bare 32x32 -> 64 product)
//  12 acc_mac             deferred MAC, products accumulate inside IMAD.WIDE (4 wide + carries)
//  13 acc_mac2            two such MACs with merged carries (the node-solve loop's form; counts 2 MACs)
//  14 acc_mac_split       bare products, all additions on the alu pipe
//  15 acc_mac_hyb         even lattice inside IMAD.WIDE, middle products bare + alu
//  16 as 3 with the multiplicand in an even register (register-bank experiment: 3 has both multiplicands odd)
//  8/20/21 forms of the Montgomery product (8 mont_mul_v1: columns; 20 mont_mul: 64-bit REDC, in use; 21 mont_mul_v3: bare products + 32-bit chains)
//  17/18/19 as 3 with multiplicands (lo, hi) / (lo, lo) / (hi, hi) halves of live 64-bit pairs: even+odd / even+even / odd+odd
#pragma once
#include "modarith.cuh"

// ---- forms of the Montgomery product and of the deferred MAC that lost against the ones in modarith.cuh; kept for the
// ---- micro-benchmarks only (kinds 8, 21, 14, 15) --------------------------------------------------------------------
// Montgomery product, column form (mont_mul_v1: the first version, kept for the micro-benchmark).  Requires a*b < p*2^64 (true for a < 2^64, b < p); a_hi, b_hi < 2^31
// is NOT required.  With T = a*b and two 32-bit REDC rounds:
//   T + m0*p + m1*p*2^32 = (P00 + Q0) + (P01 + P10 + Q1 + S0)*2^32 + (P11 + S1)*2^64,  divisible by 2^64.
// Column 0: the low words of P00 and Q0 cancel, its carry is c0 = hi(P00) + hi(Q0) + (lo(P00) != 0) < 2^33.
// Column 1: P01 + P10 + Q1 + S0 + c0 may exceed 64 bits; `carry` counts the overflows (weight 2^64).
// Result (T + ...)/2^64 < p + p = 2p < 2^64, then one conditional subtraction.
ZP_DEV uint64_t mont_mul_v1(uint64_t a, uint64_t b, const ZpMod& k) {
  const uint32_t a0 = (uint32_t)a, a1 = (uint32_t)(a >> 32), b0 = (uint32_t)b, b1 = (uint32_t)(b >> 32);
  const uint64_t P00 = zp_mulw(a0, b0);
  const uint64_t P01 = zp_mulw(a0, b1);
  const uint64_t P10 = zp_mulw(a1, b0);
  const uint64_t P11 = zp_mulw(a1, b1);
  const uint32_t m0 = (uint32_t)P00 * k.pinv;
  const uint64_t Q0 = zp_mulw(m0, k.p0), Q1 = zp_mulw(m0, k.p1);
  const uint64_t c0 = (P00 >> 32) + (Q0 >> 32) + ((uint32_t)P00 != 0);
  uint64_t col1;
  uint32_t carry;
  asm("{\n\t"
      ".reg .u64 t;\n\t"
      "add.cc.u64 t, %2, %3;\n\t"
      "addc.u32 %1, 0, 0;\n\t"
      "add.cc.u64 t, t, %4;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "add.cc.u64 %0, t, %5;\n\t"
      "addc.u32 %1, %1, 0;\n\t"
      "}"
      : "=l"(col1), "=r"(carry)
      : "l"(P01), "l"(P10), "l"(Q1), "l"(c0));
  const uint32_t m1 = (uint32_t)col1 * k.pinv;
  const uint64_t S0 = zp_mulw(m1, k.p0);
  const uint64_t c1 = (col1 >> 32) + (S0 >> 32) + ((uint32_t)col1 != 0) + ((uint64_t)carry << 32);
  // P11 + S1 + c1 = exact quotient < 2p + 1 <= 2^64 - ... : no overflow
  const uint64_t r = zp_madw(m1, k.p1, P11 + c1);
  const uint64_t s = r - k.p;
  return (r >= k.p) ? s : r;
}

// v3: two 32-bit REDC rounds, every product a bare mul.wide, every addition a 32-bit carry chain (alu pipe).
ZP_DEV uint64_t mont_mul_v3(uint64_t a, uint64_t b, const ZpMod& k) {
  const uint32_t a0 = (uint32_t)a, a1 = (uint32_t)(a >> 32), b0 = (uint32_t)b, b1 = (uint32_t)(b >> 32);
  const uint64_t P00 = zp_mulw(a0, b0), P01 = zp_mulw(a0, b1), P10 = zp_mulw(a1, b0), P11 = zp_mulw(a1, b1);
  uint32_t t0, t1, t2, t3;
  asm("{\n\t.reg .u32 x1, y0, y1, z0, z1, w0, w1;\n\t"
      "mov.b64 {%0, x1}, %4;\n\tmov.b64 {y0, y1}, %5;\n\tmov.b64 {z0, z1}, %6;\n\tmov.b64 {w0, w1}, %7;\n\t"
      "add.cc.u32 %1, x1, y0;\n\taddc.cc.u32 %2, y1, w0;\n\taddc.u32 %3, w1, 0;\n\t"
      "add.cc.u32 %1, %1, z0;\n\taddc.cc.u32 %2, %2, z1;\n\taddc.u32 %3, %3, 0;\n\t}"
      : "=r"(t0), "=r"(t1), "=r"(t2), "=r"(t3)
      : "l"(P00), "l"(P01), "l"(P10), "l"(P11));
  const uint32_t m0 = t0 * k.pinv;
  const uint64_t Q0 = zp_mulw(m0, k.p0), Q1 = zp_mulw(m0, k.p1);
  asm("{\n\t.reg .u32 q0, q1, r0, r1, dummy;\n\t"
      "mov.b64 {q0, q1}, %4;\n\tmov.b64 {r0, r1}, %5;\n\t"
      "add.cc.u32 dummy, %3, q0;\n\taddc.cc.u32 %0, %0, q1;\n\taddc.cc.u32 %1, %1, r1;\n\taddc.u32 %2, %2, 0;\n\t"
      "add.cc.u32 %0, %0, r0;\n\taddc.cc.u32 %1, %1, 0;\n\taddc.u32 %2, %2, 0;\n\t}"
      : "+r"(t1), "+r"(t2), "+r"(t3)
      : "r"(t0), "l"(Q0), "l"(Q1));
  const uint32_t m1 = t1 * k.pinv;
  const uint64_t S0 = zp_mulw(m1, k.p0), S1 = zp_mulw(m1, k.p1);
  asm("{\n\t.reg .u32 q0, q1, r0, r1, dummy;\n\t"
      "mov.b64 {q0, q1}, %3;\n\tmov.b64 {r0, r1}, %4;\n\t"
      "add.cc.u32 dummy, %2, q0;\n\taddc.cc.u32 %0, %0, q1;\n\taddc.u32 %1, %1, r1;\n\t"
      "add.cc.u32 %0, %0, r0;\n\taddc.u32 %1, %1, 0;\n\t}"
      : "+r"(t2), "+r"(t3)
      : "r"(t1), "l"(S0), "l"(S1));
  const uint64_t r = ((uint64_t)t3 << 32) | t2;
  const uint64_t s = r - k.p;
  return (r >= k.p) ? s : r;
}

// Alternative forms of the same MAC, for the pipe-balance micro-benchmarks (zippel_ubench kinds 12-16).
// acc_mac_split: every product is a bare IMAD.WIDE (zero addend, 4 pipe cycles instead of the > 5 of the
// accumulating form, profiles/r01_baseline.md); the 160-bit additions run on the alu pipe as 32-bit carry chains.
ZP_DEV void acc_mac_split(Acc& a, uint64_t x, uint64_t y) {
  const uint32_t x0 = (uint32_t)x, x1 = (uint32_t)(x >> 32), y0 = (uint32_t)y, y1 = (uint32_t)(y >> 32);
  const uint64_t lo = zp_mulw(x0, y0), hi = zp_mulw(x1, y1), m0 = zp_mulw(x0, y1), m1 = zp_mulw(x1, y0);
  asm("{\n\t.reg .u32 a0, a1, a2, a3, l0, l1, h0, h1;\n\t"
      "mov.b64 {a0, a1}, %0;\n\tmov.b64 {a2, a3}, %1;\n\tmov.b64 {l0, l1}, %3;\n\tmov.b64 {h0, h1}, %4;\n\t"
      "add.cc.u32 a0, a0, l0;\n\taddc.cc.u32 a1, a1, l1;\n\taddc.cc.u32 a2, a2, h0;\n\taddc.cc.u32 a3, a3, h1;\n\t"
      "addc.u32 %2, %2, 0;\n\t"
      "mov.b64 %0, {a0, a1};\n\tmov.b64 %1, {a2, a3};\n\t}"
      : "+l"(a.e0), "+l"(a.e1), "+r"(a.e2)
      : "l"(lo), "l"(hi));
  asm("{\n\t.reg .u32 a0, a1, l0, l1, h0, h1;\n\t"
      "mov.b64 {a0, a1}, %0;\n\tmov.b64 {l0, l1}, %2;\n\tmov.b64 {h0, h1}, %3;\n\t"
      "add.cc.u32 a0, a0, l0;\n\taddc.cc.u32 a1, a1, l1;\n\taddc.u32 %1, %1, 0;\n\t"
      "add.cc.u32 a0, a0, h0;\n\taddc.cc.u32 a1, a1, h1;\n\taddc.u32 %1, %1, 0;\n\t"
      "mov.b64 %0, {a0, a1};\n\t}"
      : "+l"(a.o0), "+r"(a.o1)
      : "l"(m0), "l"(m1));
}
// acc_mac_hyb: the two 64-bit aligned products of the even lattice accumulate inside IMAD.WIDE (as acc_mac),
// the two middle products are bare and are added on the alu pipe.
ZP_DEV void acc_mac_hyb(Acc& a, uint64_t x, uint64_t y) {
  const uint32_t x0 = (uint32_t)x, x1 = (uint32_t)(x >> 32), y0 = (uint32_t)y, y1 = (uint32_t)(y >> 32);
  const uint64_t lo = zp_mulw(x0, y0), hi = zp_mulw(x1, y1), m0 = zp_mulw(x0, y1), m1 = zp_mulw(x1, y0);
  asm("add.cc.u64 %0, %0, %3;\n\t"
      "addc.cc.u64 %1, %1, %4;\n\t"
      "addc.u32 %2, %2, 0;"
      : "+l"(a.e0), "+l"(a.e1), "+r"(a.e2)
      : "l"(lo), "l"(hi));
  asm("{\n\t.reg .u32 a0, a1, l0, l1, h0, h1;\n\t"
      "mov.b64 {a0, a1}, %0;\n\tmov.b64 {l0, l1}, %2;\n\tmov.b64 {h0, h1}, %3;\n\t"
      "add.cc.u32 a0, a0, l0;\n\taddc.cc.u32 a1, a1, l1;\n\taddc.u32 %1, %1, 0;\n\t"
      "add.cc.u32 a0, a0, h0;\n\taddc.cc.u32 a1, a1, h1;\n\taddc.u32 %1, %1, 0;\n\t"
      "mov.b64 %0, {a0, a1};\n\t}"
      : "+l"(a.o0), "+r"(a.o1)
      : "l"(m0), "l"(m1));
}


#define ZP_UB_THREADS 256
#define ZP_UB_CH 8

template <int KIND>
__global__ void __launch_bounds__(ZP_UB_THREADS)
k_ubench(int iters, ZpMod k, uint64_t* __restrict__ out) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  uint32_t a = tid * 2654435761u + 12345u, b = (tid ^ 0x9e3779b9u) | 1u;
  uint64_t acc[ZP_UB_CH];
  uint32_t car[ZP_UB_CH];
#pragma unroll
  for (int c = 0; c < ZP_UB_CH; ++c) {
    acc[c] = ((uint64_t)(tid + c) << 32) | (a + c);
    car[c] = c;
  }
  if (KIND == 7 || KIND == 8 || KIND == 20 || KIND == 21) {
#pragma unroll
    for (int c = 0; c < ZP_UB_CH; ++c) acc[c] %= k.p;
  }
  const double dk1 = 1.0 + 1e-9 * (double)(tid & 7), dk2 = 1e-3 * (double)(tid & 3);
  uint64_t wacc[ZP_UB_CH];
#pragma unroll
  for (int c = 0; c < ZP_UB_CH; ++c) wacc[c] = acc[c] ^ 0x5555;
  if (KIND == 9 || KIND == 10) {
#pragma unroll
    for (int c = 0; c < ZP_UB_CH; ++c) acc[c] = (uint64_t)__double_as_longlong(1.0 + (double)c);
  }
  const uint64_t m = (((uint64_t)a << 32) | b) % k.p;
  const uint64_t mp = shoup_companion(to_mont(m, k), k);
  const uint64_t ad = (((uint64_t)b << 32) | a) % k.p;
  const uint64_t adp = shoup_companion(to_mont(ad, k), k);
  Acc macc[ZP_UB_CH];
#pragma unroll
  for (int c = 0; c < ZP_UB_CH; ++c) acc_zero(macc[c]);
  uint64_t xw = m, xw2 = ad;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      if (KIND >= 12 && KIND <= 15) {
        xw ^= xw << 13; xw ^= xw >> 7;     // alu-only walk of the per-lane operand
        xw2 ^= xw2 << 11; xw2 ^= xw2 >> 5;
      }
#pragma unroll
      for (int c = 0; c < ZP_UB_CH; ++c) {
        // every multiplicand comes from the chain itself, so that nothing can be hoisted out of the loop
        uint32_t lo = (uint32_t)acc[c];
        const uint32_t nb = (uint32_t)(acc[(c + 1) % ZP_UB_CH] >> 32);  // neighbour chain's high word
        if (KIND == 0) {
          asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(lo) : "r"(b), "r"(a));
          acc[c] = (acc[c] & 0xffffffff00000000ull) | lo;
        } else if (KIND == 1) {
          asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(acc[c]) : "r"(nb), "r"(b));
        } else if (KIND == 2) {
          asm volatile("mad.hi.u32 %0, %0, %1, %2;" : "+r"(lo) : "r"(b), "r"(a));
          acc[c] = (acc[c] & 0xffffffff00000000ull) | lo;
        } else if (KIND == 3) {
          asm volatile("{\n\t.reg .u64 t;\n\tmul.wide.u32 t, %2, %3;\n\tadd.cc.u64 %0, %0, t;\n\taddc.u32 %1, %1, 0;\n\t}"
                       : "+l"(acc[c]), "+r"(car[c]) : "r"(nb), "r"(b));
        } else if (KIND == 16) {  // as 3, multiplicand = the neighbour chain's LOW word (even register of its pair)
          const uint32_t nl = (uint32_t)acc[(c + 1) % ZP_UB_CH];
          asm volatile("{\n\t.reg .u64 t;\n\tmul.wide.u32 t, %2, %3;\n\tadd.cc.u64 %0, %0, t;\n\taddc.u32 %1, %1, 0;\n\t}"
                       : "+l"(acc[c]), "+r"(car[c]) : "r"(nl), "r"(b));
        } else if (KIND >= 17 && KIND <= 19) {  // register-bank experiment: both multiplicands are halves of live pairs
          const uint64_t n1 = acc[(c + 1) % ZP_UB_CH], n2 = acc[(c + 2) % ZP_UB_CH];
          const uint32_t ma = (KIND == 19) ? (uint32_t)(n1 >> 32) : (uint32_t)n1;  // 17: lo, 18: lo, 19: hi
          const uint32_t mb = (KIND == 18) ? (uint32_t)n2 : (uint32_t)(n2 >> 32);  // 17: hi, 18: lo, 19: hi
          asm volatile("{\n\t.reg .u64 t;\n\tmul.wide.u32 t, %2, %3;\n\tadd.cc.u64 %0, %0, t;\n\taddc.u32 %1, %1, 0;\n\t}"
                       : "+l"(acc[c]), "+r"(car[c]) : "r"(ma), "r"(mb));
        } else if (KIND == 4) {
          asm volatile("add.u32 %0, %0, %1;" : "+r"(car[c]) : "r"(lo));
          asm volatile("xor.b32 %0, %0, %1;" : "+r"(lo) : "r"(car[c]));
          acc[c] = (acc[c] & 0xffffffff00000000ull) | lo;
        } else if (KIND == 5) {
          asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(acc[c]) : "r"(nb), "r"(b));
          asm volatile("add.u32 %0, %0, %1;" : "+r"(car[c]) : "r"(nb));
        } else if (KIND == 6) {
          asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(acc[c]) : "r"(nb), "r"(b));
          asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(car[c]) : "r"(b), "r"(lo));
          asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(car[c]) : "r"(a), "r"(lo));
        } else if (KIND == 11) {
          asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(acc[c]) : "r"(nb), "r"(b));
        } else if (KIND == 9) {
          double x = __longlong_as_double((long long)acc[c]);
          asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x) : "d"(dk1), "d"(dk2));
          acc[c] = (uint64_t)__double_as_longlong(x);
        } else if (KIND == 10) {
          double x = __longlong_as_double((long long)acc[c]);
          asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x) : "d"(dk1), "d"(dk2));
          acc[c] = (uint64_t)__double_as_longlong(x);
          asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(wacc[c]) : "r"((uint32_t)(wacc[(c + 1) % ZP_UB_CH] >> 32)), "r"(b));
        } else if (KIND >= 12 && KIND <= 15) {
          // deferred MAC forms: 8 accumulators per lane, the per-lane operand x walks (alu only), the other
          // operand is a per-chain constant (as the broadcast v of the node-solve loop)
          Acc& A = macc[c];
          const uint64_t yv = ad + (uint64_t)c * 0x9e3779b97f4a7c15ull;
          if (KIND == 12) acc_mac(A, xw, yv);
          if (KIND == 13) acc_mac2(A, xw, yv, xw2, yv ^ mp);
          if (KIND == 14) acc_mac_split(A, xw, yv);
          if (KIND == 15) acc_mac_hyb(A, xw, yv);
        } else if (KIND == 7) {
          acc[c] = horner_step(acc[c], m, mp, ad, adp, k);
        } else if (KIND == 8) {
          acc[c] = mont_mul_v1(acc[c], m, k);
        } else if (KIND == 20) {
          acc[c] = mont_mul(acc[c], m, k);
        } else if (KIND == 21) {
          acc[c] = mont_mul_v3(acc[c], m, k);
        }
      }
    }
  }
  uint64_t s = 0;
#pragma unroll
  for (int c = 0; c < ZP_UB_CH; ++c) s += acc[c] + car[c] + (KIND == 10 ? wacc[c] : 0);
  if (KIND >= 12 && KIND <= 15) {
#pragma unroll
    for (int c = 0; c < ZP_UB_CH; ++c) s += macc[c].e0 + macc[c].e1 + macc[c].o0 + macc[c].e2 + macc[c].o1;
  }
  if (s == 0x123456789abcdefull) out[tid] = s;  // keeps the chains alive, practically never taken
}
