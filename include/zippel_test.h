/*
 * zippel_test.h -- entry points of libzippel_test.so, the TEST AND MEASUREMENT build of the library: everything in
 * include/zippel.h (same sources) plus the hooks below.  libzippel.so, the product, exports none of them.
 * Same conventions as zippel.h (device pointers unless h_, asynchronous on `stream`, ZP_* return codes).
 */
#ifndef ZIPPEL_TEST_H
#define ZIPPEL_TEST_H

#include "zippel.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Self-test hook for the arithmetic substrate (a0), section 2.1: out[i] = op(a[i], b[i]) mod p,
 * op: 0 mul, 1 add, 2 sub, 3 pow (b = exponent), 4 inverse of a (0 -> 0),
 *     5 deferred dot: out[0] = sum_i a[i]*b[i] mod p through the 160-bit accumulator,
 *     6 Horner step: out[i] = (b[i] * a[i] + a[(i+1) % n]) mod p, where the multiplicand a[i] is taken as a
 *       LAZY value (any 64-bit number, not reduced first) -- the hot recurrence of (a3). */
int zippel_modarith_selftest(int op, const uint64_t* a, const uint64_t* b, int64_t n, uint64_t p, uint64_t* out,
                             void* stream);

/* Roofline micro-benchmarks of the integer multiplier pipe:
 * launches `blocks` CTAs of 256 lanes, each running `iters` x 64 statements of `kind` per chain group
 * (kinds: csrc/ubench.cuh).  out: device scratch [blocks * 256].  *h_chain_steps (host, optional)
 * receives the number of lane-statements executed, for the caller to divide by its event time. */
int zippel_ubench(int kind, int iters, int blocks, uint64_t p, uint64_t* out, double* h_chain_steps, void* stream);

/* Constants of the three-prime NTT engine (csrc/ntt.cuh), host only, no device needed:
 * h_out[0..2] = q1 > q2 > q3, h_out[3..5] = their roots of unity of order 2^24 (plain residues), h_out[6] = 24. */
void zippel_test_ntt_constants(uint64_t* h_out);

/* A product of two polynomials over Z/pZ through the NTT engine (csrc/ntt.cuh): out[0 .. na+nb-1) = a * b mod p,
 * one cyclic convolution of length n = 2^ceil(log2(na+nb-1)) <= 2^24 modulo the three primes + CRT.
 * roundtrip != 0: out [6 n] = inverse(forward([a | b] zero-padded)) / n per prime (must reproduce the input). */
size_t zippel_test_polymul_workspace_bytes(int64_t na, int64_t nb);
int zippel_test_polymul(const uint64_t* a, int64_t na, const uint64_t* b, int64_t nb, uint64_t p, uint64_t* out,
                        int roundtrip, void* workspace, size_t workspace_bytes, void* stream);

/* Intermediates of the sub-quadratic solve (csrc/subq.cuh): the next call that takes that route copies one stage to
 * `out` (device, caller-sized): 1 = top-level master polynomials [T_run] in Montgomery form (x 2^64 mod p),
 * 2 = alpha = 1 / rev(M) mod x^k of the run's last function (Montgomery form), 3 = root tails [(B+1) x T_run],
 * 4 = leaf tails [(B+1) x T_run], 5 = unscaled numerators [(B+1) x T_run]; 0 = off.  Process-wide, not thread-safe. */
int zippel_test_subq_dump(int stage, uint64_t* out);

#ifdef __cplusplus
}
#endif
#endif
