// test_hooks.cuh -- entry points of libzippel_test.so only (include/zippel_test.h): the substrate self-test, the
// multiplier-pipe micro-benchmarks, and direct doors to the NTT engine and to the intermediates of the sub-quadratic
// route.  Compiled into zippel_capi.cu when ZP_TEST_HOOKS is defined; libzippel.so, the product, has none of this.
// This file is included INSIDE the extern "C" block of zippel_capi.cu; kernels therefore come first, wrapped in
// extern "C++".
extern "C++" {
#include "ubench.cuh"

// (a0) self-test kernel for the substrate
__global__ void k_modarith_selftest(int op, const uint64_t* a, const uint64_t* b, int64_t n, ZpMod k, uint64_t* out) {
  if (op == 5) {  // deferred dot through the wide accumulator, one CTA
    __shared__ uint64_t part[256];
    Acc acc;
    acc_zero(acc);
    for (int64_t i = threadIdx.x; i < n; i += blockDim.x) acc_mac(acc, to_mont(zp_canon(a[i], k.p), k), b[i]);
    part[threadIdx.x] = mont_mul(acc_redc160(acc, k), k.c160, k);  // mont * plain -> plain
    __syncthreads();
    if (threadIdx.x == 0) {
      uint64_t r = 0;
      for (int x = 0; x < (int)blockDim.x; ++x) r = mod_add(r, part[x], k.p);
      out[0] = r;
    }
    return;
  }
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const uint64_t x = zp_canon(a[i], k.p), y = b ? b[i] : 0;
    uint64_t r = 0;
    if (op == 0) r = from_mont(mont_mul(to_mont(x, k), to_mont(zp_canon(y, k.p), k), k), k);
    if (op == 1) r = mod_add(x, zp_canon(y, k.p), k.p);
    if (op == 2) r = mod_sub(x, zp_canon(y, k.p), k.p);
    if (op == 3) r = from_mont(mont_pow(to_mont(x, k), y, k), k);
    if (op == 4) r = from_mont(mont_inv(to_mont(x, k), k), k);
    if (op == 6) {  // Horner step on a LAZY x (any 64-bit value): (y x + a[(i+1) % n]) mod p
      const uint64_t m = zp_canon(y, k.p), ad = zp_canon(a[(i + 1) % n], k.p);
      r = lazy_canon(horner_step(a[i], m, shoup_companion(to_mont(m, k), k), ad, shoup_companion(to_mont(ad, k), k), k), k.p);
    }
    out[i] = r;
  }
}

// linear product through the NTT engine: X[0] = a, X[1] = b zero-padded to n = 2^logn
__global__ void k_test_pm_prep(const uint64_t* __restrict__ a, int64_t na, const uint64_t* __restrict__ b, int64_t nb, int logn,
                               ZpMod kp, uint64_t* __restrict__ X) {
  const int64_t n = (int64_t)1 << logn, EX = 2 * n;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < EX; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = e & (n - 1);
    uint64_t v = 0;
    if (e < n) v = i < na ? zp_canon(a[i], kp.p) : 0;
    else v = i < nb ? zp_canon(b[i], kp.p) : 0;
    X[e] = v;
    X[EX + e] = v;
    X[2 * EX + e] = v;
  }
}
__global__ void k_test_pm_fin(const uint64_t* __restrict__ O, int logn, int64_t nout, NttCtx cx, CrtOut co, ZpMod kp,
                              uint64_t* __restrict__ out) {
  const int64_t n = (int64_t)1 << logn;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nout; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = ntt_crt(O[i], O[n + i], O[2 * n + i], cx, co, kp);
}
// round-trip helper: canonicalise the words of x (lazy, < 4q) and, if scale, multiply them by 1/n -- what the pointwise
// product does between the forward and the inverse transform (the inverse butterflies take values below 2q)
__global__ void k_test_canon(uint64_t* __restrict__ x, int64_t E, int scale, NttCtx cx, uint64_t Kq0, uint64_t Kq1, uint64_t Kq2) {
  const int j = blockIdx.y;
  const ZpMod q = cx.q[j];
  const uint64_t Kq = j == 0 ? Kq0 : j == 1 ? Kq1 : Kq2;  // 2^128 / n
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < E; e += (int64_t)gridDim.x * blockDim.x) {
    uint64_t v = x[(int64_t)j * E + e];
    v = (v >= 2 * q.p) ? v - 2 * q.p : v;
    v = lazy_canon(v, q.p);
    x[(int64_t)j * E + e] = scale ? mont_mul(mont_mul(v, 1, q), Kq, q) : v;  // v 2^-64 2^128/n 2^-64 = v / n
  }
}
}  // extern "C++"

int zippel_modarith_selftest(int op, const uint64_t* a, const uint64_t* b, int64_t n, uint64_t p, uint64_t* out,
                             void* stream) {
  ZpMod k;
  if (!a || !out || n <= 0 || op < 0 || op > 6 || !make_mod(p, &k) || ((op <= 3 || op >= 5) && !b)) return ZP_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (op == 5) {
    ++g_launches, k_modarith_selftest<<<1, 256, 0, st>>>(op, a, b, n, k, out);
  } else {
    int64_t blocks = (n + 255) / 256;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    ++g_launches, k_modarith_selftest<<<(unsigned)blocks, 256, 0, st>>>(op, a, b, n, k, out);
  }
  return cuda_ok();
}

int zippel_ubench(int kind, int iters, int blocks, uint64_t p, uint64_t* out, double* h_chain_steps, void* stream) {
  ZpMod k;
  if (kind < 0 || kind > 21 || iters <= 0 || blocks <= 0 || !out || !make_mod(p, &k)) return ZP_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
#define ZP_UB(K) case K: ++g_launches, k_ubench<K><<<blocks, ZP_UB_THREADS, 0, st>>>(iters, k, out); break;
  switch (kind) { ZP_UB(0) ZP_UB(1) ZP_UB(2) ZP_UB(3) ZP_UB(4) ZP_UB(5) ZP_UB(6) ZP_UB(7) ZP_UB(8) ZP_UB(9) ZP_UB(10) ZP_UB(11) ZP_UB(12) ZP_UB(13) ZP_UB(14) ZP_UB(15) ZP_UB(16) ZP_UB(17) ZP_UB(18) ZP_UB(19) ZP_UB(20) ZP_UB(21) }
#undef ZP_UB
  if (h_chain_steps) *h_chain_steps = (double)blocks * ZP_UB_THREADS * (double)iters * 8.0 * ZP_UB_CH;
  return cuda_ok();
}

// the constants of the NTT engine, for the CPU-side pin (tests/test_ntt_constants.py):
// out[0..2] = q1, q2, q3;  out[3..5] = their roots of unity of order 2^24 (plain);  out[6] = 24
void zippel_test_ntt_constants(uint64_t* h_out) {
  const SqHost& H = sq_host();
  for (int j = 0; j < 3; ++j) {
    h_out[j] = kNttQ[j];
    h_out[3 + j] = h_mulmod(H.wroot_mont[j], h_invmod(H.cx.q[j].r1, kNttQ[j]), kNttQ[j]);
  }
  h_out[6] = ZP_NTT_LOGMAX;
}

size_t zippel_test_polymul_workspace_bytes(int64_t na, int64_t nb) {
  if (na <= 0 || nb <= 0 || na + nb - 1 > ((int64_t)1 << ZP_NTT_LOGMAX)) return 0;
  const int64_t n = (int64_t)1 << ceil_log2(na + nb - 1);
  return al(16 * (size_t)12 * ZP_NTT_TAB) + al(8 * 3 * 2 * (size_t)n) + al(8 * 3 * (size_t)n);
}
// out[0 .. na+nb-1) = a * b mod p by one cyclic convolution of length 2^ceil(log2(na+nb-1)) modulo the three primes.
// roundtrip != 0: instead, out[0 .. 3n) = inverse(forward(X)) / n for X = [a | b] zero-padded (must equal the input
// residues modulo each prime); n = 2^ceil(log2(na+nb-1)), out holds 6 n words.
int zippel_test_polymul(const uint64_t* a, int64_t na, const uint64_t* b, int64_t nb, uint64_t p, uint64_t* out,
                        int roundtrip, void* workspace, size_t workspace_bytes, void* stream) {
  ZpMod k;
  if (!a || !b || !out || !make_mod(p, &k) || !ws_ok(workspace, workspace_bytes, zippel_test_polymul_workspace_bytes(na, nb)) ||
      zippel_test_polymul_workspace_bytes(na, nb) == 0)
    return ZP_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int logn = ceil_log2(na + nb - 1 > 2 ? na + nb - 1 : 2);
  const int64_t n = (int64_t)1 << logn;
  Ws w;
  memset(&w, 0, sizeof(w));
  char* base = (char*)workspace;
  w.ntt_tab = (ulonglong2*)base;
  uint64_t* X = (uint64_t*)(base + al(16 * (size_t)12 * ZP_NTT_TAB));
  uint64_t* O = (uint64_t*)((char*)X + al(8 * 3 * 2 * (size_t)n));
  const NttCtx cx = ntt_begin(w, st);
  ++g_launches, k_test_pm_prep<<<sq_blocks(2 * n), 256, 0, st>>>(a, na, b, nb, logn, k, X);
  if (roundtrip) {
    ntt_run(false, X, 2 * n, logn, cx, st);
    uint64_t Kq[3];
    make_kq(logn, Kq);
    ++g_launches, k_test_canon<<<dim3(sq_blocks(2 * n), 3), 256, 0, st>>>(X, 2 * n, 1, cx, Kq[0], Kq[1], Kq[2]);
    ntt_run(true, X, 2 * n, logn, cx, st);
    ++g_launches, k_test_canon<<<dim3(sq_blocks(2 * n), 3), 256, 0, st>>>(X, 2 * n, 0, cx, Kq[0], Kq[1], Kq[2]);
    cudaMemcpyAsync(out, X, 8 * 6 * (size_t)n, cudaMemcpyDeviceToDevice, st);
    return cuda_ok();
  }
  ntt_mul_pairs(X, 2 * n, O, logn, cx, st);
  ++g_launches, k_test_pm_fin<<<sq_blocks(na + nb - 1), 256, 0, st>>>(O, logn, na + nb - 1, cx, make_crt_out(k, 0), k, out);
  return cuda_ok();
}

// Intermediates of the sub-quadratic route: the next solve that takes it copies stage `stage` to `out` (device):
//   1 top-level master polynomials [T] (Montgomery form), 2 alpha = 1/rev(M) of the LAST function (Montgomery),
//   3 root tails [(B+1) x T], 4 leaf tails [(B+1) x T], 5 numerators [(B+1) x T]; 0 switches the dump off.
int zippel_test_subq_dump(int stage, uint64_t* out) {
  g_sq_dump_stage = stage;
  g_sq_dump_out = out;
  return ZP_OK;
}
