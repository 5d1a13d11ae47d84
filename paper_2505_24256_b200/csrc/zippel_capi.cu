// zippel_capi.cu -- the C-ABI boundary (include/zippel.h): argument checks, Montgomery constants,
// workspace carving and kernel launches.  No torch types, no allocation, no CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/zippel.h"
#include "kernels.cuh"
#include "subq.cuh"
#include "small.cuh"

namespace {

typedef unsigned __int128 u128;

// ---- host: Montgomery constants for an odd p < 2^63 -------------------------------------------
bool make_mod(uint64_t p, ZpMod* k) {
  if (p < 3 || (p & 1) == 0 || (p >> 63)) return false;
  k->p = p;
  k->p0 = (uint32_t)p;
  k->p1 = (uint32_t)(p >> 32);
  uint32_t inv = 1;  // Newton: inv = p^-1 mod 2^32
  for (int i = 0; i < 5; ++i) inv *= 2u - (uint32_t)p * inv;
  k->pinv = 0u - inv;
  auto pow2 = [&](int e) {  // 2^e mod p
    uint64_t r = 1 % p;
    for (int i = 0; i < e; ++i) r = (uint64_t)(((u128)r * 2) % p);
    return r;
  };
  k->r1 = pow2(64);
  k->r2 = pow2(128);
  k->c96 = pow2(96);
  k->c160 = pow2(160);
  k->c224 = pow2(224);
  k->np = 0ull - p;
  uint64_t inv64 = 1;  // Newton: inv64 = p^-1 mod 2^64
  for (int i = 0; i < 6; ++i) inv64 *= 2ull - p * inv64;
  k->ninv64 = 0ull - inv64;
  return true;
}

// ---- sub-quadratic route (subq.cuh): host constants, plan, workspace sizes -----------------------------------------
// The three NTT primes q = c 2^26 + 1 just below 2^62 and a generator of their 2-power subgroups (x^((q-1)/2^24) has
// order 2^24); tests/test_ntt_constants.py re-derives both facts with Python integers through zippel_ntt_constants().
const uint64_t kNttQ[3] = {4611686017554972673ull, 4611686015004835841ull, 4611686009971671041ull};
const uint64_t kNttGen[3] = {5, 3, 3};
int64_t g_subq_min_t = 0;  // > 0: functions with at least this many terms take the sub-quadratic route (zippel_set_tuning);
                           // 0: the measured rule of sq_threshold below

uint64_t h_mulmod(uint64_t a, uint64_t b, uint64_t m) { return (uint64_t)((u128)a * b % m); }
uint64_t h_powmod(uint64_t a, uint64_t e, uint64_t m) {
  uint64_t r = 1 % m;
  a %= m;
  while (e) {
    if (e & 1) r = h_mulmod(r, a, m);
    a = h_mulmod(a, a, m);
    e >>= 1;
  }
  return r;
}
uint64_t h_invmod(uint64_t a, uint64_t m) { return h_powmod(a, m - 2, m); }  // m prime

struct SqHost {
  NttCtx cx;               // table pointers are filled per call
  uint64_t wroot_mont[3];  // the root of order 2^24 of each prime, Montgomery form
};
const SqHost& sq_host() {
  static const SqHost H = [] {
    SqHost h;
    memset(&h, 0, sizeof(h));
    for (int j = 0; j < 3; ++j) {
      const uint64_t q = kNttQ[j];
      make_mod(q, &h.cx.q[j]);
      const uint64_t w = h_powmod(kNttGen[j], (q - 1) >> ZP_NTT_LOGMAX, q);
      h.wroot_mont[j] = h_mulmod(w, h.cx.q[j].r1, q);
    }
    const uint64_t q1 = kNttQ[0], q2 = kNttQ[1], q3 = kNttQ[2];
    h.cx.g2 = h_mulmod(h_invmod(q1 % q2, q2), h.cx.q[1].r1, q2);
    h.cx.g3a = h_mulmod(q1 % q3, h.cx.q[2].r1, q3);
    h.cx.g3b = h_mulmod(h_invmod(h_mulmod(q1 % q3, q2 % q3, q3), q3), h.cx.q[2].r1, q3);
    return h;
  }();
  return H;
}
// c K mod p with K = 2^(-64 kexp)
CrtOut make_crt_out(const ZpMod& k, int kexp) {
  const uint64_t p = k.p;
  const uint64_t K = h_powmod((p + 1) / 2, 64 * (uint64_t)kexp, p);  // (1/2)^(64 kexp): p odd
  CrtOut co;
  co.C1 = h_mulmod(K, k.r1, p);
  co.C2 = h_mulmod(co.C1, kNttQ[0] % p, p);
  co.C3 = h_mulmod(co.C2, kNttQ[1] % p, p);
  return co;
}
// 2^128 / n mod q_j
void make_kq(int logn, uint64_t Kq[3]) {
  for (int j = 0; j < 3; ++j) {
    const uint64_t q = kNttQ[j];
    const ZpMod& m = sq_host().cx.q[j];
    Kq[j] = h_mulmod(m.r2, h_powmod((q + 1) / 2, (uint64_t)logn, q), q);
  }
}

inline int ceil_log2(int64_t x) {
  int l = 0;
  while (((int64_t)1 << l) < x) ++l;
  return l;
}

// one run of consecutive long functions [f0, f1): slots [a0, a0 + T)
struct SqRun {
  int f0, f1;
  int64_t a0, T, tmax;
  int nlev;  // levels 0 .. nlev; block size at level l = ZP_SQ_LEAF << l
};
struct SqSizes {
  bool any = false;
  int64_t maxT = 0, alphaN = 0, maxX = 0, maxY = 0, maxO = 0, maxTasks = 0, maxLeaves = 0, maxFns = 0, sumXl = 0, maxO2 = 0;
  int maxLev = 0, Vc = 1;
  int64_t thr = 0;  // the threshold the runs were found with (sq_threshold on the whole batch)
};
// Which functions take the sub-quadratic route: those with at least sq_threshold terms.  Measured on B200 (profiles/
// r02_crossover.md): a batch with enough functions to fill the GPU crosses over between t = 800 and t = 1000 for every B
// (one tree level above two leaves already halves the t^2 work of the leaves); a single function (or a few) is bound by
// the latency of the route's ~150 dependent launches and crosses over later, the later the fewer right-hand sides
// there are to amortise them (B = 1: 12288, B = 3: 8192, B = 9: 4096, B = 21: 2048).
#define ZP_SQ_BATCH_T 960
int64_t sq_threshold(const int64_t* h_offs, int F, int B) {
  if (g_subq_min_t > 0) return g_subq_min_t;
  int64_t sum = 0;
  for (int f = 0; f < F; ++f) {
    const int64_t t = h_offs[f + 1] - h_offs[f];
    if (t >= ZP_SQ_BATCH_T) sum += t;
  }
  if (sum >= 65536) return ZP_SQ_BATCH_T;
  return B >= 16 ? 2048 : B >= 6 ? 4096 : B >= 2 ? 8192 : 12288;
}
// leaves of the sub-quadratic route: blocks of at most this many nodes are solved by the quadratic kernels (at most ZP_LEAF)
#ifndef ZP_SQ_LEAF
#define ZP_SQ_LEAF 512
#endif
inline bool sq_is_long(int64_t t, int64_t thr) { return t >= thr && t > ZP_SQ_LEAF; }

// pair and copy tasks of level l (children of size a = LEAF << l) for a run; slots relative to the run
void sq_level_tasks(const int64_t* h_offs, const SqRun& r, int l, std::vector<SqTask>* pairs, std::vector<SqTask>* copies) {
  const int64_t a = (int64_t)ZP_SQ_LEAF << l;
  for (int f = r.f0; f < r.f1; ++f) {
    const int64_t off = h_offs[f] - r.a0, t = h_offs[f + 1] - h_offs[f];
    int64_t base = 0;
    for (; base + a < t; base += 2 * a) {
      const int64_t b = (t - base - a < a) ? t - base - a : a;
      if (pairs) pairs->push_back(SqTask{off + base, (int32_t)a, (int32_t)b});
    }
    if (base < t && copies) {  // a last block without a sibling (or a function already complete): copy through, in
      for (int64_t c = base; c < t; c += ((int64_t)1 << 30))  // pieces that fit the 32-bit length field
        copies->push_back(SqTask{off + c, (int32_t)((t - c < ((int64_t)1 << 30)) ? t - c : ((int64_t)1 << 30)), 0});
    }
  }
}

void sq_find_runs(const int64_t* h_offs, int F, int64_t thr, std::vector<SqRun>* runs) {
  for (int f = 0; f < F;) {
    if (!sq_is_long(h_offs[f + 1] - h_offs[f], thr)) {
      ++f;
      continue;
    }
    SqRun r;
    r.f0 = f;
    r.tmax = 0;
    while (f < F && sq_is_long(h_offs[f + 1] - h_offs[f], thr)) {
      const int64_t t = h_offs[f + 1] - h_offs[f];
      r.tmax = t > r.tmax ? t : r.tmax;
      ++f;
    }
    r.f1 = f;
    r.a0 = h_offs[r.f0];
    r.T = h_offs[r.f1] - r.a0;
    r.nlev = ceil_log2((r.tmax + ZP_SQ_LEAF - 1) / ZP_SQ_LEAF);
    runs->push_back(r);
  }
}

SqSizes sq_sizes(const int64_t* h_offs, int F, int B) {
  SqSizes z;
  z.thr = sq_threshold(h_offs, F, B);
  std::vector<SqRun> runs;
  sq_find_runs(h_offs, F, z.thr, &runs);
  if (runs.empty()) return z;
  z.any = true;
  auto mx = [](int64_t& a, int64_t b) { a = b > a ? b : a; };
  for (const SqRun& r : runs) mx(z.maxT, r.T);
  // vectors per down-tree chunk: the product buffer holds 2 Vc T words per prime; cap it at 2^27 words in all
  int64_t vc = ((int64_t)1 << 27) / (6 * z.maxT);
  z.Vc = (int)(vc < 1 ? 1 : (vc > B + 1 ? B + 1 : vc));
  for (const SqRun& r : runs) {
    z.maxLev = r.nlev > z.maxLev ? r.nlev : z.maxLev;
    int64_t ntasks = 0, leaves = 0, sumXl = 0;
    for (int l = 0; l < r.nlev; ++l) {
      std::vector<SqTask> pairs, copies;
      sq_level_tasks(h_offs, r, l, &pairs, &copies);
      const int64_t n = (int64_t)2 * ZP_SQ_LEAF << l, P = (int64_t)pairs.size();
      sumXl += 2 * P * n;  // the level's transformed (reversed) children stay for the down-tree
      mx(z.maxO, P * n);
      mx(z.maxY, z.Vc * P * n);
      mx(z.maxO, 2 * z.Vc * P * n);
      ntasks += (int64_t)pairs.size() + (int64_t)copies.size();
    }
    mx(z.maxTasks, ntasks);
    mx(z.sumXl, sumXl);
    int64_t sumK = 0, sumR = 0;  // the functions of a run take the Newton steps and the root products together
    for (int f = r.f0; f < r.f1; ++f) {
      const int64_t t = h_offs[f + 1] - h_offs[f];
      leaves += (t + ZP_SQ_LEAF - 1) / ZP_SQ_LEAF;
      int64_t kf = ZP_SQ_KB;
      while (kf < t) kf <<= 1;
      sumK += kf;                                 // final precision of alpha; Newton's last step: n = kf
      sumR += (int64_t)1 << ceil_log2(2 * t);     // root product
    }
    mx(z.alphaN, sumK);
    mx(z.maxX, 2 * (sumK > sumR ? sumK : sumR));
    mx(z.maxO2, sumK > sumR ? sumK : sumR);
    mx(z.maxFns, r.f1 - r.f0);
    mx(z.maxLeaves, leaves);
  }
  return z;
}

// ---- workspace ----------------------------------------------------------------------------------
struct Ws {
  int64_t* d_offsets;
  int32_t *st_pre, *st_solve, *st_newton;
  uint64_t *nodes, *M0, *M1, *scale, *R, *V, *newtI, *newtL;
  ulonglong2 *invd, *smont;  // Newton: {w, w'} tables
  ulonglong4* tab;
  // sub-quadratic route (null unless some function is long)
  SqSizes sq;
  ulonglong2* ntt_tab;  // [3][4][4096]: U, Ui, Tlo, Thi per prime
  SqTask* sq_tasks;
  SqFn* sq_fns;
  int64_t* sq_leafoffs;
  uint64_t *sq_lev, *sq_tailA, *sq_tailB, *sq_alpha, *sq_X, *sq_Xl, *sq_Y, *sq_O, *sq_O2;
  size_t bytes;
};

inline size_t al(size_t x) { return (x + 255) & ~(size_t)255; }

Ws carve(void* base, int64_t T_tot, int F, int B, int flags, const SqSizes& sq = SqSizes()) {
  Ws w;
  size_t o = 0;
  auto take = [&](size_t n) {
    char* p = base ? (char*)base + o : nullptr;
    o += al(n);
    return (void*)p;
  };
  w.d_offsets = (int64_t*)take(sizeof(int64_t) * (size_t)(F + 1));
  w.st_pre = (int32_t*)take(sizeof(int32_t) * (size_t)F);
  w.st_solve = (int32_t*)take(sizeof(int32_t) * (size_t)F);
  w.st_newton = (int32_t*)take(sizeof(int32_t) * 4);
  w.nodes = (uint64_t*)take(8 * (size_t)T_tot);
  w.M0 = (uint64_t*)take(8 * (size_t)T_tot);
  w.M1 = (uint64_t*)take(8 * (size_t)T_tot);
  w.scale = (uint64_t*)take(8 * (size_t)T_tot);
  w.tab = (ulonglong4*)take(32 * (size_t)T_tot);
  w.invd = (ulonglong2*)take(16 * (size_t)B * B);
  w.smont = (ulonglong2*)take(16 * (size_t)B);
  w.newtI = (uint64_t*)take(8 * (size_t)B * B);  // identity, then L = k_newton(identity)
  w.newtL = (uint64_t*)take(8 * (size_t)B * B);
  w.R = (uint64_t*)take(8 * (size_t)T_tot);
  w.V = (flags & ZP_WS_BALANCED) ? (uint64_t*)take(8 * (size_t)T_tot * B) : nullptr;
  w.sq = sq;
  w.ntt_tab = nullptr;
  if (sq.any) {
    w.ntt_tab = (ulonglong2*)take(16 * (size_t)12 * ZP_NTT_TAB);
    w.sq_tasks = (SqTask*)take(sizeof(SqTask) * (size_t)(sq.maxTasks + 1));
    w.sq_fns = (SqFn*)take(sizeof(SqFn) * (size_t)(sq.maxFns + 1));
    w.sq_leafoffs = (int64_t*)take(8 * (size_t)(sq.maxLeaves + 1));
    w.sq_lev = (uint64_t*)take(8 * (size_t)(sq.maxLev + 1) * sq.maxT);
    w.sq_tailA = (uint64_t*)take(8 * (size_t)(B + 1) * sq.maxT);
    w.sq_tailB = (uint64_t*)take(8 * (size_t)(B + 1) * sq.maxT);
    w.sq_alpha = (uint64_t*)take(8 * (size_t)sq.alphaN);
    w.sq_X = (uint64_t*)take(8 * 3 * (size_t)sq.maxX);
    w.sq_Xl = (uint64_t*)take(8 * 3 * (size_t)sq.sumXl);  // per tree level: the transforms of the reversed children
    w.sq_Y = (uint64_t*)take(8 * 3 * (size_t)sq.maxY);
    w.sq_O = (uint64_t*)take(8 * 3 * (size_t)sq.maxO);
    w.sq_O2 = (uint64_t*)take(8 * 3 * (size_t)sq.maxO2);  // products of the Newton chain (second stream)
  }
  w.bytes = o;
  return w;
}

bool check_offsets(const int64_t* h, int F, int64_t* T_tot, int64_t* tmax) {
  if (!h || F <= 0 || h[0] != 0) return false;
  int64_t mx = 0;
  for (int f = 0; f < F; ++f) {
    const int64_t t = h[f + 1] - h[f];
    if (t <= 0 || t >= ((int64_t)1 << 23)) return false;  // status index field; NTT length (zippel.h)
    if (t > mx) mx = t;
  }
  if (h[F] >= ((int64_t)1 << 31)) return false;
  *T_tot = h[F];
  *tmax = mx;
  return true;
}

// ---- measurement hook (zippel_profile_events) ----------------------------------------------------
unsigned long long g_launches = 0;  // kernels enqueued by this library in this process
int g_prof_kernel = 0, g_prof_ordinal = -1, g_prof_seen = 0;
cudaEvent_t g_prof_start = nullptr, g_prof_stop = nullptr;
struct ProfScope {  // records start at construction and stop at destruction when `kernel` is the hooked one
  bool on;
  cudaStream_t st;
  ProfScope(int kernel, cudaStream_t s) : on(false), st(s) {
    if (kernel == g_prof_kernel && g_prof_start && g_prof_stop) {
      on = g_prof_ordinal < 0 || g_prof_seen == g_prof_ordinal;  // ordinal: n-th occurrence since the hook was set
      ++g_prof_seen;
    }
    if (on) cudaEventRecord(g_prof_start, st);
  }
  ~ProfScope() {
    if (on) cudaEventRecord(g_prof_stop, st);
  }
};

inline int cuda_ok() { return cudaGetLastError() == cudaSuccess ? ZP_OK : ZP_ERR_CUDA; }
// SMs of the current device (grid caps of the grid-stride kernels are multiples of it)
int sm_count() {
  static int n_cached[16] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 16) return 148;
  if (!n_cached[dev]) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    n_cached[dev] = n;
  }
  return n_cached[dev];
}
inline unsigned grid_y(int F) { return (unsigned)(F < 65535 ? F : 65535); }
// CTAs of k_inv_finish (128 lanes, ZP_INV_N slots per lane) for n slots
inline unsigned inv_blocks(int64_t n) { return (unsigned)((n + 4 * 32 * ZP_INV_N - 1) / (4 * 32 * ZP_INV_N)); }

// ---- K3 dispatch ----------------------------------------------------------------------------------
#define ZP_NB_MAX 25

template <int NB>
void launch_node_solve(dim3 grid, cudaStream_t st, const uint64_t* nodes, const ulonglong4* M, const int64_t* offs, int F,
                       const uint64_t* vals, int64_t T_tot, int b0, int s0, const ZpMod& k, uint64_t* scale,
                       uint64_t* coefs, int32_t* status) {
  ++g_launches, k_node_solve<NB><<<grid, ZP_K3_THREADS, 0, st>>>(nodes, M, offs, F, vals, T_tot, b0, s0, k, scale, coefs, status);
}

void dispatch_node_solve(int nb, dim3 grid, cudaStream_t st, const uint64_t* nodes, const ulonglong4* M,
                         const int64_t* offs, int F, const uint64_t* vals, int64_t T_tot, int b0, int s0,
                         const ZpMod& k, uint64_t* scale, uint64_t* coefs, int32_t* status) {
#define ZP_CASE(N) \
  case N: launch_node_solve<N>(grid, st, nodes, M, offs, F, vals, T_tot, b0, s0, k, scale, coefs, status); break;
  switch (nb) {
    ZP_CASE(1) ZP_CASE(2) ZP_CASE(3) ZP_CASE(4) ZP_CASE(5) ZP_CASE(6) ZP_CASE(7) ZP_CASE(8) ZP_CASE(9)
    ZP_CASE(10) ZP_CASE(11) ZP_CASE(12) ZP_CASE(13) ZP_CASE(14) ZP_CASE(15) ZP_CASE(16) ZP_CASE(17)
    ZP_CASE(18) ZP_CASE(19) ZP_CASE(20) ZP_CASE(21) ZP_CASE(22) ZP_CASE(23) ZP_CASE(24) ZP_CASE(25)
    default: break;
  }
#undef ZP_CASE
}

#define ZP_EVAL2_MIN_T 4096  // B = 1: from this skeleton length on the correlation + two-chain path is used

// ---- stages (device offsets already in w.d_offsets) ---------------------------------------------
// (a2) master polynomial of every function -> returns the buffer holding M' (Montgomery)
const uint64_t* run_master_poly(const Ws& w, const uint64_t* nodes, int F, int64_t tmax, const ZpMod& k,
                                cudaStream_t st) {
  ProfScope prof(ZP_K_MASTER_POLY, st);
  dim3 g((unsigned)((tmax + ZP_LEAF - 1) / ZP_LEAF), grid_y(F));
  ++g_launches, k_tree_leaf<<<g, ZP_K2_THREADS, 0, st>>>(nodes, w.d_offsets, F, k, w.M0);
  uint64_t *src = w.M0, *dst = w.M1;
  for (int64_t a = ZP_LEAF; a < tmax; a <<= 1) {
    dim3 gl((unsigned)((tmax + ZP_K2_TC - 1) / ZP_K2_TC), grid_y(F));
    ++g_launches, k_tree_level<<<gl, ZP_K2_TC, 0, st>>>(src, w.d_offsets, F, a, k, dst);
    uint64_t* tmp = src;
    src = dst;
    dst = tmp;
  }
  return src;
}

// ---- sub-quadratic route: launches ---------------------------------------------------------------------------------
inline unsigned sq_blocks(int64_t n, int per = 256) {
  int64_t b = (n + per - 1) / per;
  const int64_t cap = (int64_t)sm_count() * 64;
  return (unsigned)(b < 1 ? 1 : (b > cap ? cap : b));
}
// The route is a chain of some two hundred dependent launches, many of them a few microseconds long: they are launched
// with programmatic stream serialization, so that a kernel becomes resident while its predecessor drains (every kernel
// launched this way starts with zp_grid_dep_wait(), modarith.cuh: the order of the memory operations is that of a plain
// launch).  g_launches counts them like the others.
template <typename... P, typename... A>
inline void launch_dep(void (*kern)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  ++g_launches;
  cudaLaunchKernelEx(&cfg, kern, static_cast<P>(args)...);
}
// Pass plan of a transform of length 2^logn (ntt.cuh): up to two strided passes of lr1 and lr2 stages, then the chunk
// stages (lc <= 12 of them) on rows that are twisted by their parent's row index (lrp stages above them).
struct NttPlan {
  int lr1 = 0, lr2 = 0, lc, lrp;
};
NttPlan ntt_plan(int logn) {
  NttPlan pl;
  if (logn > ZP_NTT_LOGC) {
    const int e = logn - ZP_NTT_LOGC;
    if (e <= 9) pl.lr1 = e;
    else pl.lr1 = (e + 1) / 2, pl.lr2 = e - pl.lr1;
  }
  pl.lc = logn - pl.lr1 - pl.lr2;
  pl.lrp = pl.lr2 ? pl.lr2 : pl.lr1;
  return pl;
}
inline dim3 ntt_grid(int64_t E) { return dim3((unsigned)((E + ZP_NTT_C - 1) / ZP_NTT_C), 3); }
// grids that do not fill the GPU run 512 lanes per CTA (one group per lane and round: half the latency per tile)
inline bool ntt_small_grid(int64_t E) { return 3 * ((E + ZP_NTT_C - 1) / ZP_NTT_C) < 2 * (int64_t)sm_count(); }
template <bool INV>
void ntt_pass_launch(uint64_t* buf, int64_t E, int logn, int logR, int logRp, const NttCtx& cx, cudaStream_t st) {
  if (ntt_small_grid(E))
    launch_dep(k_ntt_pass<INV, ZP_NTT_THREADS_SMALL>, ntt_grid(E), ZP_NTT_THREADS_SMALL, 0, st, buf, E, logn, logR, logRp, cx);
  else
    launch_dep(k_ntt_pass<INV, ZP_NTT_THREADS>, ntt_grid(E), ZP_NTT_THREADS, 0, st, buf, E, logn, logR, logRp, cx);
}
// the strided passes alone, on every segment of `buf` ([3][E] words, segments of 2^logn), in place
void ntt_strided(bool inverse, uint64_t* buf, int64_t E, int logn, const NttCtx& cx, cudaStream_t st) {
  const NttPlan pl = ntt_plan(logn);
  if (!inverse) {
    if (pl.lr1) ntt_pass_launch<false>(buf, E, logn, pl.lr1, 0, cx, st);
    if (pl.lr2) ntt_pass_launch<false>(buf, E, logn - pl.lr1, pl.lr2, pl.lr1, cx, st);
  } else {
    if (pl.lr2) ntt_pass_launch<true>(buf, E, logn - pl.lr1, pl.lr2, pl.lr1, cx, st);
    if (pl.lr1) ntt_pass_launch<true>(buf, E, logn, pl.lr1, 0, cx, st);
  }
}
// complete transforms of every segment, in place (one to three passes)
void ntt_run(bool inverse, uint64_t* buf, int64_t E, int logn, const NttCtx& cx, cudaStream_t st) {
  const NttPlan pl = ntt_plan(logn);
  if (!inverse) {
    ntt_strided(false, buf, E, logn, cx, st);
    ntt_pass_launch<false>(buf, E, pl.lc, 0, pl.lrp, cx, st);
  } else {
    ntt_pass_launch<true>(buf, E, pl.lc, 0, pl.lrp, cx, st);
    ntt_strided(true, buf, E, logn, cx, st);
  }
}
template <int MODE>
void ntt_mul_launch(int64_t Edrv, const uint64_t* A, int64_t EA, int64_t SA, const uint64_t* B, int64_t EB, uint64_t* O, int64_t EO, int lc,
                    int lrp, int logn, int64_t P, const NttCtx& cx, const uint64_t (&Kq)[3], cudaStream_t st) {
  const size_t smem = 16 * ZP_NTT_SMEM;
  if (ntt_small_grid(Edrv)) {
    cudaFuncSetAttribute(k_ntt_mul<MODE, ZP_NTT_THREADS_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    launch_dep(k_ntt_mul<MODE, ZP_NTT_THREADS_SMALL>, ntt_grid(Edrv), ZP_NTT_THREADS_SMALL, smem, st, A, EA, SA, B, EB, O, EO, lc, lrp, logn, P,
                                                                                                       cx, Kq[0], Kq[1], Kq[2]);
  } else {
    cudaFuncSetAttribute(k_ntt_mul<MODE, ZP_NTT_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    launch_dep(k_ntt_mul<MODE, ZP_NTT_THREADS>, ntt_grid(Edrv), ZP_NTT_THREADS, smem, st, A, EA, SA, B, EB, O, EO, lc, lrp, logn, P, cx, Kq[0],
                                                                                           Kq[1], Kq[2]);
  }
}
// products of segments of 2^logn words (k_ntt_mul): the strided passes on the operands, the fused chunk kernel, the
// strided passes on the product.
//   pairs: O segment o = X segment 2o * X segment 2o + 1 (EO = EX / 2); X is overwritten by its strided passes
//   keep: X ends up holding the COMPLETE forward transforms of its segments (the chunk stages are written back)
void ntt_mul_pairs(uint64_t* X, int64_t EX, uint64_t* O, int logn, const NttCtx& cx, cudaStream_t st, bool keep = false) {
  const NttPlan pl = ntt_plan(logn);
  const int64_t EO = EX / 2;
  uint64_t Kq[3];
  make_kq(logn, Kq);
  ntt_strided(false, X, EX, logn, cx, st);
  ntt_mul_launch<0>(EO, X, EX, EX, keep ? X : nullptr, 0, O, EO, pl.lc, pl.lrp, logn, 1, cx, Kq, st);
  ntt_strided(true, O, EO, logn, cx, st);
}
// copies of Y that k_sq_down_prepy writes: one serves the three primes when the transform has no strided pass
inline int ntt_down_copies(int logn) { return logn <= ZP_NTT_LOGC ? 1 : 3; }
//   down: O segments 2 vt + side = Y segment vt * Xhat segment 2 (vt mod P) + 1 - side (EO = 2 EY); Xhat holds the complete
//   transforms times 2^64 / n that ntt_mul_pairs(keep) left; Y is overwritten by its strided passes
void ntt_mul_down(uint64_t* Y, int64_t EY, const uint64_t* Xhat, int64_t EX, uint64_t* O, int logn, int64_t P, const NttCtx& cx,
                  cudaStream_t st) {
  const NttPlan pl = ntt_plan(logn);
  const int64_t EO = 2 * EY;
  uint64_t Kq[3];
  make_kq(logn, Kq);
  ntt_strided(false, Y, EY, logn, cx, st);
  ntt_mul_launch<1>(EY, Y, EY, ntt_down_copies(logn) == 1 ? 0 : EY, Xhat, EX, O, EO, pl.lc, pl.lrp, logn, P, cx, Kq, st);
  ntt_strided(true, O, EO, logn, cx, st);
}
// the per-call context: host constants + this workspace's tables (built by the first launch of the call)
NttCtx ntt_begin(const Ws& w, cudaStream_t st) {
  NttCtx cx = sq_host().cx;
  for (int j = 0; j < 3; ++j) {
    ulonglong2* t = w.ntt_tab + (size_t)j * 4 * ZP_NTT_TAB;
    cx.U[j] = t;
    cx.Ui[j] = t + ZP_NTT_TAB;
    cx.Tlo[j] = t + 2 * ZP_NTT_TAB;
    cx.Thi[j] = t + 3 * ZP_NTT_TAB;
    ++g_launches, k_ntt_tables<<<4 * ZP_NTT_TAB / 256, 256, 0, st>>>(cx.q[j], sq_host().wroot_mont[j], t, t + ZP_NTT_TAB,
                                                                   t + 2 * ZP_NTT_TAB, t + 3 * ZP_NTT_TAB);
  }
  return cx;
}

#ifdef ZP_TEST_HOOKS
int g_sq_dump_stage = 0;  // zippel_test_subq_dump
uint64_t* g_sq_dump_out = nullptr;
#define SQ_DUMP(stage, ptr, words) \
  if (g_sq_dump_stage == (stage) && g_sq_dump_out) cudaMemcpyAsync(g_sq_dump_out, (ptr), 8 * (size_t)(words), cudaMemcpyDeviceToDevice, st)
#else
#define SQ_DUMP(stage, ptr, words)
#endif

// second stream of the sub-quadratic route (created once per device, kept for the process; zippel_shutdown destroys
// it): the Newton iteration for the M' tail runs on it beside the value vectors' down-tree
struct SqAux {
  bool ready = false;
  cudaStream_t s2 = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
};
SqAux g_sqaux[16];
SqAux* get_sqaux() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 16) return nullptr;
  SqAux& A = g_sqaux[dev];
  if (!A.ready) {
    if (cudaStreamCreateWithFlags(&A.s2, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&A.ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&A.ev_join, cudaEventDisableTiming) != cudaSuccess)
      return nullptr;
    A.ready = true;
  }
  return &A;
}

// (a2)-(a4) for one run of long functions; nodes / vals / coefs point at the run's first slot (row strides ldv, ldc)
void sq_solve(const Ws& w, const NttCtx& cx, const int64_t* h_offs, const SqRun& r, const uint64_t* nodes,
              const uint64_t* vals, int64_t ldv, int B, int s0, const ZpMod& k, uint64_t* coefs, int64_t ldc,
              cudaStream_t st) {
  const int64_t T = r.T;
  const int Fr = r.f1 - r.f0;
  ProfScope prof(ZP_K_NODE_SOLVE, st);  // the whole route of the run: leaf trees, up-tree, tails, leaves, division
  const CrtOut co0 = make_crt_out(k, 0), co1 = make_crt_out(k, 1), co2 = make_crt_out(k, 2);
  (void)co0;
  // task lists of every level, and the leaf offsets: one upload per array
  std::vector<SqTask> tasks;
  std::vector<size_t> pair0(r.nlev + 1), copy0(r.nlev + 1), copy1(r.nlev + 1);
  for (int l = 0; l < r.nlev; ++l) {
    pair0[l] = tasks.size();
    sq_level_tasks(h_offs, r, l, &tasks, nullptr);
    copy0[l] = tasks.size();
    sq_level_tasks(h_offs, r, l, nullptr, &tasks);
    copy1[l] = tasks.size();
  }
  std::vector<int64_t> leafoffs;
  for (int f = r.f0; f < r.f1; ++f)
    for (int64_t x = h_offs[f]; x < h_offs[f + 1]; x += ZP_SQ_LEAF) leafoffs.push_back(x - r.a0);
  leafoffs.push_back(T);
  const int nleaves = (int)leafoffs.size() - 1;
  if (!tasks.empty()) cudaMemcpyAsync(w.sq_tasks, tasks.data(), sizeof(SqTask) * tasks.size(), cudaMemcpyHostToDevice, st);
  cudaMemcpyAsync(w.sq_leafoffs, leafoffs.data(), 8 * leafoffs.size(), cudaMemcpyHostToDevice, st);
  const int64_t* d_offs = w.d_offsets + r.f0;  // absolute slots: kernels that use them get pointers at slot 0 of the batch

  // (up) leaves, then one product per pair and level
  auto lev = [&](int l) { return w.sq_lev + (size_t)l * T; };
  std::vector<int64_t> xoff(r.nlev + 1, 0);  // words per prime of the levels below l in sq_Xl
  for (int l = 0; l < r.nlev; ++l) xoff[l + 1] = xoff[l] + 2 * (int64_t)(copy0[l] - pair0[l]) * ((int64_t)2 * ZP_SQ_LEAF << l);
  {
    ProfScope prof(ZP_K_MASTER_POLY, st);
    // the leaves as functions of at most ZP_SQ_LEAF nodes (run-local slots): one CTA builds each leaf's polynomial
    ++g_launches, k_tree_leaf<<<dim3(1, grid_y(nleaves)), ZP_K2_THREADS, 0, st>>>(nodes, w.sq_leafoffs, nleaves, k, lev(0));
    for (int l = 0; l < r.nlev; ++l) {
      const int logn = ceil_log2((int64_t)2 * ZP_SQ_LEAF << l);
      const int64_t n = (int64_t)1 << logn, P = (int64_t)(copy0[l] - pair0[l]);
      const SqTask* tp = w.sq_tasks + pair0[l];
      if (P) {
        const int64_t EX = 2 * P * n, EO = P * n;
        // the REVERSED children are multiplied (rev(A') rev(B') = rev(A' B')): their transforms are what the down-tree
        // correlates the tails with, and they are kept for it
        uint64_t* Xl = w.sq_Xl + 3 * xoff[l];
        launch_dep(k_sq_down_prepx, sq_blocks(EX), 256, 0, st, lev(l), tp, P, logn, Xl, EX);
        ntt_mul_pairs(Xl, EX, w.sq_O, logn, cx, st, true);
        launch_dep(k_sq_up_fin, sq_blocks(EO), 256, 0, st, lev(l), tp, P, logn, w.sq_O, EO, cx, co1, k, lev(l + 1));
      }
      const int nc = (int)(copy1[l] - copy0[l]);
      if (nc) launch_dep(k_sq_copy, dim3(64, (unsigned)(nc < 1024 ? nc : 1024)), 256, 0, st, w.sq_tasks + copy0[l], nc, lev(l), lev(l + 1), 1, 0);
    }
  }
  SQ_DUMP(1, lev(r.nlev), T);
  // root tails: rows 0 .. B-1 = the values; row B = rev(M') / rev(M) mod x^t per function
  const int V = B + 1;
  uint64_t *cur = w.sq_tailA, *nxt = w.sq_tailB;
  // The M' tail needs the power-series inverse of rev(M) (a chain of small dependent launches); the value vectors do
  // not: their down-tree runs on st while the Newton iteration runs on a second stream, then the M' vector follows.
  SqAux* aux = get_sqaux();
  const cudaStream_t sn = aux ? aux->s2 : st;
  int64_t dump_alpha_off = 0, dump_alpha_t = 0;  // (test hook: the longest function's inverse series)
  ++g_launches, k_sq_load_vals<<<dim3(sq_blocks(T), (unsigned)(B < 64 ? B : 64)), 256, 0, st>>>(vals, ldv, B, T, k, cur, T);
  {
    // the functions of the run, longest first: those still iterating at precision kk (t > kk) are a prefix
    std::vector<SqFn> fns;
    for (int f = r.f0; f < r.f1; ++f) fns.push_back(SqFn{h_offs[f] - r.a0, 0, h_offs[f + 1] - h_offs[f]});
    std::stable_sort(fns.begin(), fns.end(), [](const SqFn& a, const SqFn& b) { return a.t > b.t; });
    int64_t ao = 0;
    for (SqFn& fn : fns) {
      fn.aoff = ao;
      int64_t kf = ZP_SQ_KB;
      while (kf < fn.t) kf <<= 1;
      ao += kf;
    }
    cudaMemcpyAsync(w.sq_fns, fns.data(), sizeof(SqFn) * fns.size(), cudaMemcpyHostToDevice, st);
    if (aux) {  // fork: the second stream starts after everything queued on st so far (up-tree, uploads)
      cudaEventRecord(aux->ev_fork, st);
      cudaStreamWaitEvent(aux->s2, aux->ev_fork, 0);
    }
    const uint64_t* top = lev(r.nlev);
    ++g_launches, k_sq_inv_base<<<(unsigned)Fr, 512, 0, sn>>>(top, w.sq_fns, k, w.sq_alpha);
    for (int64_t kk = ZP_SQ_KB; kk < r.tmax; kk <<= 1) {  // precision kk -> 2 kk, products of length n = 2 kk
      int64_t nact = 0;
      while (nact < Fr && fns[nact].t > kk) ++nact;
      const int logn = ceil_log2(2 * kk);
      const int64_t n = 2 * kk, EX = 2 * nact * n;
      launch_dep(k_sq_newton_prep1, sq_blocks(EX), 256, 0, sn, top, w.sq_fns, nact, w.sq_alpha, logn, k, w.sq_X);
      ntt_mul_pairs(w.sq_X, EX, w.sq_O2, logn, cx, sn);
      launch_dep(k_sq_newton_mid, sq_blocks(EX), 256, 0, sn, w.sq_O2, w.sq_fns, nact, logn, cx, co1, k, w.sq_alpha, w.sq_X);
      ntt_mul_pairs(w.sq_X, EX, w.sq_O2, logn, cx, sn);
      launch_dep(k_sq_newton_fin, sq_blocks(nact * kk), 256, 0, sn, w.sq_O2, w.sq_fns, nact, logn, cx, co1, k, w.sq_alpha);
    }
    dump_alpha_off = fns[0].aoff;
    dump_alpha_t = fns[0].t;
    for (int g0 = 0; g0 < Fr;) {  // root products: the functions with the same product length n >= 2 t together
      const int logn = ceil_log2(2 * fns[g0].t);
      int g1 = g0;
      while (g1 < Fr && ceil_log2(2 * fns[g1].t) == logn) ++g1;
      const int64_t n = (int64_t)1 << logn, ng = g1 - g0, EX = 2 * ng * n;
      launch_dep(k_sq_root_prep, sq_blocks(EX), 256, 0, sn, top, w.sq_fns + g0, ng, w.sq_alpha, logn, k, w.sq_X);
      ntt_mul_pairs(w.sq_X, EX, w.sq_O2, logn, cx, sn);
      launch_dep(k_sq_root_fin, sq_blocks(ng * n), 256, 0, sn, w.sq_O2, w.sq_fns + g0, ng, logn, cx, co2, k, cur + (size_t)B * T);
      g0 = g1;
    }
  }
  // (down) level by level for the vector rows [va, vb), in chunks of Vc; returns with the rows in `cur`'s final buffer
  auto down = [&](int va, int vb, uint64_t* c, uint64_t* n2) {
    const int Vr = vb - va;
    for (int l = r.nlev - 1; l >= 0; --l) {
      const int logn = ceil_log2((int64_t)2 * ZP_SQ_LEAF << l);
      const int64_t n = (int64_t)1 << logn, P = (int64_t)(copy0[l] - pair0[l]);
      const SqTask* tp = w.sq_tasks + pair0[l];
      if (P) {
        const int64_t EX = 2 * P * n;
        const uint64_t* Xl = w.sq_Xl + 3 * xoff[l];  // the transforms of the reversed children, from the up-tree
        for (int v0 = va; v0 < vb; v0 += w.sq.Vc) {
          const int nv = (vb - v0 < w.sq.Vc) ? vb - v0 : w.sq.Vc;
          const int64_t EY = (int64_t)nv * P * n, EO = 2 * EY;
          launch_dep(k_sq_down_prepy, sq_blocks(EY), 256, 0, st, c + (size_t)v0 * T, T, tp, P, logn, w.sq_Y, EY, ntt_down_copies(logn));
          ntt_mul_down(w.sq_Y, EY, Xl, EX, w.sq_O, logn, P, cx, st);
          launch_dep(k_sq_down_fin, sq_blocks(EO), 256, 0, st, c + (size_t)v0 * T, T, tp, P, logn, w.sq_O, EO, cx, co1, k,
                                                                      n2 + (size_t)v0 * T);
        }
      }
      const int nc = (int)(copy1[l] - copy0[l]);
      if (nc) {
        const int ny = nc * Vr;
        launch_dep(k_sq_copy, dim3(64, (unsigned)(ny < 1024 ? ny : 1024)), 256, 0, st, w.sq_tasks + copy0[l], nc, c + (size_t)va * T,
                                                                                             n2 + (size_t)va * T, Vr, T);
      }
      uint64_t* tmp = c;
      c = n2;
      n2 = tmp;
    }
    return c;
  };
  SQ_DUMP(3, cur, (size_t)B * T);        // (the root tails of the values, before their buffer is reused)
  uint64_t* fin = down(0, B, cur, nxt);  // the value vectors, beside the Newton chain
  if (aux) {                             // join: the M' tail is complete
    cudaEventRecord(aux->ev_join, sn);
    cudaStreamWaitEvent(st, aux->ev_join, 0);
  }
  SQ_DUMP(2, w.sq_alpha + dump_alpha_off, dump_alpha_t);
#ifdef ZP_TEST_HOOKS
  if (g_sq_dump_stage == 3 && g_sq_dump_out)  // (and the root tail of M')
    cudaMemcpyAsync(g_sq_dump_out + (size_t)B * T, cur + (size_t)B * T, 8 * (size_t)T, cudaMemcpyDeviceToDevice, st);
#endif
  (void)dump_alpha_off, (void)dump_alpha_t;
  down(B, V, cur, nxt);  // the M' vector
  if (fin != cur) {
    nxt = cur;
    cur = fin;
  }
  SQ_DUMP(4, cur, (size_t)V * T);
  // (leaf) the synthetic-division dots of (a3) on the leaves as functions, B + 1 right-hand sides, unscaled
  {
    dim3 gt((unsigned)((ZP_SQ_LEAF + 255) / 256), grid_y(nleaves));
    ++g_launches, k_solve_table<<<gt, 256, 0, st>>>(lev(0), w.sq_leafoffs, nleaves, k, w.tab, w.R);
    ++g_launches, k_fill_u64<<<sq_blocks(T), 256, 0, st>>>(w.scale, T, k.c224);  // scale = 1: plain numerators out
    const int passes = (V + ZP_NB_MAX - 1) / ZP_NB_MAX;
    const int per = (V + passes - 1) / passes;
    dim3 g((unsigned)((ZP_SQ_LEAF + ZP_K3_THREADS - 1) / ZP_K3_THREADS), grid_y(nleaves));
    ProfScope prof_leaf(ZP_K_LEAF_SOLVE, st);
    for (int b0 = 0; b0 < V; b0 += per) {
      const int nb = (V - b0 < per) ? (V - b0) : per;
      dispatch_node_solve(nb, g, st, nodes, w.tab, w.sq_leafoffs, nleaves, cur, T, b0, 0, k, w.scale, nxt, nullptr);
    }
  }
  SQ_DUMP(5, nxt, (size_t)V * T);
  // c = N(m_i) / M'(m_i) [/ m_i]: one batched inversion
  // (all pointers shifted to the batch's slot 0: d_offs holds absolute slots)
  ++g_launches, k_inv_finish<true><<<inv_blocks(T), 128, 0, st>>>(nxt + (size_t)B * T - r.a0, nodes - r.a0, s0, r.a0, T, d_offs, Fr, k,
                                                                   nxt - r.a0, T, B, coefs - r.a0, ldc, w.st_solve + r.f0);
}

// (a2)-(a4) by the quadratic route of PAPER.md section 2.2 for the functions [0, F) behind w.d_offsets
// (the functions cover the slots [a0, a0 + n) of the batch)
void run_solve_quadratic(const Ws& w, const uint64_t* nodes, int F, int64_t a0, int64_t n, int64_t T_tot, int64_t tmax,
                         const uint64_t* vals, int B, int s0, const ZpMod& k, uint64_t* coefs, cudaStream_t st) {
  const uint64_t* Mt = run_master_poly(w, nodes, F, tmax, k, st);
  if (B == 1 && tmax >= ZP_EVAL2_MIN_T) {
    // one right-hand side, long skeleton: num_i = W(m_i) with W = correlation of v and M (kernels.cuh, k_corr_w)
    uint64_t* Wt = (Mt == w.M0) ? w.M1 : w.M0;  // the tree's other buffer is free now
    ProfScope prof(ZP_K_NODE_SOLVE, st);
    dim3 gc((unsigned)((tmax + ZP_K2_TC - 1) / ZP_K2_TC), grid_y(F));
    ++g_launches, k_corr_w<<<gc, ZP_K2_TC, 0, st>>>(vals, Mt, w.d_offsets, F, k, Wt);
    dim3 gt((unsigned)((tmax + 255) / 256), grid_y(F));
    ++g_launches, k_solve_table_w<<<gt, 256, 0, st>>>(Wt, Mt, w.d_offsets, F, k, reinterpret_cast<ulonglong2*>(w.tab));
    dim3 ge((unsigned)((tmax + ZP_K3_THREADS - 1) / ZP_K3_THREADS), grid_y(F));
    ++g_launches, k_node_eval2<<<ge, ZP_K3_THREADS, 0, st>>>(nodes, reinterpret_cast<const ulonglong2*>(w.tab), w.d_offsets, F, k, w.R,
                                                               w.scale);
    ++g_launches, k_inv_finish<true><<<inv_blocks(n), 128, 0, st>>>(w.scale, nodes, s0, a0, n, w.d_offsets, F, k, w.R, 0, 1, coefs, 0,
                                                                     w.st_solve);
    return;
  }
  {
    dim3 gt((unsigned)((tmax + 255) / 256), grid_y(F));
    ++g_launches, k_solve_table<<<gt, 256, 0, st>>>(Mt, w.d_offsets, F, k, w.tab, w.R);
  }
  const ulonglong4* M = w.tab;
  const int passes = (B + ZP_NB_MAX - 1) / ZP_NB_MAX;
  const int per = (B + passes - 1) / passes;
  ProfScope prof(ZP_K_NODE_SOLVE, st);
  dim3 g((unsigned)((tmax + ZP_K3_THREADS - 1) / ZP_K3_THREADS), grid_y(F));
  ++g_launches, k_node_den<<<g, ZP_K3_THREADS, 0, st>>>(nodes, w.R, w.d_offsets, F, k, w.scale);
  ++g_launches, k_inv_finish<false><<<inv_blocks(n), 128, 0, st>>>(w.scale, nodes, s0, a0, n, w.d_offsets, F, k, nullptr, 0, 0, w.scale, 0,
                                                                    w.st_solve);
  for (int b0 = 0; b0 < B; b0 += per) {
    const int nb = (B - b0 < per) ? (B - b0) : per;
    dispatch_node_solve(nb, g, st, nodes, M, w.d_offsets, F, vals, T_tot, b0, s0, k, w.scale, coefs, w.st_solve);
  }
}

// (a2)-(a4): solve into coefs; per-function codes into w.st_solve (NONE = ok).  h_offs: the host offsets of the functions
// behind w.d_offsets (absolute slots).  Runs of consecutive long functions take the sub-quadratic route (subq.cuh), the
// others the quadratic one.
void run_solve(const Ws& w, const int64_t* h_offs, const uint64_t* nodes, int F, int64_t T_tot, int64_t tmax,
               const uint64_t* vals, int B, int s0, const ZpMod& k, uint64_t* coefs, cudaStream_t st) {
  ++g_launches, k_fill_i32<<<(F + 255) / 256, 256, 0, st>>>(w.st_solve, F, ZP_ST_NONE);
  std::vector<SqRun> runs;
  if (w.sq.any) sq_find_runs(h_offs, F, w.sq.thr, &runs);
  if (runs.empty()) {
    run_solve_quadratic(w, nodes, F, h_offs[0], h_offs[F] - h_offs[0], T_tot, tmax, vals, B, s0, k, coefs, st);
    return;
  }
  const NttCtx cx = ntt_begin(w, st);
  auto quad = [&](int f0, int f1) {  // the functions [f0, f1) by the quadratic route: same launches on shifted offsets
    if (f1 <= f0) return;
    int64_t tm = 0;
    for (int f = f0; f < f1; ++f) tm = (h_offs[f + 1] - h_offs[f] > tm) ? h_offs[f + 1] - h_offs[f] : tm;
    Ws wc = w;
    wc.d_offsets += f0;
    wc.st_solve += f0;
    run_solve_quadratic(wc, nodes, f1 - f0, h_offs[f0], h_offs[f1] - h_offs[f0], T_tot, tm, vals, B, s0, k, coefs, st);
  };
  int f = 0;
  for (const SqRun& r : runs) {
    quad(f, r.f0);
    sq_solve(w, cx, h_offs, r, nodes + r.a0, vals + r.a0, T_tot, B, s0, k, coefs + r.a0, T_tot, st);
    f = r.f1;
  }
  quad(f, F);
}

// (a5): Newton on [B x n] with leading dimension ld; code into w.st_newton[0]
void run_newton(const Ws& w, const uint64_t* samples, int B, const uint64_t* vals, int64_t n, int64_t ld,
                const ZpMod& k, int basis, uint64_t* out, cudaStream_t st, bool canonical_in) {
  ++g_launches, k_fill_i32<<<1, 32, 0, st>>>(w.st_newton, 1, ZP_ST_NONE);
  ++g_launches, k_newton_prep<<<(B * B + 127) / 128, 128, 0, st>>>(samples, B, k, w.invd, w.smont, w.st_newton);
  ProfScope prof(ZP_K_NEWTON, st);
  const size_t smem = 16 * ((size_t)B * B + B) + 8 * (size_t)B * ZP_K5_THREADS;
  int64_t blocks = (n + ZP_K5_THREADS - 1) / ZP_K5_THREADS;
  if (blocks > sm_count() * 64) blocks = sm_count() * 64;
  if (n >= 4 * (int64_t)B) {
    // many coefficients: L = Newton(identity) once, then the batch is the product L x vals (k_newton_apply)
    ++g_launches, k_set_identity<<<(B * B + 255) / 256, 256, 0, st>>>(w.newtI, B);
    cudaFuncSetAttribute(k_newton<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    ++g_launches, k_newton<true><<<1, ZP_K5_THREADS, smem, st>>>(w.invd, w.smont, B, w.newtI, B, B, k, basis, w.newtL);
    const size_t smem2 = 8 * ((size_t)(B + 3) * B + (size_t)B * ZP_K5_THREADS);
    if (canonical_in) {
      cudaFuncSetAttribute(k_newton_apply<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
      ++g_launches, k_newton_apply<true><<<(unsigned)blocks, ZP_K5_THREADS, smem2, st>>>(w.newtL, B, vals, n, ld, k, basis, out);
    } else {
      cudaFuncSetAttribute(k_newton_apply<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
      ++g_launches, k_newton_apply<false><<<(unsigned)blocks, ZP_K5_THREADS, smem2, st>>>(w.newtL, B, vals, n, ld, k, basis, out);
    }
    return;
  }
  if (canonical_in) {
    cudaFuncSetAttribute(k_newton<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    ++g_launches, k_newton<true><<<(unsigned)blocks, ZP_K5_THREADS, smem, st>>>(w.invd, w.smont, B, vals, n, ld, k, basis, out);
  } else {
    cudaFuncSetAttribute(k_newton<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    ++g_launches, k_newton<false><<<(unsigned)blocks, ZP_K5_THREADS, smem, st>>>(w.invd, w.smont, B, vals, n, ld, k, basis, out);
  }
}

void upload_offsets(const Ws& w, const int64_t* h_offsets, int F, cudaStream_t st) {
  cudaMemcpyAsync(w.d_offsets, h_offsets, sizeof(int64_t) * (size_t)(F + 1), cudaMemcpyHostToDevice, st);
}

void run_eval_nodes(const uint16_t* exps, int64_t T_tot, int nv, const uint64_t* anchors, const ZpMod& k,
                    uint64_t* nodes, cudaStream_t st) {
  ProfScope prof(ZP_K_EVAL_NODES, st);
  int64_t blocks = (T_tot + ZP_K1_THREADS - 1) / ZP_K1_THREADS;
  if (blocks > sm_count() * 16) blocks = sm_count() * 16;
  ++g_launches, k_eval_nodes<<<(unsigned)blocks, ZP_K1_THREADS, 0, st>>>(exps, T_tot, nv, anchors, k, nodes);
}

void run_power_sums(const Ws& w, const uint64_t* nodes, int F, int64_t T_tot, int64_t tmax, const uint64_t* coef,
                    int B, int s0, const ZpMod& k, uint64_t* out, cudaStream_t st) {
  ProfScope prof(ZP_K_POWER_SUMS, st);
  dim3 g((unsigned)((tmax + ZP_K6_SBLOCK - 1) / ZP_K6_SBLOCK), grid_y(F));
  ++g_launches, k_power_sums<<<g, ZP_K6_THREADS, 0, st>>>(nodes, w.d_offsets, F, coef, T_tot, B, s0, k, out);
}

bool ws_ok(const void* ws, size_t have, size_t need) {
  return ws && ((uintptr_t)ws & 255) == 0 && have >= need;
}

// staging of the host-buffer entry: [exps | anchors | samples | vals | out | status | inner workspace]
struct HostWs {
  uint16_t* exps;
  uint64_t *anchors, *samples, *vals, *out;
  int32_t* status;
  void* inner;
  size_t inner_bytes, bytes;
};
HostWs carve_host(void* base, int64_t T_tot, int F, int nv, int B, const SqSizes& sq) {
  HostWs h;
  size_t o = 0;
  auto take = [&](size_t n) {
    char* p = base ? (char*)base + o : nullptr;
    o += al(n);
    return (void*)p;
  };
  h.exps = (uint16_t*)take(2 * (size_t)T_tot * nv);
  h.anchors = (uint64_t*)take(8 * (size_t)nv);
  h.samples = (uint64_t*)take(8 * (size_t)B);
  h.vals = (uint64_t*)take(8 * (size_t)T_tot * B);
  h.out = (uint64_t*)take(8 * (size_t)T_tot * B);
  h.status = (int32_t*)take(4 * (size_t)F);
  h.inner_bytes = carve(nullptr, T_tot, F, B, 0, sq).bytes;
  h.inner = take(h.inner_bytes);
  h.bytes = o;
  return h;
}

// (a1)-(a5) on the functions [f0, f1) of a batch whose arrays are resident in full (row stride T_tot): the
// kernels index by absolute term offsets, so a chunk is the same launch sequence on shifted offset/status
// pointers.  The whole batch is the chunk [0, F).
// Small batches take one fused launch (small.cuh): at most ZP_SMALL_MAXF functions of at most ZP_SMALL_MAXT terms, and
// little enough work per lane (pipe cycles of the chain, the B dot products and Newton's B^2 / 2 steps) that one lane
// per node beats the launch and dependency latency of the general path (about 100 us for its thirteen launches).
inline int small_groups(int B) {  // lanes per node: one per ZP_SMALL_NB right-hand sides, at most ZP_SMALL_MAXG
  const int g = (B + ZP_SMALL_NB - 1) / ZP_SMALL_NB;
  return g > ZP_SMALL_MAXG ? ZP_SMALL_MAXG : g;
}
bool small_ok(const int64_t* h_offs, int F, int B) {
  if (F > ZP_SMALL_MAXF || B > ZP_SMALL_MAXB) return false;
  int64_t tmax = 0;
  for (int f = 0; f < F; ++f) tmax = (h_offs[f + 1] - h_offs[f] > tmax) ? h_offs[f + 1] - h_offs[f] : tmax;
  if (tmax > ZP_SMALL_MAXT) return false;
  const int G = small_groups(B), per = (B + G - 1) / G;
  const int64_t cost = tmax * (18 * (int64_t)per + 108 * ((per + ZP_SMALL_NB - 1) / ZP_SMALL_NB)) + 80 * (int64_t)B * B;
  return cost <= 50000;
}
void lift_small(const int64_t* h_offs, int F, int64_t T_tot, int nv, const uint16_t* exps, const uint64_t* anchors,
                const uint64_t* samples, int B, int s0, const uint64_t* vals, const ZpMod& k, int basis, uint64_t* out,
                uint64_t* nodes_out, int32_t* status, cudaStream_t st) {
  ProfScope prof(ZP_K_NODE_SOLVE, st);
  SmallOffs so;
  for (int f = 0; f <= F; ++f) so.o[f] = h_offs[f];  // absolute slots, by value: no upload
  const size_t smem = 2 * 8 * (size_t)B * ZP_SMALL_MAXT;  // the columns of Newton's recurrence and the function's values
  cudaFuncSetAttribute(k_lift_small, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 8 * ZP_MAX_B * ZP_SMALL_MAXT);
  const int G = small_groups(B);
  // (programmatic stream serialization: in a loop of small lifts the next launch becomes resident while this one drains)
  launch_dep(k_lift_small, dim3((unsigned)F), dim3(ZP_SMALL_MAXT * (G + 1)), smem, st, exps, so, nv, anchors, samples, B, G, s0, vals,
             T_tot, k, basis, out, nodes_out, status);
}

void lift_chunk(const Ws& w, const int64_t* h_offsets, int f0, int f1, int64_t T_tot, int nv, const uint16_t* exps,
                const uint64_t* anchors, const uint64_t* samples, int B, int s0, const uint64_t* vals, const ZpMod& k,
                int basis, uint64_t* out, uint64_t* nodes, int32_t* status, cudaStream_t st) {
  const int64_t a = h_offsets[f0], n = h_offsets[f1] - a;
  int64_t tmax = 0;
  for (int f = f0; f < f1; ++f) tmax = (h_offsets[f + 1] - h_offsets[f] > tmax) ? h_offsets[f + 1] - h_offsets[f] : tmax;
  Ws wc = w;
  wc.d_offsets += f0;
  wc.st_solve += f0;
  wc.st_pre += f0;
  const int Fc = f1 - f0;
  run_eval_nodes(exps + a * nv, n, nv, anchors, k, nodes + a, st);
  run_solve(wc, h_offsets + f0, nodes, Fc, T_tot, tmax, vals, B, s0, k, out, st);
  run_newton(wc, samples, B, out + a, n, T_tot, k, basis, out + a, st, true);
  ++g_launches, k_status_finish<<<(Fc + 255) / 256, 256, 0, st>>>(nullptr, wc.st_solve, wc.st_newton, Fc, status + f0);
}

// copy streams and events of the host-buffer entry (created once per device, kept for the process)
#define ZP_PIPE_MAX_CHUNKS 24
struct Pipe {
  bool ready = false;
  cudaStream_t s_in = nullptr, s_out = nullptr;
  cudaEvent_t ev_start = nullptr, ev_end = nullptr, ev_in[ZP_PIPE_MAX_CHUNKS], ev_done[ZP_PIPE_MAX_CHUNKS];
};
Pipe g_pipe[16];
Pipe* get_pipe() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 16) return nullptr;
  Pipe& P = g_pipe[dev];
  if (!P.ready) {
    bool ok = cudaStreamCreateWithFlags(&P.s_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&P.s_out, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&P.ev_start, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&P.ev_end, cudaEventDisableTiming) == cudaSuccess;
    for (int c = 0; ok && c < ZP_PIPE_MAX_CHUNKS; ++c)
      ok = cudaEventCreateWithFlags(&P.ev_in[c], cudaEventDisableTiming) == cudaSuccess &&
           cudaEventCreateWithFlags(&P.ev_done[c], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) return nullptr;
    P.ready = true;
  }
  return &P;
}

}  // namespace

extern "C" {

const char* zippel_strerror(int code) {
  switch (code) {
    case ZP_OK: return "ok";
    case ZP_ERR_ARG: return "bad argument";
    case ZP_ERR_WORKSPACE: return "workspace too small or misaligned";
    case ZP_ERR_CUDA: return "CUDA error";
    case ZP_ERR_SCRATCH_LIMIT: return "batch exceeds the static scratch array (ZP_STATIC_SCRATCH_BYTES = 1 MiB: offsets + scan descriptors)";
    case ZP_ST_DUPLICATE_NODE: return "duplicate (or zero) node";
    case ZP_ST_DUPLICATE_SAMPLE: return "duplicate sample";
    case ZP_ST_ZERO_PIVOT: return "zero pivot in balancing";
    case ZP_ST_THIELE_DEGENERATE: return "degenerate inverse difference in Thiele reconstruction";
    case ZP_ST_NO_RATIONAL: return "no rational number within the bounds";
    default: return "unknown";
  }
}

size_t zippel_workspace_bytes(const int64_t* h_offsets, int F, int B, int flags) {
  int64_t T_tot, tmax;
  if (!check_offsets(h_offsets, F, &T_tot, &tmax) || B <= 0 || B > ZP_MAX_B) return 0;
  return carve(nullptr, T_tot, F, B, flags, sq_sizes(h_offsets, F, B)).bytes;
}

int zippel_eval_nodes(const uint16_t* exps, int64_t T_tot, int nv, const uint64_t* anchors, uint64_t p,
                      uint64_t* nodes, void* stream) {
  ZpMod k;
  if (!exps || !anchors || !nodes || T_tot <= 0 || T_tot >= ((int64_t)1 << 31) || nv <= 0 || nv > ZP_MAX_NV ||
      !make_mod(p, &k))
    return ZP_ERR_ARG;
  run_eval_nodes(exps, T_tot, nv, anchors, k, nodes, (cudaStream_t)stream);
  return cuda_ok();
}

int vandermonde_solve_batch(const uint64_t* nodes, const int64_t* h_offsets, int F, const uint64_t* vals, int B,
                            int s0, uint64_t p, uint64_t* coefs, int32_t* status, void* workspace,
                            size_t workspace_bytes, void* stream) {
  ZpMod k;
  int64_t T_tot, tmax;
  if (!nodes || !vals || !coefs || !status || B <= 0 || B > ZP_MAX_B || (s0 != 0 && s0 != 1) || !make_mod(p, &k) ||
      !check_offsets(h_offsets, F, &T_tot, &tmax))
    return ZP_ERR_ARG;
  const SqSizes sq = sq_sizes(h_offsets, F, B);
  if (!ws_ok(workspace, workspace_bytes, carve(nullptr, T_tot, F, B, 0, sq).bytes)) return ZP_ERR_WORKSPACE;
  const Ws w = carve(workspace, T_tot, F, B, 0, sq);
  cudaStream_t st = (cudaStream_t)stream;
  upload_offsets(w, h_offsets, F, st);
  run_solve(w, h_offsets, nodes, F, T_tot, tmax, vals, B, s0, k, coefs, st);
  ++g_launches, k_status_finish<<<(F + 255) / 256, 256, 0, st>>>(nullptr, w.st_solve, nullptr, F, status);
  return cuda_ok();
}

int newton_interp_batch(const uint64_t* samples, int B, const uint64_t* vals, int64_t n, int64_t ld, uint64_t p,
                        int basis, uint64_t* out, int32_t* status, void* workspace, size_t workspace_bytes,
                        void* stream) {
  ZpMod k;
  if (!samples || !vals || !out || !status || B <= 0 || B > ZP_MAX_B || n <= 0 || ld < n || (basis != 0 && basis != 1) ||
      !make_mod(p, &k))
    return ZP_ERR_ARG;
  if (!ws_ok(workspace, workspace_bytes, carve(nullptr, 1, 1, B, 0).bytes)) return ZP_ERR_WORKSPACE;
  const Ws w = carve(workspace, 1, 1, B, 0);
  cudaStream_t st = (cudaStream_t)stream;
  run_newton(w, samples, B, vals, n, ld, k, basis, out, st, false);
  ++g_launches, k_status_finish<<<1, 32, 0, st>>>(nullptr, nullptr, w.st_newton, 1, status);
  return cuda_ok();
}

int zippel_lift_step(const uint16_t* exps, const int64_t* h_offsets, int F, int nv, const uint64_t* anchors,
                     const uint64_t* samples, int B, int s0, const uint64_t* vals, uint64_t p, int basis,
                     uint64_t* out, uint64_t* nodes_out, int32_t* status, void* workspace, size_t workspace_bytes,
                     void* stream) {
  ZpMod k;
  int64_t T_tot, tmax;
  if (!exps || !anchors || !samples || !vals || !out || !status || nv <= 0 || nv > ZP_MAX_NV || B <= 0 ||
      B > ZP_MAX_B || (s0 != 0 && s0 != 1) || (basis != 0 && basis != 1) || !make_mod(p, &k) ||
      !check_offsets(h_offsets, F, &T_tot, &tmax))
    return ZP_ERR_ARG;
  const SqSizes sq = sq_sizes(h_offsets, F, B);
  if (!ws_ok(workspace, workspace_bytes, carve(nullptr, T_tot, F, B, 0, sq).bytes)) return ZP_ERR_WORKSPACE;
  const Ws w = carve(workspace, T_tot, F, B, 0, sq);
  cudaStream_t st = (cudaStream_t)stream;
  if (small_ok(h_offsets, F, B)) {
    lift_small(h_offsets, F, T_tot, nv, exps, anchors, samples, B, s0, vals, k, basis, out, nodes_out, status, st);
    return cuda_ok();
  }
  upload_offsets(w, h_offsets, F, st);
  lift_chunk(w, h_offsets, 0, F, T_tot, nv, exps, anchors, samples, B, s0, vals, k, basis, out,
             nodes_out ? nodes_out : w.nodes, status, st);
  return cuda_ok();
}

size_t zippel_host_workspace_bytes(const int64_t* h_offsets, int F, int nv, int B) {
  int64_t T_tot, tmax;
  if (!check_offsets(h_offsets, F, &T_tot, &tmax) || B <= 0 || B > ZP_MAX_B || nv <= 0 || nv > ZP_MAX_NV) return 0;
  return carve_host(nullptr, T_tot, F, nv, B, sq_sizes(h_offsets, F, B)).bytes;
}

int zippel_lift_step_host(const uint16_t* h_exps, const int64_t* h_offsets, int F, int nv,
                          const uint64_t* h_anchors, const uint64_t* h_samples, int B, int s0,
                          const uint64_t* h_vals, uint64_t p, int basis, uint64_t* h_out, int32_t* h_status,
                          void* workspace, size_t workspace_bytes, void* stream) {
  ZpMod k;
  int64_t T_tot, tmax;
  if (!h_exps || !h_anchors || !h_samples || !h_vals || !h_out || !h_status || nv <= 0 || nv > ZP_MAX_NV ||
      B <= 0 || B > ZP_MAX_B || (s0 != 0 && s0 != 1) || (basis != 0 && basis != 1) || !make_mod(p, &k) ||
      !check_offsets(h_offsets, F, &T_tot, &tmax))
    return ZP_ERR_ARG;
  const SqSizes sq = sq_sizes(h_offsets, F, B);
  if (!ws_ok(workspace, workspace_bytes, carve_host(nullptr, T_tot, F, nv, B, sq).bytes)) return ZP_ERR_WORKSPACE;
  const HostWs h = carve_host(workspace, T_tot, F, nv, B, sq);
  const Ws w = carve(h.inner, T_tot, F, B, 0, sq);
  cudaStream_t st = (cudaStream_t)stream;
  Pipe* P = get_pipe();
  if (!P) return ZP_ERR_CUDA;
  // chunks of whole functions; small batches go in one piece.  The first and the last chunks are small because the
  // first H2D copy and the last D2H copy cannot overlap with anything; the sizes grow and shrink by about 4x, so that
  // the input of chunk c + 1 has arrived (55 GB/s: the whole input of C2 takes 13 ms) when the kernels of chunk c end
  // and the output of chunk c is out when the kernels of chunk c + 1 end.  A chunk costs about 0.65 ms of its own
  // (partial waves of the large kernels, some fifty dependent launches of the route), so fewer is better.  Measured on C2
  // (device-resident 43.9 ms): 7 chunks {2,5,13,24,13,5,2}/64 49.4 ms, 6 chunks {2,8,22,22,8,2}/64 48.7, 5 chunks 48.5.
  static const int kCut64[] = {0, 3, 16, 48, 61, 64};
  const size_t bytes = 8 * (size_t)T_tot * B;
  int nch = 1;
  int cut[ZP_PIPE_MAX_CHUNKS + 1];
  cut[0] = 0;
  if (bytes >= ((size_t)8 << 20) && F >= 64) {
    nch = (int)(sizeof(kCut64) / sizeof(kCut64[0])) - 1;
    for (int c = 1, f = 0; c <= nch; ++c) {
      const int64_t target = T_tot / 64 * kCut64[c];
      while (f < F && h_offsets[f] < target) ++f;
      cut[c] = (c == nch) ? F : f;
    }
  } else {
    cut[1] = F;
  }
  cudaMemcpyAsync(h.anchors, h_anchors, 8 * (size_t)nv, cudaMemcpyHostToDevice, st);
  cudaMemcpyAsync(h.samples, h_samples, 8 * (size_t)B, cudaMemcpyHostToDevice, st);
  upload_offsets(w, h_offsets, F, st);
  cudaEventRecord(P->ev_start, st);  // the copy streams start after everything already queued on `stream`
  cudaStreamWaitEvent(P->s_in, P->ev_start, 0);
  cudaStreamWaitEvent(P->s_out, P->ev_start, 0);
  const size_t pitch = 8 * (size_t)T_tot;
  for (int c = 0; c < nch; ++c) {  // H2D of chunk c+1 and D2H of chunk c-1 overlap the kernels of chunk c
    const int f0 = cut[c], f1 = cut[c + 1];
    if (f1 <= f0) continue;
    const int64_t a = h_offsets[f0], n = h_offsets[f1] - a;
    cudaMemcpyAsync(h.exps + a * nv, h_exps + a * nv, 2 * (size_t)n * nv, cudaMemcpyHostToDevice, P->s_in);
    cudaMemcpy2DAsync(h.vals + a, pitch, h_vals + a, pitch, 8 * (size_t)n, (size_t)B, cudaMemcpyHostToDevice, P->s_in);
    cudaEventRecord(P->ev_in[c], P->s_in);
    cudaStreamWaitEvent(st, P->ev_in[c], 0);
    if (nch == 1 && small_ok(h_offsets, F, B))
      lift_small(h_offsets, F, T_tot, nv, h.exps, h.anchors, h.samples, B, s0, h.vals, k, basis, h.out, nullptr, h.status, st);
    else
      lift_chunk(w, h_offsets, f0, f1, T_tot, nv, h.exps, h.anchors, h.samples, B, s0, h.vals, k, basis, h.out, w.nodes,
                 h.status, st);
    cudaEventRecord(P->ev_done[c], st);
    cudaStreamWaitEvent(P->s_out, P->ev_done[c], 0);
    cudaMemcpy2DAsync(h_out + a, pitch, h.out + a, pitch, 8 * (size_t)n, (size_t)B, cudaMemcpyDeviceToHost, P->s_out);
    cudaMemcpyAsync(h_status + f0, h.status + f0, 4 * (size_t)(f1 - f0), cudaMemcpyDeviceToHost, P->s_out);
  }
  cudaEventRecord(P->ev_end, P->s_out);
  cudaStreamWaitEvent(st, P->ev_end, 0);  // a synchronize on `stream` covers the result copies
  return cuda_ok();
}

int zippel_power_sums(const uint64_t* nodes, const int64_t* h_offsets, int F, const uint64_t* coef, int B, int s0,
                      uint64_t p, uint64_t* out, void* workspace, size_t workspace_bytes, void* stream) {
  ZpMod k;
  int64_t T_tot, tmax;
  if (!nodes || !coef || !out || B <= 0 || B > ZP_MAX_B || (s0 != 0 && s0 != 1) || !make_mod(p, &k) ||
      !check_offsets(h_offsets, F, &T_tot, &tmax))
    return ZP_ERR_ARG;
  if (!ws_ok(workspace, workspace_bytes, carve(nullptr, T_tot, F, B, 0).bytes)) return ZP_ERR_WORKSPACE;
  const Ws w = carve(workspace, T_tot, F, B, 0);
  cudaStream_t st = (cudaStream_t)stream;
  upload_offsets(w, h_offsets, F, st);
  run_power_sums(w, nodes, F, T_tot, tmax, coef, B, s0, k, out, st);
  return cuda_ok();
}

int balanced_zippel_lift_step(const zp_part* num, const zp_part* den, int F, int nv, const uint64_t* anchors,
                              const uint64_t* samples, int B, int s0, uint64_t p, int basis, int32_t* status,
                              void* workspace, size_t workspace_bytes, void* stream) {
  ZpMod k;
  if (!num || !den || !anchors || !samples || !status || nv <= 0 || nv > ZP_MAX_NV || B <= 0 || B > ZP_MAX_B ||
      (s0 != 0 && s0 != 1) || (basis != 0 && basis != 1) || !make_mod(p, &k))
    return ZP_ERR_ARG;
  const zp_part* parts[2] = {num, den};
  int64_t T_tot[2], tmax[2];
  for (int x = 0; x < 2; ++x) {
    const zp_part* q = parts[x];
    if (!q->exps || !q->skel || !q->uvals || !q->out || !check_offsets(q->h_offsets, F, &T_tot[x], &tmax[x]))
      return ZP_ERR_ARG;
    if (!ws_ok(workspace, workspace_bytes, carve(nullptr, T_tot[x], F, B, ZP_WS_BALANCED, sq_sizes(q->h_offsets, F, B)).bytes))
      return ZP_ERR_WORKSPACE;
  }
  cudaStream_t st = (cudaStream_t)stream;
  for (int x = 0; x < 2; ++x) {  // the two parts run back to back on the stream and reuse the workspace
    const zp_part* q = parts[x];
    const Ws w = carve(workspace, T_tot[x], F, B, ZP_WS_BALANCED, sq_sizes(q->h_offsets, F, B));
    upload_offsets(w, q->h_offsets, F, st);
    ++g_launches, k_fill_i32<<<(F + 255) / 256, 256, 0, st>>>(w.st_pre, F, ZP_ST_NONE);
    run_eval_nodes(q->exps, T_tot[x], nv, anchors, k, w.nodes, st);
    run_power_sums(w, w.nodes, F, T_tot[x], tmax[x], q->skel, 1, s0, k, w.R, st);
    {
      ProfScope prof(ZP_K_BALANCE, st);
      const int64_t cb = (T_tot[x] + 256 * ZP_BAL_N - 1) / (256 * ZP_BAL_N);
      ulonglong2* sc = reinterpret_cast<ulonglong2*>(w.tab);  // free until the solve builds its table
      ++g_launches, k_balance_scale<<<(unsigned)(cb > sm_count() * 8 ? sm_count() * 8 : cb), 256, 0, st>>>(
                        q->uvals, w.R, w.d_offsets, F, T_tot[x], k, sc, w.st_pre);
      const dim3 g((unsigned)cb, (unsigned)((B + ZP_BAL_ROWS - 1) / ZP_BAL_ROWS));  // T_tot < 2^31: cb < 2^21
      ++g_launches, k_balance_apply<<<g, 256, 0, st>>>(q->uvals, sc, T_tot[x], B, k, w.V);
    }
    run_solve(w, q->h_offsets, w.nodes, F, T_tot[x], tmax[x], w.V, B, s0, k, q->out, st);
    run_newton(w, samples, B, q->out, T_tot[x], T_tot[x], k, basis, q->out, st, true);
    ++g_launches, k_status_finish<<<(F + 255) / 256, 256, 0, st>>>(w.st_pre, w.st_solve, w.st_newton, F, status + (size_t)x * F);
  }
  return cuda_ok();
}

int thiele_reconstruct_batch(const uint64_t* points, int T, const uint64_t* vals, int64_t n, int64_t ld, uint64_t p,
                             uint64_t* num, uint64_t* den, int32_t* degs, uint64_t* cf, int32_t* status,
                             void* workspace, size_t workspace_bytes, void* stream) {
  ZpMod k;
  if (!points || !vals || !num || !den || !degs || !status || T <= 0 || T > ZP_MAX_B || n <= 0 || ld < n ||
      !make_mod(p, &k))
    return ZP_ERR_ARG;
  if (!ws_ok(workspace, workspace_bytes, carve(nullptr, 1, 1, T, 0).bytes)) return ZP_ERR_WORKSPACE;
  const Ws w = carve(workspace, 1, 1, T, 0);
  cudaStream_t st = (cudaStream_t)stream;
  ulonglong2* xd = w.invd;   // [T*T] {x_j - x_k, companion}
  ulonglong2* xm = w.smont;  // [T]   {x_j, companion}
  ++g_launches, k_fill_i32<<<1, 32, 0, st>>>(w.st_newton, 1, ZP_ST_NONE);
  ++g_launches, k_thiele_prep<<<(T * T + 127) / 128, 128, 0, st>>>(points, T, k, xd, xm, w.st_newton);
  const size_t smem = 8 * 2 * (size_t)(T + 2) * ZP_K8_THREADS;  // two columns per lane
  cudaFuncSetAttribute(k_thiele, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  int64_t blocks = (n + ZP_K8_THREADS - 1) / ZP_K8_THREADS;
  if (blocks > sm_count() * 64) blocks = sm_count() * 64;
  ++g_launches, k_thiele<<<(unsigned)blocks, ZP_K8_THREADS, smem, st>>>(xd, xm, w.st_newton, T, vals, n, ld, k, num, den,
                                                                         degs, cf, status);
  return cuda_ok();
}

int zippel_extend_skeleton(const uint16_t* exps, const int64_t* h_offsets, int F, int nv, const uint64_t* coefs, int B,
                           uint64_t p, uint16_t* new_exps, uint64_t* new_coefs, int64_t cap, int64_t* new_offsets,
                           int32_t* degs, void* workspace, size_t workspace_bytes, void* stream) {
  ZpMod k;
  int64_t T_tot, tmax;
  if (!exps || !coefs || !new_exps || !new_coefs || !new_offsets || !degs || nv <= 0 || nv >= ZP_MAX_NV || B <= 0 ||
      B > ZP_MAX_B || cap < 0 || !make_mod(p, &k) || !check_offsets(h_offsets, F, &T_tot, &tmax))
    return ZP_ERR_ARG;
  if (!ws_ok(workspace, workspace_bytes, carve(nullptr, T_tot, F, B, 0).bytes)) return ZP_ERR_WORKSPACE;
  const Ws w = carve(workspace, T_tot, F, B, 0);
  cudaStream_t st = (cudaStream_t)stream;
  upload_offsets(w, h_offsets, F, st);
  const int64_t nb = (T_tot + ZP_K9_BLOCK - 1) / ZP_K9_BLOCK;
  unsigned long long* desc = reinterpret_cast<unsigned long long*>(w.tab);  // [nb + 1] (the slice holds 32 T_tot bytes)
  ++g_launches, k_fill_i32<<<(F + 255) / 256, 256, 0, st>>>(degs, F, -1);
  cudaMemsetAsync(desc, 0, 8 * (size_t)(nb + 1), st);
  // staging buffer: room for one row per term and a quarter more, within 64 KB (else the blocks write directly)
  int stage_rows = ZP_K9_BLOCK + ZP_K9_BLOCK / 4;
  size_t smem = (size_t)stage_rows * (8 + 2 * (size_t)(nv + 1)) + 2 * (size_t)nv * ZP_K9_BLOCK + 32;
  if (smem > 98304) stage_rows = 0, smem = 0;
  cudaFuncSetAttribute(k_ext_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, 98304);
  ++g_launches, k_ext_fused<<<(unsigned)nb, ZP_K9_THREADS, smem, st>>>(exps, nv, coefs, T_tot, B, w.d_offsets, F, k, desc, nb, new_exps,
                                                                        new_coefs, cap, new_offsets, degs, stage_rows);
  return cuda_ok();
}

// ---- the entry point that allocates nothing (zippel.h: zippel_extend_skeleton_static) ---------------------------------
// The scratch of k_ext_fused -- [offsets (F + 1) int64, rounded to 256 bytes | descriptors (nb + 1) x 8 bytes] -- in a
// file-scope device array.  In host code the NAME g_static_scratch is a host-side stand-in, not a device address: the
// kernels get the address that cudaGetSymbolAddress returns for the CURRENT device, looked up once per device.
static __device__ __align__(256) unsigned char g_static_scratch[ZP_STATIC_SCRATCH_BYTES];
static unsigned char* g_static_scratch_ptr[64] = {nullptr};  // per device ordinal
static std::mutex g_static_scratch_mu;
static unsigned char* static_scratch() {  // device address on the current device, or nullptr
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  std::lock_guard<std::mutex> lock(g_static_scratch_mu);
  if (!g_static_scratch_ptr[dev]) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess || !ptr) {
      cudaGetLastError();  // (clear it: the caller gets ZP_ERR_CUDA)
      return nullptr;
    }
    g_static_scratch_ptr[dev] = static_cast<unsigned char*>(ptr);
  }
  return g_static_scratch_ptr[dev];
}
size_t zippel_static_scratch_bytes(void) { return ZP_STATIC_SCRATCH_BYTES; }

int zippel_extend_skeleton_static(const uint16_t* exps, const int64_t* h_offsets, int F, int nv, const uint64_t* coefs,
                                  int B, uint64_t p, uint16_t* new_exps, uint64_t* new_coefs, int64_t cap,
                                  int64_t* new_offsets, int32_t* degs, void* stream) {
  ZpMod k;
  int64_t T_tot, tmax;
  if (!exps || !coefs || !new_exps || !new_coefs || !new_offsets || !degs || nv <= 0 || nv >= ZP_MAX_NV || B <= 0 ||
      B > ZP_MAX_B || cap < 0 || !make_mod(p, &k) || !check_offsets(h_offsets, F, &T_tot, &tmax))
    return ZP_ERR_ARG;
  const int64_t nb = (T_tot + ZP_K9_BLOCK - 1) / ZP_K9_BLOCK;
  const size_t offs_bytes = al(sizeof(int64_t) * (size_t)(F + 1)), desc_bytes = 8 * (size_t)(nb + 1);
  if (offs_bytes + desc_bytes > ZP_STATIC_SCRATCH_BYTES) return ZP_ERR_SCRATCH_LIMIT;
  unsigned char* base = static_scratch();
  if (!base) return ZP_ERR_CUDA;
  int64_t* d_offsets = reinterpret_cast<int64_t*>(base);
  unsigned long long* desc = reinterpret_cast<unsigned long long*>(base + offs_bytes);
  cudaStream_t st = (cudaStream_t)stream;
  cudaMemcpyAsync(d_offsets, h_offsets, sizeof(int64_t) * (size_t)(F + 1), cudaMemcpyHostToDevice, st);
  ++g_launches, k_fill_i32<<<(F + 255) / 256, 256, 0, st>>>(degs, F, -1);
  cudaMemsetAsync(desc, 0, desc_bytes, st);  // the array keeps the last call's tickets and flags: they start at zero
  int stage_rows = ZP_K9_BLOCK + ZP_K9_BLOCK / 4;  // (as zippel_extend_skeleton)
  size_t smem = (size_t)stage_rows * (8 + 2 * (size_t)(nv + 1)) + 2 * (size_t)nv * ZP_K9_BLOCK + 32;
  if (smem > 98304) stage_rows = 0, smem = 0;
  cudaFuncSetAttribute(k_ext_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, 98304);
  ++g_launches, k_ext_fused<<<(unsigned)nb, ZP_K9_THREADS, smem, st>>>(exps, nv, coefs, T_tot, B, d_offsets, F, k, desc, nb, new_exps,
                                                                        new_coefs, cap, new_offsets, degs, stage_rows);
  return cuda_ok();
}

int crt_rational_reconstruct_batch(const uint64_t* r1, const uint64_t* r2, int64_t n, uint64_t p1, uint64_t p2,
                                   int64_t* num, int64_t* den, int32_t* status, void* stream) {
  ZpMod k1, k2;
  if (!r1 || !r2 || !num || !den || !status || n <= 0 || p1 == p2 || !make_mod(p1, &k1) || !make_mod(p2, &k2))
    return ZP_ERR_ARG;
  const u128 m = (u128)p1 * p2;
  u128 N = 0;  // floor(sqrt((m - 1) / 2))
  for (int b = 63; b >= 0; --b) {
    const u128 cnd = N | ((u128)1 << b);
    if (cnd * cnd <= (m - 1) / 2) N = cnd;
  }
  uint64_t inv = 1, base = p1 % p2, e = p2 - 2;  // p1^-1 mod p2 (Fermat; p2 prime is the caller's contract)
  while (e) {
    if (e & 1) inv = (uint64_t)((u128)inv * base % p2);
    base = (uint64_t)((u128)base * base % p2);
    e >>= 1;
  }
  int64_t blocks = (n + 255) / 256;
  if (blocks > sm_count() * 32) blocks = sm_count() * 32;
  ++g_launches, k_crt_rational<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(
      r1, r2, n, p1, k2, inv, (uint64_t)(m >> 64), (uint64_t)m, (uint64_t)N, num, den, status);
  return cuda_ok();
}

unsigned long long zippel_launch_count(void) { return g_launches; }

int zippel_profile_events(int kernel, void* ev_start, void* ev_stop) {
  if (kernel < 0 || (kernel & 0xff) > 8 || (kernel != 0 && (!ev_start || !ev_stop))) return ZP_ERR_ARG;
  g_prof_ordinal = (kernel >> 8) - 1;  // bits 8.. : 0 = every occurrence, n = only the n-th (1-based) after this call
  g_prof_seen = 0;
  kernel &= 0xff;
  g_prof_kernel = kernel;
  g_prof_start = kernel ? (cudaEvent_t)ev_start : nullptr;
  g_prof_stop = kernel ? (cudaEvent_t)ev_stop : nullptr;
  return ZP_OK;
}

int zippel_shutdown(void) {
  for (int dev = 0; dev < 16; ++dev) {
    Pipe& P = g_pipe[dev];
    if (!P.ready) continue;
    cudaSetDevice(dev);
    cudaStreamDestroy(P.s_in);
    cudaStreamDestroy(P.s_out);
    cudaEventDestroy(P.ev_start);
    cudaEventDestroy(P.ev_end);
    for (int c = 0; c < ZP_PIPE_MAX_CHUNKS; ++c) {
      cudaEventDestroy(P.ev_in[c]);
      cudaEventDestroy(P.ev_done[c]);
    }
    P = Pipe();
  }
  for (int dev = 0; dev < 16; ++dev) {
    SqAux& A = g_sqaux[dev];
    if (!A.ready) continue;
    cudaSetDevice(dev);
    cudaStreamDestroy(A.s2);
    cudaEventDestroy(A.ev_fork);
    cudaEventDestroy(A.ev_join);
    A = SqAux();
  }
  return cuda_ok();
}

int zippel_set_tuning(int key, int64_t value) {
  if (key == ZP_TUNE_SUBQ_MIN_T && value >= 0) {  // 0: back to the built-in rule
    g_subq_min_t = value;
    return ZP_OK;
  }
  return ZP_ERR_ARG;
}

#ifdef ZP_TEST_HOOKS
#include "test_hooks.cuh"
#endif

}  // extern "C"
