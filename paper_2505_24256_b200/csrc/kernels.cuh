// kernels.cuh -- device kernels of the Zippel lifting step.
// Notation follows the paper: t terms, nodes m_i, master polynomial M, right-hand sides v_{b,s},
// B = D+1 samples c_j of x_k.  "~" marks Montgomery form (modarith.cuh).
#pragma once
#include "modarith.cuh"

#define ZP_ST_DUPLICATE_NODE 16
#define ZP_ST_DUPLICATE_SAMPLE 17
#define ZP_ST_ZERO_PIVOT 18
#define ZP_ST_NONE 0x7fffffff

// ------------------------------------------------------------------------------------------------
// (a1) K1 eval_nodes: one lane per term.  m_i = prod_j y_j^{e_ij}  (eq. (3)).
// The CTA first builds Y[j][k] = (y_j^(2^k))~ for k < 16 in shared memory (powers
// from precomputed powers); each lane then multiplies the table entries its exponent bits select.
// HBM-bound: 2*nv bytes in, 8 (or 16) bytes out per term.
// ------------------------------------------------------------------------------------------------
#define ZP_K1_THREADS 256
__global__ void __launch_bounds__(ZP_K1_THREADS)
k_eval_nodes(const uint16_t* __restrict__ exps, int64_t T_tot, int nv, const uint64_t* __restrict__ anchors,
             ZpMod k, uint64_t* __restrict__ nodes) {
  __shared__ uint64_t Y[32 * 16];
  if (threadIdx.x < nv) {
    uint64_t y = to_mont(zp_canon(anchors[threadIdx.x], k.p), k);
    for (int b = 0; b < 16; ++b) {
      Y[threadIdx.x * 16 + b] = y;
      y = mont_mul(y, y, k);
    }
  }
  __syncthreads();
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < T_tot; i += (int64_t)gridDim.x * blockDim.x) {
    const uint16_t* e = exps + i * nv;
    uint64_t m = k.r1;
    for (int j = 0; j < nv; ++j) {
      uint32_t ej = e[j];
      for (int b = 0; ej; ++b, ej >>= 1)
        if (ej & 1) m = mont_mul(m, Y[j * 16 + b], k);
    }
    nodes[i] = from_mont(m, k);
  }
}

// ------------------------------------------------------------------------------------------------
// (a2) K2 master polynomial M(z) = prod_i (z - m_i), as a product tree.
// A monic polynomial of degree n is stored WITHOUT its leading 1, as n Montgomery coefficients, in
// the slots of the nodes it covers: the block of nodes [lo, hi) of a function owns buf[off+lo .. off+hi).
// Merging the monic A (degree a) and B (degree b):  C' = A' * B' + z^a B' + z^b A'   (a + b slots).
// Convolutions are deferred sums, one reduction per output coefficient.
//
// k_tree_leaf: one CTA builds the product of up to LEAF consecutive nodes of one function in shared
// memory (all levels up to LEAF).  k_tree_level: one merge level in global memory for blocks > LEAF.
// ------------------------------------------------------------------------------------------------
#define ZP_LEAF 1024
#define ZP_K2_THREADS 256

// conv + shifts for output slot c of the merged block (A' = src[0..a), B' = src[a..a+b))
template <typename SrcPtr>
ZP_DEV uint64_t tree_merge_coef(SrcPtr src, int a, int b, int c, const ZpMod& k) {
  // sum_{j} A'_j B'_{c-j},  max(0, c-b+1) <= j <= min(a-1, c)
  const int jlo = c - b + 1 > 0 ? c - b + 1 : 0;
  const int jhi = c < a - 1 ? c : a - 1;
  uint64_t r = 0;
  if (jhi >= jlo) {
    Acc acc;
    acc_zero(acc);
    for (int j = jlo; j <= jhi; ++j) acc_mac(acc, src[j], src[a + c - j]);
    r = mont_mul(acc_redc160(acc, k), k.c160, k);
  }
  if (c >= a) r = mod_add(r, src[a + (c - a)], k.p);  // z^a B'
  if (c >= b) r = mod_add(r, src[c - b], k.p);        // z^b A'
  return r;
}

__global__ void __launch_bounds__(ZP_K2_THREADS)
k_tree_leaf(const uint64_t* __restrict__ nodes, const int64_t* __restrict__ offsets, int F, ZpMod k,
            uint64_t* __restrict__ out) {
  __shared__ uint64_t buf[2][ZP_LEAF];
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int64_t t = offsets[f + 1] - off;
    const int64_t lo = (int64_t)blockIdx.x * ZP_LEAF;
    if (lo >= t) continue;  // uniform per CTA
    const int n = (int)((t - lo < ZP_LEAF) ? (t - lo) : ZP_LEAF);
    for (int i = threadIdx.x; i < n; i += blockDim.x)
      buf[0][i] = mod_neg(to_mont(zp_canon(nodes[off + lo + i], k.p), k), k.p);  // (z - m_i)' = -m_i~
    __syncthreads();
    int cur = 0;
    for (int a = 1; a < n; a <<= 1) {  // merge blocks [2j a, 2j a + a) and [2j a + a, 2j a + 2a)
      const uint64_t* src = buf[cur];
      uint64_t* dst = buf[cur ^ 1];
      for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const int base = i & ~(2 * a - 1);
        const int b = (n - base - a) < a ? (n - base - a) : a;  // right block length (may be <= 0)
        dst[i] = (b <= 0) ? src[i] : tree_merge_coef(src + base, a, b, i - base, k);
      }
      __syncthreads();
      cur ^= 1;
    }
    for (int i = threadIdx.x; i < n; i += blockDim.x) out[off + lo + i] = buf[cur][i];
    __syncthreads();
  }
}

// one level: left block length a (a multiple of LEAF, so a tile of TC output slots never straddles two
// merges).  CTA = TC consecutive output slots of one function, one per lane; the convolution runs over
// j-tiles of TJ coefficients of A' (broadcast reads) against a window of TC + TJ - 1 coefficients of B'
// (unit-stride reads), both staged in shared memory and zero-padded outside their ranges, so the inner
// loop is branch-free deferred MACs.
#define ZP_K2_TC 256
#define ZP_K2_TJ 256
__global__ void __launch_bounds__(ZP_K2_TC)
k_tree_level(const uint64_t* __restrict__ src, const int64_t* __restrict__ offsets, int F, int64_t a, ZpMod k,
             uint64_t* __restrict__ dst) {
  __shared__ uint64_t sA[ZP_K2_TJ];
  __shared__ uint64_t sB[ZP_K2_TC + ZP_K2_TJ];
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int64_t t = offsets[f + 1] - off;
    for (int64_t i0 = (int64_t)blockIdx.x * ZP_K2_TC; i0 < t; i0 += (int64_t)gridDim.x * ZP_K2_TC) {
      const int64_t base = i0 - (i0 % (2 * a));
      const int64_t b = (t - base - a) < a ? (t - base - a) : a;  // right block length (<= 0: nothing to merge)
      const int64_t i = i0 + threadIdx.x;
      if (b <= 0) {  // uniform per CTA
        if (i < t) dst[off + i] = src[off + i];
        continue;
      }
      const uint64_t* A = src + off + base;      // A'[0 .. a)
      const uint64_t* Bp = src + off + base + a;  // B'[0 .. b)
      const int64_t c0 = i0 - base, c = c0 + threadIdx.x;
      const int64_t jlo = c0 - b + 1 > 0 ? c0 - b + 1 : 0;
      const int64_t jhi = c0 + ZP_K2_TC - 1 < a - 1 ? c0 + ZP_K2_TC - 1 : a - 1;
      Acc acc;
      acc_zero(acc);
      for (int64_t j0 = jlo; j0 <= jhi; j0 += ZP_K2_TJ) {
        __syncthreads();
        if (threadIdx.x < ZP_K2_TJ) sA[threadIdx.x] = (j0 + threadIdx.x < a) ? A[j0 + threadIdx.x] : 0;
        for (int x = threadIdx.x; x < ZP_K2_TC + ZP_K2_TJ - 1; x += ZP_K2_TC) {
          const int64_t kb = c0 - j0 - (ZP_K2_TJ - 1) + x;  // B' index of window slot x
          sB[x] = (kb >= 0 && kb < b) ? Bp[kb] : 0;
        }
        __syncthreads();
        const uint64_t* win = sB + threadIdx.x + (ZP_K2_TJ - 1);  // win[-jj] = B'[c - (j0 + jj)]
#pragma unroll 8
        for (int jj = 0; jj < ZP_K2_TJ; jj += 2) acc_mac2(acc, sA[jj], win[-jj], sA[jj + 1], win[-jj - 1]);
      }
      if (i < t) {
        uint64_t r = mont_mul(acc_redc160(acc, k), k.c160, k);
        if (c >= a) r = mod_add(r, Bp[c - a], k.p);  // z^a B'
        if (c >= b) r = mod_add(r, A[c - b], k.p);   // z^b A'
        dst[off + i] = r;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// (a3) prologue k_solve_table: the 32-byte record the hot loop broadcasts for the Horner step from stage l
// to stage l-1 (q_{l-1} = M_l + m q_l), stored at slot l-1, l = 1 .. t:
//     { M_l, M_l', D_l, D_l' },  D_l = l M_l (coefficient of z^(l-1) in M'(z)),  M_t = 1,
// w' = floor(w 2^64 / p) the Shoup companion (modarith.cuh).  Input: the product tree's M~ (Montgomery,
// coefficients 0 .. t-1).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_solve_table(const uint64_t* __restrict__ Mt, const int64_t* __restrict__ offsets, int F, ZpMod k,
              ulonglong4* __restrict__ tab, uint64_t* __restrict__ Dplain) {
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int64_t t = offsets[f + 1] - off;
    for (int64_t l = 1 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; l <= t; l += (int64_t)gridDim.x * blockDim.x) {
      const uint64_t Mm = (l < t) ? Mt[off + l] : k.r1;
      const uint64_t Dm = mont_mul(Mm, to_mont((uint64_t)zp_canon(l, k.p), k), k);  // (l M_l)~
      ulonglong4 r;
      r.x = from_mont(Mm, k);
      r.y = shoup_companion(Mm, k);
      r.z = from_mont(Dm, k);
      r.w = shoup_companion(Dm, k);
      tab[off + l - 1] = r;
      Dplain[off + l - 1] = r.z;  // coefficient of z^(l-1) in M': the table of k_node_den
    }
  }
}

// ------------------------------------------------------------------------------------------------
// (a3)+(a4) K3 node_solve: the hot loop (PAPER.md L189-197 ZippelMultiplePrime(), L203-213).
// One lane per node i of one function; the CTA streams tiles of the table above and of the NB right-hand
// sides through shared memory (every lane needs the same M_l, v_{b,l}: warp-uniform broadcast reads).
// Per lane, stages l = t-1 .. 0 with q = q_l (q_{t-1} = 1):
//     acc_b += q_l * v_{b,l}              NB deferred MACs (L194-195 "vector of powers" x "values", L205-209)
//     q_{l-1} = M_l + m q_l   (l >= 1)    one Horner step (L193: synthetic division)
// then  c_{b,i} = acc_b * scale_i,  scale_i = 1 / (M'(m_i) [m_i if s0 = 1])  (L196) from k_node_den below:
// M'(m_i) = Q_i(m_i) = prod_{j != i}(m_i - m_j) (G15) is the paper's "polynomial value computed via Horner's
// method"; it is a polynomial evaluation and is cheaper by blocked deferred MACs in its own launch than as a
// second Horner chain in this loop (which is what the first measured profiles of round 1 show).
// Stages are taken in pairs (2j+1, 2j), j = J-1 .. 0, J = t/2 + 1, starting from q = 0 at a stage >= t
// (records beyond t and values v_{b,l}, l >= t, are zero; record t carries M_t = 1): the two MACs of a
// pair go into the accumulator together (acc_mac2).
// All values are plain residues; q stays lazy in [0, 2p) (horner_step); nothing of length t is stored per
// lane (reading G7).  Template NB = right-hand sides handled per pass.
// ------------------------------------------------------------------------------------------------
#define ZP_K3_THREADS 128
#define ZP_K3_PAIRS 32
// Orientation of the 16-byte value record per template instance.  Both orders put the two limbs of one operand
// into registers of the same parity; which of the two ptxas's register allocation serves with fewer bank
// conflicts differs from instance to instance, so it is read off the SASS (share of accumulating IMAD.WIDE whose
// multiplicands have equal parity; profiles/r02_k3_orient.md) and tabulated per instance: bit NB = 1 -> odd stage first.
#ifdef ZP_K3_FORCE_ORIENT
#define ZP_K3_ORIENT(NB) (ZP_K3_FORCE_ORIENT)
#else
#define ZP_K3_ORIENT_MASK 0x1810740u
#define ZP_K3_ORIENT(NB) ((ZP_K3_ORIENT_MASK >> (NB)) & 1u)
#endif

// cp.async (LDGSTS) with zero fill: src-size 0 reads nothing and writes zeros
ZP_DEV void cp_async8(void* smem, const void* g, bool ok) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(g),
               "r"(ok ? 8 : 0) : "memory");
}
ZP_DEV void cp_async4(void* smem, const void* g, bool ok) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(g),
               "r"(ok ? 4 : 0) : "memory");
}
ZP_DEV void cp_async16(void* smem, const void* g, bool ok) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(g),
               "r"(ok ? 16 : 0) : "memory");
}
ZP_DEV void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
ZP_DEV void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int NB>
__global__ void __launch_bounds__(ZP_K3_THREADS)
k_node_solve(const uint64_t* __restrict__ nodes, const ulonglong4* __restrict__ tab, const int64_t* __restrict__ offsets,
             int F, const uint64_t* __restrict__ vals, int64_t T_tot, int b0, int s0, ZpMod k,
             const uint64_t* __restrict__ scale, uint64_t* __restrict__ coefs, int32_t* __restrict__ status) {
  // two buffers: the tile after the current one is in flight (cp.async) while the current one is consumed
  __shared__ __align__(16) ulonglong4 sT[2][2 * ZP_K3_PAIRS];      // record of stage l = 2 j0 + x
  __shared__ __align__(16) ulonglong2 sV[2][ZP_K3_PAIRS * NB];     // [pair][b]: 16-byte record of limbs, see issue_tile
  constexpr int ORIENT = ZP_K3_ORIENT(NB);
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int t = (int)(offsets[f + 1] - off);
    const int i0 = blockIdx.x * ZP_K3_THREADS;
    if (i0 >= t) continue;  // uniform per CTA
    const int i = i0 + threadIdx.x;
    const bool live = i < t;
    const uint64_t m = live ? zp_canon(nodes[off + i], k.p) : 0;
    const uint64_t mp = shoup_companion(to_mont(m, k), k);
    uint64_t q = 0;
    Acc acc[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) acc_zero(acc[b]);
    const ulonglong4* Tf = tab + off;
    const int J = t / 2 + 1;
    // tile = pairs [j0, j1), j0 = max(j1 - PAIRS, 0); out-of-range stages are zero-filled (src-size 0)
    auto issue_tile = [&](int j1, int buf) {
      const int j0 = j1 - ZP_K3_PAIRS > 0 ? j1 - ZP_K3_PAIRS : 0;
      const int np = j1 - j0;
      for (int x = threadIdx.x; x < 4 * np; x += ZP_K3_THREADS) {  // 16-byte halves of the 32-byte records
        const int l = 2 * j0 + (x >> 1);
        const bool ok = l >= 1 && l <= t;
        cp_async16(reinterpret_cast<ulonglong2*>(&sT[buf][0]) + x,
                   reinterpret_cast<const ulonglong2*>(Tf + (ok ? l - 1 : 0)) + (x & 1), ok);
      }
      for (int x = threadIdx.x; x < 2 * ZP_K3_PAIRS * NB; x += ZP_K3_THREADS) {
        const int b = x / (2 * ZP_K3_PAIRS), r = x % (2 * ZP_K3_PAIRS);  // r = stage offset inside the tile (shifts)
        if (r >= 2 * np) continue;  // only the lowest tile can be short
        const int l = 2 * j0 + r;
        const bool ok = l < t;
        // 16-byte record of (pair, b): ORIENT = 1: { v_odd.lo, v_even.lo, v_odd.hi, v_even.hi }, 0: even first
        // (the odd stage pairs with qa)
        uint32_t* rec = reinterpret_cast<uint32_t*>(&sV[buf][0]) + ((r >> 1) * NB + b) * 4 + ((r & 1) ^ ORIENT);
        const uint32_t* src = reinterpret_cast<const uint32_t*>(vals + (int64_t)(b0 + b) * T_tot + off + (ok ? l : 0));
        cp_async4(rec, src, ok);
        cp_async4(rec + 2, src + 1, ok);
      }
      cp_async_commit();
    };
    __syncthreads();  // the previous function's last tile has been consumed
    issue_tile(J, 0);
    int buf = 0;
    for (int j1 = J; j1 > 0; j1 -= ZP_K3_PAIRS, buf ^= 1) {  // tile covers pairs [j0, j1)
      const int j0 = j1 - ZP_K3_PAIRS > 0 ? j1 - ZP_K3_PAIRS : 0;
      const int np = j1 - j0;
      if (j0 > 0) {
        issue_tile(j0, buf ^ 1);
        cp_async_wait<1>();
      } else {
        cp_async_wait<0>();
      }
      __syncthreads();
      const ulonglong4* cT = sT[buf];
      const ulonglong2* cV = sV[buf];
      for (int jj = np - 1; jj >= 0; --jj) {
        const ulonglong4 r1 = cT[2 * jj + 1];
        const uint64_t qa = q;
        const uint64_t qb = horner_step(qa, m, mp, r1.x, r1.y, k);
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          const uint4 w = reinterpret_cast<const uint4*>(cV)[jj * NB + b];
          if (ORIENT)
            acc_mac2_limbs(acc[b], (uint32_t)qa, (uint32_t)(qa >> 32), w.x, w.z, (uint32_t)qb, (uint32_t)(qb >> 32), w.y, w.w);
          else
            acc_mac2_limbs(acc[b], (uint32_t)qa, (uint32_t)(qa >> 32), w.y, w.w, (uint32_t)qb, (uint32_t)(qb >> 32), w.x, w.z);
        }
        if (j0 + jj > 0) {
          const ulonglong4 r0 = cT[2 * jj];
          q = horner_step(qb, m, mp, r0.x, r0.y, k);
        }
      }
      __syncthreads();  // this buffer is refilled by the next iteration's prefetch
    }
    if (live) {
      const uint64_t sc = scale[off + i];  // plain d^-1 * 2^224: acc_redc160 (x 2^-160) and mont_mul (x 2^-64) undo it
#pragma unroll
      for (int b = 0; b < NB; ++b)
        coefs[(int64_t)(b0 + b) * T_tot + off + i] = mont_mul(acc_redc160(acc[b], k), sc, k);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// (a4) batched inversion (Montgomery's trick: "scalar-multiplied by the modular inverse
// of the polynomial value").  A warp inverts 32 N values with ONE modular inversion: every lane multiplies its N values
// up (prefix products in registers), the 32 lane products are scanned from both ends with shuffles (10 products per
// lane), all lanes invert the warp's total together (the same argument in every lane: the binary algorithm of
// modarith.cuh, mont_inv_uniform), and each lane unwinds its own prefix products: about 3 N + 14 products per lane for N
// inverses against 125 per value for a Fermat power each.  x[] Montgomery, in place -> inverses; zeros are skipped
// (left 0) and reported through the returned mask.  Every lane of the warp must call it (full-mask shuffles).
// ------------------------------------------------------------------------------------------------
ZP_DEV uint64_t shfl_up64(uint64_t v, int o) {
  return ((uint64_t)__shfl_up_sync(0xffffffffu, (uint32_t)(v >> 32), o) << 32) | __shfl_up_sync(0xffffffffu, (uint32_t)v, o);
}
ZP_DEV uint64_t shfl_down64(uint64_t v, int o) {
  return ((uint64_t)__shfl_down_sync(0xffffffffu, (uint32_t)(v >> 32), o) << 32) | __shfl_down_sync(0xffffffffu, (uint32_t)v, o);
}
ZP_DEV uint64_t shfl_idx64(uint64_t v, int l) {
  return ((uint64_t)__shfl_sync(0xffffffffu, (uint32_t)(v >> 32), l) << 32) | __shfl_sync(0xffffffffu, (uint32_t)v, l);
}
template <int N>
ZP_DEV uint32_t warp_batch_inv(uint64_t (&x)[N], const ZpMod& k) {
  uint64_t pre[N];
  uint64_t run = k.r1;
  uint32_t zero = 0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    pre[i] = run;
    if (x[i] == 0) zero |= 1u << i;
    else run = mont_mul(run, x[i], k);
  }
  const int lane = threadIdx.x & 31;
  uint64_t below = run, above = run;  // products over the lanes <= this one / >= this one
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint64_t a = mont_mul(below, shfl_up64(below, o), k), b = mont_mul(above, shfl_down64(above, o), k);
    below = (lane >= o) ? a : below;
    above = (lane + o < 32) ? b : above;
  }
  const uint64_t tinv = mont_inv_uniform(shfl_idx64(below, 31), k);  // 1 / (product of the whole warp): uniform
  const uint64_t lo = shfl_up64(below, 1), hi = shfl_down64(above, 1);
  uint64_t inv = tinv;  // 1 / run = tinv * (lanes below) * (lanes above)
  if (lane > 0) inv = mont_mul(inv, lo, k);
  if (lane < 31) inv = mont_mul(inv, hi, k);
#pragma unroll
  for (int i = N - 1; i >= 0; --i) {
    if (zero >> i & 1) continue;
    const uint64_t xi = x[i];
    x[i] = mont_mul(inv, pre[i], k);
    inv = mont_mul(inv, xi, k);
  }
  return zero;
}

// The same over a whole CTA (blockDim.x a multiple of 32, sh = 64 words of shared memory): the warps' totals meet in
// shared memory and warp 0 runs the one inversion for all of them -- the inversion is ~3000 instructions, as many as a
// warp spends on streaming ~60 products, so it pays to share it wider where the CTA can wait for it.  Two barriers;
// every lane of the CTA must call.
template <int N>
ZP_DEV uint32_t cta_batch_inv(uint64_t (&x)[N], const ZpMod& k, uint64_t* sh) {
  uint64_t pre[N];
  uint64_t run = k.r1;
  uint32_t zero = 0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    pre[i] = run;
    if (x[i] == 0) zero |= 1u << i;
    else run = mont_mul(run, x[i], k);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint64_t below = run, above = run;  // products over the lanes <= this one / >= this one
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint64_t a = mont_mul(below, shfl_up64(below, o), k), b = mont_mul(above, shfl_down64(above, o), k);
    below = (lane >= o) ? a : below;
    above = (lane + o < 32) ? b : above;
  }
  if (lane == 31) sh[warp] = below;  // the warp's total
  __syncthreads();
  if (warp == 0) {
    uint64_t tb = lane < nw ? sh[lane] : k.r1, ta = tb;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint64_t a = mont_mul(tb, shfl_up64(tb, o), k), b = mont_mul(ta, shfl_down64(ta, o), k);
      tb = (lane >= o) ? a : tb;
      ta = (lane + o < 32) ? b : ta;
    }
    uint64_t winv = mont_inv_uniform(shfl_idx64(tb, 31), k);  // 1 / (product of the whole CTA)
    const uint64_t lo = shfl_up64(tb, 1), hi = shfl_down64(ta, 1);
    if (lane > 0) winv = mont_mul(winv, lo, k);
    if (lane < 31) winv = mont_mul(winv, hi, k);
    if (lane < nw) sh[32 + lane] = winv;  // 1 / (total of warp `lane`)
  }
  __syncthreads();
  uint64_t inv = sh[32 + warp];
  const uint64_t lo = shfl_up64(below, 1), hi = shfl_down64(above, 1);
  if (lane > 0) inv = mont_mul(inv, lo, k);
  if (lane < 31) inv = mont_mul(inv, hi, k);
#pragma unroll
  for (int i = N - 1; i >= 0; --i) {
    if (zero >> i & 1) continue;
    const uint64_t xi = x[i];
    x[i] = mont_mul(inv, pre[i], k);
    inv = mont_mul(inv, xi, k);
  }
  return zero;
}

// The division that ends every solve: for the slots i of the functions behind `offs` (all pointers at the batch's slot
// 0, the functions cover the slots [a0, a0 + T)),  d_i = den_i [m_i if s0 = 1]  (den plain) and
//   APPLY = false:  scale_i = 2^224 / d_i  (plain; the factor k_node_solve multiplies its reduced sums by), in place or not
//   APPLY = true :  out_{b,i} = num_{b,i} / d_i,  b < B  (num plain, rows of ldn; out rows of ldo)
// d_i = 0 (duplicate node, or a zero node with s0 = 1: readings G24/G25) -> ZP_ST_DUPLICATE_NODE with the term index.
// A warp owns 32 N consecutive slots (lane + 32 j: unit-stride rows).
#define ZP_INV_N 8
template <bool APPLY>
__global__ void __launch_bounds__(128)
k_inv_finish(const uint64_t* den, const uint64_t* __restrict__ nodes, int s0, int64_t a0, int64_t T,
             const int64_t* __restrict__ offs, int F, ZpMod kp, const uint64_t* num, int64_t ldn, int B, uint64_t* out,
             int64_t ldo, int32_t* __restrict__ status) {
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t i0 = a0 + warp * (32 * ZP_INV_N) + (threadIdx.x & 31), iend = a0 + T;
  if (i0 - (threadIdx.x & 31) >= iend) return;  // uniform per warp
  uint64_t d[ZP_INV_N];
#pragma unroll
  for (int x = 0; x < ZP_INV_N; ++x) {
    const int64_t i = i0 + 32 * x;
    uint64_t v = kp.r1;
    if (i < iend) {
      v = to_mont(den[i], kp);
      if (s0) v = mont_mul(v, to_mont(zp_canon(nodes[i], kp.p), kp), kp);
    }
    d[x] = v;
  }
  const uint32_t zero = warp_batch_inv<ZP_INV_N>(d, kp);
#pragma unroll
  for (int x = 0; x < ZP_INV_N; ++x) {
    const int64_t i = i0 + 32 * x;
    if (i >= iend) continue;
    if (zero >> x & 1) {
      int lo = 0, hi = F;  // function of slot i: offs[lo] <= i < offs[lo + 1]
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (offs[mid] <= i) lo = mid; else hi = mid;
      }
      atomicMin(&status[lo], (int32_t)(((uint32_t)(i - offs[lo]) << 8) | ZP_ST_DUPLICATE_NODE));
    }
    if (!APPLY) out[i] = mont_mul(d[x], kp.c224, kp);
  }
  if (APPLY)
    for (int b = 0; b < B; ++b) {  // row by row, the warp's eight loads of a row in flight together (num may be out)
      uint64_t v[ZP_INV_N];
#pragma unroll
      for (int x = 0; x < ZP_INV_N; ++x) v[x] = (i0 + 32 * x < iend) ? __ldcs(num + (int64_t)b * ldn + i0 + 32 * x) : 0;
#pragma unroll
      for (int x = 0; x < ZP_INV_N; ++x)
        if (i0 + 32 * x < iend) out[(int64_t)b * ldo + i0 + 32 * x] = mont_mul(v[x], d[x], kp);  // plain x Montgomery
    }
}

// ------------------------------------------------------------------------------------------------
// (a3) for ONE right-hand side and a long skeleton (C5): with q_{i,l} = sum_{k>l} M_k m_i^(k-l-1),
//     num_i = sum_l q_{i,l} v_l = sum_j W_j m_i^j = W(m_i),    W_j = sum_l v_l M_{l+j+1}   (M_t = 1),
// so the per-node work is the evaluation of two fixed polynomials (W and M') at m_i, which needs no modular product
// per coefficient: 2 deferred MACs = 16 units per (node, stage) instead of 2 x 16 + 8, for t^2/2 extra MACs once
// per function (k_corr_w, a tiled correlation like k_tree_level).  Pays only for B = 1 (the quotient q_{i,l} of the
// general path is needed coefficient by coefficient, one modular multiply-add each).
//   k_corr_w         W~_j (Montgomery) from the plain values v and the tree's M~
//   k_solve_table_w  records { W_j, D_{j+1} } (plain), j = 0 .. t-1
//   k_node_eval2     one lane per node: W(m_i) and M'(m_i) by blocked deferred evaluation; k_inv_finish<true> divides
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(ZP_K2_TC)
k_corr_w(const uint64_t* __restrict__ vals, const uint64_t* __restrict__ Mt, const int64_t* __restrict__ offsets, int F,
         ZpMod k, uint64_t* __restrict__ Wt) {
  __shared__ uint64_t sA[ZP_K2_TJ];
  __shared__ uint64_t sB[ZP_K2_TC + ZP_K2_TJ];
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int64_t t = offsets[f + 1] - off;
    const uint64_t* v = vals + off;
    const uint64_t* M = Mt + off;
    for (int64_t j0 = (int64_t)blockIdx.x * ZP_K2_TC; j0 < t; j0 += (int64_t)gridDim.x * ZP_K2_TC) {
      const int64_t j = j0 + threadIdx.x;
      Acc acc;
      acc_zero(acc);
      for (int64_t l0 = 0; l0 + j0 + 1 <= t - 1; l0 += ZP_K2_TJ) {  // some (l, j) of the tile has l + j + 1 <= t - 1
        __syncthreads();
        if (threadIdx.x < ZP_K2_TJ) sA[threadIdx.x] = (l0 + threadIdx.x < t) ? zp_canon(v[l0 + threadIdx.x], k.p) : 0;
        for (int x = threadIdx.x; x < ZP_K2_TC + ZP_K2_TJ - 1; x += ZP_K2_TC) {
          const int64_t kk = l0 + j0 + 1 + x;  // index into M of window slot x
          sB[x] = (kk <= t - 1) ? M[kk] : 0;
        }
        __syncthreads();
        const uint64_t* win = sB + threadIdx.x;  // win[jj] = M_{(l0 + jj) + j + 1}
#pragma unroll 8
        for (int jj = 0; jj < ZP_K2_TJ; jj += 2) acc_mac2(acc, sA[jj], win[jj], sA[jj + 1], win[jj + 1]);
      }
      if (j < t) {
        const uint64_t r = mont_mul(acc_redc160(acc, k), k.c224, k);  // plain * Montgomery sums -> Montgomery
        Wt[off + j] = mod_add(r, to_mont(zp_canon(v[t - 1 - j], k.p), k), k.p);  // + v_{t-1-j} M_t
      }
    }
  }
}

__global__ void __launch_bounds__(256)
k_solve_table_w(const uint64_t* __restrict__ Wt, const uint64_t* __restrict__ Mt, const int64_t* __restrict__ offsets,
                int F, ZpMod k, ulonglong2* __restrict__ tab) {
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int64_t t = offsets[f + 1] - off;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < t; j += (int64_t)gridDim.x * blockDim.x) {
      const uint64_t Mm = (j + 1 < t) ? Mt[off + j + 1] : k.r1;  // M_{j+1}~, M_t = 1
      // record j = { W_j, D_{j+1} } plain: the coefficients of z^j in W and in M'  (D_l = l M_l)
      tab[off + j] = make_ulonglong2(from_mont(Wt[off + j], k), mont_mul(Mm, (uint64_t)zp_canon(j + 1, k.p), k));
    }
  }
}

// Both polynomials are evaluated at m_i in blocks of 32 coefficients against the lane's own table of powers
// m^0 .. m^31 (registers): a block is 32 deferred MACs per polynomial, one reduction, and one
// step V <- V m^32 + S of the outer Horner rule -- 17.8 pipe cycles per coefficient instead of the 35.5 of a
// modular multiply-add per coefficient.
#define ZP_K3E_BLK 32
#define ZP_K3E_TILE 128
__global__ void __launch_bounds__(ZP_K3_THREADS)
k_node_eval2(const uint64_t* __restrict__ nodes, const ulonglong2* __restrict__ tab, const int64_t* __restrict__ offsets,
             int F, ZpMod k, uint64_t* __restrict__ num, uint64_t* __restrict__ den) {
  __shared__ __align__(16) ulonglong2 sT[2][ZP_K3E_TILE];
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int t = (int)(offsets[f + 1] - off);
    const int i0 = blockIdx.x * ZP_K3_THREADS;
    if (i0 >= t) continue;  // uniform per CTA
    const int i = i0 + threadIdx.x;
    const bool live = i < t;
    const uint64_t m = live ? zp_canon(nodes[off + i], k.p) : 0;
    const uint64_t mm = to_mont(m, k);
    uint64_t pw[ZP_K3E_BLK];  // plain m^e
    pw[0] = 1 % k.p;
#pragma unroll
    for (int e = 1; e < ZP_K3E_BLK; ++e) pw[e] = mont_mul(pw[e - 1], mm, k);  // plain * Montgomery -> plain
    // The outer Horner step rides in the same accumulator: with V' = V 2^-160 and g = m^32 2^160,
    //   V'_new = (S + V' g) 2^-160 = acc_redc160(S + V' g),  no other modular product per block.
    const uint64_t g = mont_mul(mont_mul(pw[ZP_K3E_BLK - 1], mm, k), k.c224, k);  // m^32 * 2^224 * 2^-64
    uint64_t VW = 0, VD = 0;  // V' of the two polynomials
    Acc pW, pD;  // sums of the previous block: their reduction and the outer Horner step run while the MACs of the
    acc_zero(pW);  // current block are issued (two independent instruction streams in one loop body)
    acc_zero(pD);
    const ulonglong2* Tf = tab + off;
    auto issue_tile = [&](int tile, int buf) {  // records j in [128 tile, 128 tile + 128), zero beyond t
      for (int x = threadIdx.x; x < ZP_K3E_TILE; x += ZP_K3_THREADS) {
        const int j = tile * ZP_K3E_TILE + x;
        const bool ok = j < t;
        cp_async16(&sT[buf][x], Tf + (ok ? j : 0), ok);
      }
      cp_async_commit();
    };
    const int ntile = (t + ZP_K3E_TILE - 1) / ZP_K3E_TILE;
    __syncthreads();
    issue_tile(ntile - 1, 0);
    int buf = 0;
    for (int tile = ntile - 1; tile >= 0; --tile, buf ^= 1) {
      if (tile > 0) {
        issue_tile(tile - 1, buf ^ 1);
        cp_async_wait<1>();
      } else {
        cp_async_wait<0>();
      }
      __syncthreads();
#pragma unroll 1
      for (int bl = ZP_K3E_TILE / ZP_K3E_BLK - 1; bl >= 0; --bl) {
        const ulonglong2* rec = &sT[buf][bl * ZP_K3E_BLK];
        Acc aW, aD;
        acc_zero(aW);
        acc_zero(aD);
#pragma unroll
        for (int e = 0; e < ZP_K3E_BLK; e += 2) {
          const ulonglong2 r0 = rec[e], r1 = rec[e + 1];
          acc_mac2(aW, pw[e], r0.x, pw[e + 1], r1.x);
          acc_mac2(aD, pw[e], r0.y, pw[e + 1], r1.y);
        }
        acc_mac(pW, VW, g);  // previous block: V' <- (S + V' g) 2^-160
        acc_mac(pD, VD, g);
        VW = acc_redc160(pW, k);
        VD = acc_redc160(pD, k);
        pW = aW;
        pD = aD;
      }
      __syncthreads();
    }
    acc_mac(pW, VW, g);  // the last block, then back from V' to V = V' 2^160
    acc_mac(pD, VD, g);
    VW = mont_mul(acc_redc160(pW, k), k.c224, k);
    VD = mont_mul(acc_redc160(pD, k), k.c224, k);
    if (live) {  // plain W(m_i) and M'(m_i): k_inv_finish divides
      num[off + i] = VW;
      den[off + i] = VD;
    }
  }
}

// (a4) denominators for the general path: den_i = M'(m_i) by the same blocked deferred evaluation (17.8 pipe cycles
// per coefficient), one launch before k_node_solve, which then runs without its second Horner chain (35.5 cycles
// per stage).  Writes the plain den_i; k_inv_finish<false> turns them into scale_i = den_i^-1 (/ m_i) * 2^224, the factor
// k_node_solve applies.
__global__ void __launch_bounds__(ZP_K3_THREADS)
k_node_den(const uint64_t* __restrict__ nodes, const uint64_t* __restrict__ Dtab, const int64_t* __restrict__ offsets,
           int F, ZpMod k, uint64_t* __restrict__ den) {
  __shared__ __align__(16) uint64_t sT[2][ZP_K3E_TILE];
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int t = (int)(offsets[f + 1] - off);
    const int i0 = blockIdx.x * ZP_K3_THREADS;
    if (i0 >= t) continue;  // uniform per CTA
    const int i = i0 + threadIdx.x;
    const bool live = i < t;
    const uint64_t m = live ? zp_canon(nodes[off + i], k.p) : 0;
    const uint64_t mm = to_mont(m, k);
    uint64_t pw[ZP_K3E_BLK];  // plain m^e
    pw[0] = 1 % k.p;
#pragma unroll
    for (int e = 1; e < ZP_K3E_BLK; ++e) pw[e] = mont_mul(pw[e - 1], mm, k);
    const uint64_t g = mont_mul(mont_mul(pw[ZP_K3E_BLK - 1], mm, k), k.c224, k);  // m^32 2^160, see k_node_eval2
    uint64_t VD = 0;
    Acc pD;
    acc_zero(pD);
    const uint64_t* Tf = Dtab + off;
    auto issue_tile = [&](int tile, int buf) {
      for (int x = threadIdx.x; x < ZP_K3E_TILE; x += ZP_K3_THREADS) {
        const int j = tile * ZP_K3E_TILE + x;
        const bool ok = j < t;
        cp_async8(&sT[buf][x], Tf + (ok ? j : 0), ok);
      }
      cp_async_commit();
    };
    const int ntile = (t + ZP_K3E_TILE - 1) / ZP_K3E_TILE;
    __syncthreads();
    issue_tile(ntile - 1, 0);
    int buf = 0;
    for (int tile = ntile - 1; tile >= 0; --tile, buf ^= 1) {
      if (tile > 0) {
        issue_tile(tile - 1, buf ^ 1);
        cp_async_wait<1>();
      } else {
        cp_async_wait<0>();
      }
      __syncthreads();
#pragma unroll 1
      for (int bl = ZP_K3E_TILE / ZP_K3E_BLK - 1; bl >= 0; --bl) {
        const ulonglong2* rec = reinterpret_cast<const ulonglong2*>(&sT[buf][bl * ZP_K3E_BLK]);
        Acc aD;
        acc_zero(aD);
#pragma unroll
        for (int e = 0; e < ZP_K3E_BLK; e += 2) {
          const ulonglong2 r = rec[e >> 1];  // { D_e, D_{e+1} }
          acc_mac2(aD, pw[e], r.x, pw[e + 1], r.y);
        }
        acc_mac(pD, VD, g);  // previous block: V' <- (S + V' g) 2^-160
        VD = acc_redc160(pD, k);
        pD = aD;
      }
      __syncthreads();
    }
    acc_mac(pD, VD, g);
    VD = mont_mul(acc_redc160(pD, k), k.c224, k);  // plain M'(m_i)
    if (live) den[off + i] = VD;
  }
}

// ------------------------------------------------------------------------------------------------
// (a5) K5 Newton interpolation in x_k, one lane per coefficient (eq. (1)).
// k_newton_prep: invd[j*B + jj] = {w, w'} with w = 1/(c_j - c_jj) for jj < j (plain, with its Shoup companion),
// negc[j] = {-c_j, companion}, duplicate check.
// k_newton: divided differences in shared memory (column per lane), optional monomial expansion.
// ------------------------------------------------------------------------------------------------
__global__ void k_newton_prep(const uint64_t* __restrict__ samples, int B, ZpMod k, ulonglong2* __restrict__ invd,
                              ulonglong2* __restrict__ negc, int32_t* __restrict__ nstatus) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= B * B) return;
  const int j = idx / B, jj = idx % B;
  const uint64_t cj = zp_canon(samples[j], k.p), cjj = zp_canon(samples[jj], k.p);
  if (jj == 0) {  // multiplier -c_j of the monomial expansion, with its Shoup companion
    const uint64_t nc = mod_neg(cj, k.p);
    negc[j] = make_ulonglong2(nc, shoup_companion(to_mont(nc, k), k));
  }
  if (jj < j) {
    const uint64_t diff = mod_sub(cj, cjj, k.p);
    if (diff == 0) atomicMin(nstatus, (int32_t)(((uint32_t)j << 8) | ZP_ST_DUPLICATE_SAMPLE));
    const uint64_t wm = mont_inv(to_mont(diff, k), k);  // (1/(c_j - c_jj))~
    invd[idx] = make_ulonglong2(from_mont(wm, k), shoup_companion(wm, k));
  }
}


#define ZP_K5_THREADS 128
// CANON: the values are known to be canonical (the lifting step feeds the solve's output), skip the reduction
template <bool CANON>
__global__ void __launch_bounds__(ZP_K5_THREADS)
k_newton(const ulonglong2* __restrict__ invd, const ulonglong2* __restrict__ negc, int B, const uint64_t* vals, int64_t n,
         int64_t ld, ZpMod k, int basis, uint64_t* out) {
  extern __shared__ __align__(16) uint64_t sh[];
  ulonglong2* sInv = reinterpret_cast<ulonglong2*>(sh);  // [B*B] {w, w'}
  ulonglong2* sC = sInv + B * B;                         // [B]   {-c_j, companion}
  uint64_t* col = reinterpret_cast<uint64_t*>(sC + B) + threadIdx.x;  // column of this lane: col[j*TH]
  constexpr int TH = ZP_K5_THREADS;
  for (int x = threadIdx.x; x < B * B; x += TH) sInv[x] = invd[x];
  for (int x = threadIdx.x; x < B; x += TH) sC[x] = negc[x];
  __syncthreads();
  const int D = B - 1;
  for (int64_t i = (int64_t)blockIdx.x * TH + threadIdx.x; i < n; i += (int64_t)gridDim.x * TH) {
    for (int j = 0; j < B; ++j) col[j * TH] = CANON ? vals[j * ld + i] : zp_canon(vals[j * ld + i], k.p);
    // a_j <- (a_j - a_{j-1}) / (c_j - c_{j-l}), j = D .. l; four independent steps at a time (all loads of a
    // group precede its stores, so the group's products overlap in the pipe)
    for (int l = 1; l <= D; ++l) {
      int j = D;
      for (; j - 3 >= l; j -= 4) {
        const uint64_t v0 = col[j * TH], v1 = col[(j - 1) * TH], v2 = col[(j - 2) * TH], v3 = col[(j - 3) * TH],
                       v4 = col[(j - 4) * TH];
        const ulonglong2* w = sInv + j * B + (j - l);  // row stride B, same column offset j - l
        col[j * TH] = shoup_mul(v0 + k.p - v1, w[0], k);
        col[(j - 1) * TH] = shoup_mul(v1 + k.p - v2, w[-B - 1], k);
        col[(j - 2) * TH] = shoup_mul(v2 + k.p - v3, w[-2 * B - 2], k);
        col[(j - 3) * TH] = shoup_mul(v3 + k.p - v4, w[-3 * B - 3], k);
      }
      for (; j >= l; --j)
        col[j * TH] = shoup_mul(col[j * TH] + k.p - col[(j - 1) * TH], sInv[j * B + (j - l)], k);
    }
    if (basis == 1) {
      // P <- [a_D]; for j = D-1 .. 0: P <- P (x - c_j) + a_j, in place.  Before step j the polynomial P (degree
      // D-j-1) sits in slots j+1 .. D (P_x in slot j+1+x); the step is slot[s] <- slot[s] - c_j slot[s+1] for
      // s = j .. D-1 ascending (slot s holds a_j for s = j, else the old P_{s-j-1}; slot s+1 is still the old
      // P_{s-j}); slot D stays.  After step 0 slot d holds the coefficient of x^d.
      for (int j = D - 1; j >= 0; --j) {
        const ulonglong2 nc = sC[j];
        int x = j;
        for (; x + 3 < D; x += 4) {
          const uint64_t v0 = col[x * TH], v1 = col[(x + 1) * TH], v2 = col[(x + 2) * TH], v3 = col[(x + 3) * TH],
                         v4 = col[(x + 4) * TH];
          col[x * TH] = mod_add(v0, shoup_mul(v1, nc, k), k.p);
          col[(x + 1) * TH] = mod_add(v1, shoup_mul(v2, nc, k), k.p);
          col[(x + 2) * TH] = mod_add(v2, shoup_mul(v3, nc, k), k.p);
          col[(x + 3) * TH] = mod_add(v3, shoup_mul(v4, nc, k), k.p);
        }
        for (; x < D; ++x) col[x * TH] = mod_add(col[x * TH], shoup_mul(col[(x + 1) * TH], nc, k), k.p);
      }
    }
    for (int j = 0; j < B; ++j) out[j * ld + i] = col[j * TH];
  }
}

// Newton interpolation is linear in the values: out = L c with the B x B matrix L = k_newton(identity), which
// depends on the samples and the basis only (lower triangular for the Newton basis).  For many coefficients the
// batch is therefore a [B x B] x [B x n] product: B^2 (or B^2/2) deferred MACs per coefficient (17.8 pipe cycles
// each) instead of B(B-1) modular multiply-adds (35.5 each).  k_newton_apply: one lane per
// coefficient, its column in shared memory, four output rows at a time against the broadcast rows of L.
__global__ void k_set_identity(uint64_t* __restrict__ I, int B) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < B * B) I[idx] = (idx / B == idx % B) ? 1 : 0;
}

// R output rows of L x column: R deferred dot products sharing every load of the column
template <int R>
ZP_DEV void newton_apply_rows(const uint64_t* r0, int B, int bmax, const uint64_t* col, const ZpMod& k, uint64_t* o,
                              int64_t ld) {
  Acc a[R];
#pragma unroll
  for (int q = 0; q < R; ++q) acc_zero(a[q]);
  for (int b = 0; b < bmax; ++b) {
    const uint64_t x = col[b * ZP_K5_THREADS];
#pragma unroll
    for (int q = 0; q < R; ++q) acc_mac(a[q], x, r0[q * B + b]);
  }
  // plain * plain sums: 2^-160 from the reduction and 2^-64 from the product cancel against 2^224
#pragma unroll
  for (int q = 0; q < R; ++q) o[(int64_t)q * ld] = mont_mul(acc_redc160(a[q], k), k.c224, k);
}

template <bool CANON>
__global__ void __launch_bounds__(ZP_K5_THREADS)
k_newton_apply(const uint64_t* __restrict__ L, int B, const uint64_t* vals, int64_t n, int64_t ld, ZpMod k, int basis,
               uint64_t* out) {
  extern __shared__ __align__(16) uint64_t sh[];
  constexpr int TH = ZP_K5_THREADS;
  uint64_t* sL = sh;                                   // [(B + 3) x B], rows >= B are zero
  uint64_t* col = sh + (size_t)(B + 3) * B + threadIdx.x;  // column of this lane: col[b*TH]
  for (int x = threadIdx.x; x < (B + 3) * B; x += TH) sL[x] = (x < B * B) ? L[x] : 0;
  __syncthreads();
  for (int64_t i = (int64_t)blockIdx.x * TH + threadIdx.x; i < n; i += (int64_t)gridDim.x * TH) {
    for (int b = 0; b < B; ++b) col[b * TH] = CANON ? vals[b * ld + i] : zp_canon(vals[b * ld + i], k.p);
    for (int d0 = 0; d0 < B; d0 += 4) {
      const int rows = B - d0 < 4 ? B - d0 : 4;
      const int bmax = (basis == 0 && d0 + rows < B) ? d0 + rows : B;  // Newton basis: L is lower triangular
      const uint64_t* r0 = sL + (size_t)d0 * B;
      uint64_t* o = out + (int64_t)d0 * ld + i;
      switch (rows) {  // the last group has B mod 4 rows: no products against padding
        case 4: newton_apply_rows<4>(r0, B, bmax, col, k, o, ld); break;
        case 3: newton_apply_rows<3>(r0, B, bmax, col, k, o, ld); break;
        case 2: newton_apply_rows<2>(r0, B, bmax, col, k, o, ld); break;
        default: newton_apply_rows<1>(r0, B, bmax, col, k, o, ld); break;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// status plumbing
// ------------------------------------------------------------------------------------------------
__global__ void k_fill_i32(int32_t* x, int n, int32_t v) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = v;
}
// final[f] = first non-NONE of (pre[f], solve[f], newton[0]) ; NONE -> 0
__global__ void k_status_finish(const int32_t* pre, const int32_t* solve, const int32_t* newton, int F, int32_t* fin) {
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= F) return;
  int32_t s = ZP_ST_NONE;
  if (pre && pre[f] != ZP_ST_NONE) s = pre[f];
  else if (solve && solve[f] != ZP_ST_NONE) s = solve[f];
  else if (newton && newton[0] != ZP_ST_NONE) s = newton[0];
  fin[f] = (s == ZP_ST_NONE) ? 0 : s;
}

// ------------------------------------------------------------------------------------------------
// (a6) K6 power sums R_{b,s} = sum_i a_{b,i} m_i^(s+s0)  ("raise base variable
// values to various powers and substitute them into the polynomial"; strided power tables, A21).
// CTA = (function f, block of 512 consecutive s); node tiles of 64 in shared memory with the strided power
// tables  P_i[x] = a_i m_i^(sb0+s0) m_i^x (x < 16),  H_i[x] = m_i^(16x) (x < 32):  a_i m_i^(s+s0) = P_i[s & 15] * H_i[s >> 4]
// for s = sb0 + 16 s2 + s1, a deferred sum over i with no modular product in the inner loop (PAPER.md L205-209,
// L219-225).  A lane owns a 2 x 2 block of (s1, s2): two 16-byte reads of shared memory serve four multiply-adds
// (one 8-byte read each would make shared memory, not the multiplier, the limit: two wavefronts per multiply-add).
// Where the block holds fewer than 512 wanted s (short functions) the lanes left over split the nodes of a tile among
// groups instead (group g takes the nodes x = g mod ng) and the groups' residues are added at the end.
// ------------------------------------------------------------------------------------------------
#define ZP_K6_THREADS 128
#define ZP_K6_NODES 64
#define ZP_K6_SBLOCK 512
__global__ void __launch_bounds__(ZP_K6_THREADS)
k_power_sums(const uint64_t* __restrict__ nodes, const int64_t* __restrict__ offsets, int F,
             const uint64_t* __restrict__ coef, int64_t T_tot, int B, int s0, ZpMod k, uint64_t* __restrict__ out) {
  __shared__ ulonglong2 sP[ZP_K6_NODES * 8];   // Montgomery: {P_i[2a], P_i[2a+1]} at [i * 8 + a]
  __shared__ ulonglong2 sH[ZP_K6_NODES * 16];  // plain: {H_i[2c], H_i[2c+1]} at [i * 16 + c]
  const int a = threadIdx.x & 7;
  for (int f = blockIdx.y; f < F; f += gridDim.y) {
    const int64_t off = offsets[f];
    const int t = (int)(offsets[f + 1] - off);
    const int sb0 = blockIdx.x * ZP_K6_SBLOCK;
    if (sb0 >= t) continue;
    int cr = 1;  // 32 cr >= the wanted s of this block, a power of two <= 16; ng = 16 / cr groups share the nodes
    while (32 * cr < t - sb0 && cr < 16) cr <<= 1;
    const int ng = 16 / cr, c = (threadIdx.x >> 3) & (cr - 1), grp = (threadIdx.x >> 3) / cr;
    const int ls = 32 * c + 2 * a, s = sb0 + ls;  // this lane: s, s + 1, s + 16, s + 17
    for (int b = 0; b < B; ++b) {
      Acc acc[4];
#pragma unroll
      for (int x = 0; x < 4; ++x) acc_zero(acc[x]);
      for (int i0 = 0; i0 < t; i0 += ZP_K6_NODES) {
        const int n = t - i0 < ZP_K6_NODES ? t - i0 : ZP_K6_NODES;
        __syncthreads();
        {  // two builder lanes per node: lane (x, 0) fills P_x, lane (x, 1) fills H_x
          const int x = threadIdx.x >> 1, which = threadIdx.x & 1;
          if (x < n) {
            const uint64_t m = to_mont(zp_canon(nodes[off + i0 + x], k.p), k);
            uint64_t* dst;
            uint64_t pw, step;
            int cnt;
            if (which == 0) {
              const uint64_t av = to_mont(zp_canon(coef[(int64_t)b * T_tot + off + i0 + x], k.p), k);
              const int e0 = sb0 + s0;
              pw = e0 == 0 ? av : e0 == 1 ? mont_mul(av, m, k) : mont_mul(av, mont_pow(m, (uint64_t)e0, k), k);
              step = m;
              dst = reinterpret_cast<uint64_t*>(sP + x * 8);
              cnt = 16;
            } else {
              step = m;
              for (int e = 0; e < 4; ++e) step = mont_mul(step, step, k);
              pw = 1 % k.p;  // plain; plain * Montgomery -> plain
              dst = reinterpret_cast<uint64_t*>(sH + x * 16);
              cnt = 32;
            }
            for (int e = 0; e < cnt; ++e) {
              dst[e] = pw;
              pw = mont_mul(pw, step, k);
            }
          }
        }
        __syncthreads();
        const ulonglong2* pP = sP + a;
        const ulonglong2* pH = sH + c;
#pragma unroll 2
        for (int x = grp; x < n; x += ng) {
          const ulonglong2 P = pP[x * 8], H = pH[x * 16];
          acc_mac(acc[0], P.x, H.x);
          acc_mac(acc[1], P.y, H.x);
          acc_mac(acc[2], P.x, H.y);
          acc_mac(acc[3], P.y, H.y);
        }
      }
      uint64_t r[4];  // Montgomery * plain sums
#pragma unroll
      for (int x = 0; x < 4; ++x) r[x] = mont_mul(acc_redc160(acc[x], k), k.c160, k);
      if (ng > 1) {  // (uniform) the groups' partial sums meet in shared memory, over the tables
        uint64_t* red = reinterpret_cast<uint64_t*>(sH);  // [ng][32 cr] = 512 words
        __syncthreads();
#pragma unroll
        for (int x = 0; x < 4; ++x) red[grp * 32 * cr + ls + (x & 1) + 16 * (x >> 1)] = r[x];
        __syncthreads();
        if (grp == 0)
#pragma unroll
          for (int x = 0; x < 4; ++x)
            for (int g = 1; g < ng; ++g) r[x] = mod_add(r[x], red[g * 32 * cr + ls + (x & 1) + 16 * (x >> 1)], k.p);
      }
      uint64_t* o = out + (int64_t)b * T_tot + off;
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        const int sx = s + (x & 1) + 16 * (x >> 1);
        if (grp == 0 && sx < t) o[sx] = r[x];
      }
    }
  }
}

// (a6) K7 balance: V_{j,s} = u_{j,s} * R_s / u_{0,s}   (eq. (4), readings G3, G20), in two launches:
// k_balance_scale: w_s = R_s / u_{0,s} for every slot s, as the plain residue with its Shoup companion; the pivots
//   u_{0,s} are inverted 256 x ZP_BAL_N at a time per CTA (cta_batch_inv above); u_{0,s} = 0 -> ZP_ST_ZERO_PIVOT, w_s = 0.
// k_balance_apply: the HBM stream (16 bytes per probe): a CTA takes 256 x ZP_BAL_N slots x ZP_BAL_ROWS rows, the
//   multiplier of a column stays in registers down its rows, one Shoup product (any 64-bit u in, no canonicalisation
//   before it) and one conditional subtraction per probe.  The grid is (slot blocks) x (row blocks): enough CTAs for
//   an even spread over the SMs whatever the batch's shape.
#define ZP_BAL_N 4
#define ZP_BAL_ROWS 8
__global__ void __launch_bounds__(256)
k_balance_scale(const uint64_t* __restrict__ u, const uint64_t* __restrict__ R, const int64_t* __restrict__ offsets, int F,
                int64_t T_tot, ZpMod k, ulonglong2* __restrict__ sc, int32_t* __restrict__ pre) {
  __shared__ uint64_t sh[64];
  for (int64_t c0 = (int64_t)blockIdx.x * (256 * ZP_BAL_N); c0 < T_tot; c0 += (int64_t)gridDim.x * (256 * ZP_BAL_N)) {
    const int64_t x0 = c0 + threadIdx.x;
    uint64_t w[ZP_BAL_N];
#pragma unroll
    for (int y = 0; y < ZP_BAL_N; ++y) {
      const int64_t x = x0 + 256 * y;
      w[y] = (x < T_tot) ? to_mont(zp_canon(u[x], k.p), k) : k.r1;
    }
    const uint32_t zero = cta_batch_inv<ZP_BAL_N>(w, k, sh);
#pragma unroll
    for (int y = 0; y < ZP_BAL_N; ++y) {
      const int64_t x = x0 + 256 * y;
      if (x >= T_tot) continue;
      if (zero >> y & 1) {
        int lo = 0, hi = F;  // function of slot x: offsets[lo] <= x < offsets[lo+1]
        while (hi - lo > 1) {
          const int mid = (lo + hi) >> 1;
          if (offsets[mid] <= x) lo = mid; else hi = mid;
        }
        atomicMin(&pre[lo], (int32_t)(((uint32_t)(x - offsets[lo]) << 8) | ZP_ST_ZERO_PIVOT));
        sc[x] = make_ulonglong2(0, 0);
      } else {
        const uint64_t wm = mont_mul(to_mont(R[x], k), w[y], k);  // (R_s / u_{0,s})~
        sc[x] = make_ulonglong2(from_mont(wm, k), shoup_companion(wm, k));
      }
    }
  }
}
__global__ void __launch_bounds__(256)
k_balance_apply(const uint64_t* __restrict__ u, const ulonglong2* __restrict__ sc, int64_t T_tot, int B, ZpMod k,
                uint64_t* __restrict__ V) {
  const int64_t x0 = (int64_t)blockIdx.x * (256 * ZP_BAL_N) + threadIdx.x;
  const int j0 = blockIdx.y * ZP_BAL_ROWS, j1 = (j0 + ZP_BAL_ROWS < B) ? j0 + ZP_BAL_ROWS : B;
  ulonglong2 w[ZP_BAL_N];
#pragma unroll
  for (int y = 0; y < ZP_BAL_N; ++y) w[y] = (x0 + 256 * y < T_tot) ? __ldg(sc + x0 + 256 * y) : make_ulonglong2(0, 0);
#pragma unroll 2
  for (int j = j0; j < j1; ++j) {  // (unrolled: the loads of two rows, eight words a lane, are in flight together)
    uint64_t v[ZP_BAL_N];
#pragma unroll
    for (int y = 0; y < ZP_BAL_N; ++y) v[y] = (x0 + 256 * y < T_tot) ? __ldcs(u + (int64_t)j * T_tot + x0 + 256 * y) : 0;
#pragma unroll
    for (int y = 0; y < ZP_BAL_N; ++y)
      if (x0 + 256 * y < T_tot) __stcs(V + (int64_t)j * T_tot + x0 + 256 * y, shoup_mul(v[y], w[y], k));
  }
}

// ------------------------------------------------------------------------------------------------
// (f2) Thiele reconstruction in one variable, one lane per column of values (eq. (2)):
//   f(x) = b_0 + (x - x_0) / (b_1 + (x - x_1) / (b_2 + ...)),   b_k = phi_k(x_k),
//   phi_0(x_j) = f(x_j),  phi_k(x_j) = (x_j - x_{k-1}) / (phi_{k-1}(x_j) - phi_{k-1}(x_{k-1})),  j >= k.
// Level k inverts its T - k differences with ONE modular inverse (prefix products, Montgomery's trick; the
// batched inversion of SURVEY.md row a4).  The fraction ends at K = k when all differences of level k vanish;
// some but not all vanishing -> ZP_ST_THIELE_DEGENERATE.  Expansion from the tail, in place in two columns:
//   (N, D) <- (b_k N + (x - x_k) D, N),  then trim to the true degrees and scale D monic.
// Columns live in shared memory (column stride = lanes per CTA); everything is in Montgomery form.
// k_thiele_prep: xd[j*T + k] = {x_j - x_k, companion}, xm[j] = {x_j, companion} (plain residues with their Shoup
// companions, modarith.cuh), duplicate check.
// ------------------------------------------------------------------------------------------------
#define ZP_ST_THIELE_DEGENERATE 20
__global__ void k_thiele_prep(const uint64_t* __restrict__ points, int T, ZpMod k, ulonglong2* __restrict__ xd,
                              ulonglong2* __restrict__ xm, int32_t* __restrict__ dup) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= T * T) return;
  const int j = idx / T, kk = idx % T;
  const uint64_t xj = zp_canon(points[j], k.p);
  const uint64_t diff = mod_sub(xj, zp_canon(points[kk], k.p), k.p);
  if (kk < j && diff == 0) atomicMin(dup, (int32_t)(((uint32_t)j << 8) | ZP_ST_DUPLICATE_SAMPLE));
  xd[idx] = make_ulonglong2(diff, shoup_companion(to_mont(diff, k), k));
  if (kk == 0) xm[j] = make_ulonglong2(xj, shoup_companion(to_mont(xj, k), k));
}

#define ZP_K8_THREADS 64
// x * w mod p, lazily ([0, 2p) out, any 64-bit x in), for a multiplier w in [0, p) with its companion
ZP_DEV uint64_t shoup_lazy(uint64_t x, uint64_t w, uint64_t wc, const ZpMod& k) { return shoup_mul_lazy(x, w, wc, k); }
// The inverse differences are carried as fractions phi_k(x_j) = A_j / B_j, so that a level is four independent products
// per point and no inversion:
//   A_j <- (x_j - x_{k-1}) B_j B_p ,   B_j <- A_j B_p - A_p B_j      (p = k-1, the pivot; j = k .. T-1),
// B_j = 0 <=> the oracle's zero denominator.  Every product of a level has a FIXED multiplier -- the pivot's A_p or B_p
// (per lane: their Shoup companions cost one Montgomery product and one low product per level) or the table entry
// x_j - x_{k-1} -- so all four are Shoup products (16 multiplier-pipe units and no carry plumbing, against 18 and more
// for a Montgomery product); the values are plain residues, lazy where they only feed another product, and a common
// factor picked up along the way cancels in A_j / B_j.  The b_k = A_k / B_k come from ONE batched inversion at the end
// (prefix products, Montgomery's trick), the monic scaling from a second one: 2 inversions per column in all.  The
// expansion (N, D) <- (b_k N + (x - x_k) D, N) multiplies by b_k (per lane and step) and x_k (table): Shoup again.
__global__ void __launch_bounds__(ZP_K8_THREADS)
k_thiele(const ulonglong2* __restrict__ xd, const ulonglong2* __restrict__ xm, const int32_t* __restrict__ dup, int T,
         const uint64_t* __restrict__ vals, int64_t n, int64_t ld, ZpMod k, uint64_t* __restrict__ num,
         uint64_t* __restrict__ den, int32_t* __restrict__ degs, uint64_t* __restrict__ cf, int32_t* __restrict__ status) {
  extern __shared__ __align__(16) uint64_t sh[];
  constexpr int TH = ZP_K8_THREADS;
  uint64_t* Ac = sh + threadIdx.x;                 // column A_j (ends as b_0 .. b_{K-1}), stride TH
  uint64_t* Bc = Ac + (size_t)(T + 2) * TH;        // column B_j; later N (slots 0 ..) and D (slots T/2+1 ..)
  const int32_t dupst = dup[0];
  const uint64_t p = k.p;
  for (int64_t i = (int64_t)blockIdx.x * TH + threadIdx.x; i < n; i += (int64_t)gridDim.x * TH) {
    for (int d = 0; d < T; ++d) {
      num[d * ld + i] = 0;
      den[d * ld + i] = 0;
      if (cf) cf[d * ld + i] = 0;
    }
    degs[i] = -1;
    degs[ld + i] = -1;
    if (dupst != ZP_ST_NONE) {
      status[i] = dupst;
      continue;
    }
    for (int j = 0; j < T; ++j) {
      Ac[j * TH] = zp_canon(vals[j * ld + i], p);
      Bc[j * TH] = 1 % p;
    }
    int K = T, bad = 0;
    for (int kk = 1; kk < T; ++kk) {
      const uint64_t Ap = lazy_canon(Ac[(kk - 1) * TH], p), Bp = Bc[(kk - 1) * TH];  // A lazy in [0, 2p), B canonical
      const uint64_t Apc = shoup_companion(to_mont(Ap, k), k), Bpc = shoup_companion(to_mont(Bp, k), k);
      const ulonglong2* xrow = xd + (kk - 1);  // xd[j*T + kk-1] = x_j - x_{kk-1}
      int zeros = 0;
      int j = kk;
      for (; j + 1 < T; j += 2) {  // two points at a time: eight independent products in flight
        const uint64_t a0 = Ac[j * TH], b0 = Bc[j * TH], a1 = Ac[(j + 1) * TH], b1 = Bc[(j + 1) * TH];
        const ulonglong2 x0 = __ldg(xrow + (size_t)j * T), x1 = __ldg(xrow + (size_t)(j + 1) * T);
        // (2p can exceed 2^63: each lazy product is brought to [0, p) before the difference)
        const uint64_t nb0 = mod_sub(lazy_canon(shoup_lazy(a0, Bp, Bpc, k), p), lazy_canon(shoup_lazy(b0, Ap, Apc, k), p), p);
        const uint64_t nb1 = mod_sub(lazy_canon(shoup_lazy(a1, Bp, Bpc, k), p), lazy_canon(shoup_lazy(b1, Ap, Apc, k), p), p);
        const uint64_t na0 = shoup_lazy(shoup_lazy(b0, Bp, Bpc, k), x0.x, x0.y, k);
        const uint64_t na1 = shoup_lazy(shoup_lazy(b1, Bp, Bpc, k), x1.x, x1.y, k);
        zeros += (nb0 == 0) + (nb1 == 0);
        Ac[j * TH] = na0;
        Bc[j * TH] = nb0;
        Ac[(j + 1) * TH] = na1;
        Bc[(j + 1) * TH] = nb1;
      }
      if (j < T) {
        const uint64_t a0 = Ac[j * TH], b0 = Bc[j * TH];
        const ulonglong2 x0 = __ldg(xrow + (size_t)j * T);
        const uint64_t nb0 = mod_sub(lazy_canon(shoup_lazy(a0, Bp, Bpc, k), p), lazy_canon(shoup_lazy(b0, Ap, Apc, k), p), p);
        Ac[j * TH] = shoup_lazy(shoup_lazy(b0, Bp, Bpc, k), x0.x, x0.y, k);
        Bc[j * TH] = nb0;
        zeros += (nb0 == 0);
      }
      if (zeros == T - kk) {
        K = kk;
        break;
      }
      if (zeros != 0) {
        bad = kk;
        break;
      }
    }
    if (bad) {
      status[i] = (int32_t)(((uint32_t)bad << 8) | ZP_ST_THIELE_DEGENERATE);
      continue;
    }
    // b_k = A_k / B_k, k < K, by one batched inversion; the prefix products are parked in this lane's own
    // output column num[., i] (global, unit stride across lanes, overwritten with the result below).  The values are
    // plain, so the running product picks up 2^-64 per step: run_k = B_0 .. B_k 2^(-64 k), and with
    // I_k = mont_inv(run_k) = 2^128 / run_k:  mont_mul(I_k, run_{k-1}) = 2^128 / B_k,  I_{k-1} = mont_mul(I_k, B_k).
    {
      uint64_t run = Bc[0];
      num[i] = run;
      for (int kk = 1; kk < K; ++kk) {
        run = mont_mul(run, Bc[kk * TH], k);
        num[kk * ld + i] = run;  // scratch: prefix products (overwritten with zeros / results below)
      }
      uint64_t inv = mont_inv(run, k);
      for (int kk = K - 1; kk >= 0; --kk) {
        const uint64_t invk = (kk > 0) ? mont_mul(inv, num[(kk - 1) * ld + i], k) : inv;  // 2^128 / B_k
        inv = mont_mul(inv, Bc[kk * TH], k);
        Ac[kk * TH] = mont_mul(mont_mul(Ac[kk * TH], invk, k), 1, k);  // b_k, plain and canonical
        num[kk * ld + i] = 0;
      }
    }
    if (cf)
      for (int kk = 0; kk < K; ++kk) cf[kk * ld + i] = Ac[kk * TH];
    // expansion from the tail, in place: after s steps deg N <= (s+1)/2, deg D <= s/2
    uint64_t* Nc = Bc;
    uint64_t* Dc = Bc + (size_t)(T / 2 + 1) * TH;
    const int half = T / 2;
    for (int d = 0; d <= half; ++d) Nc[d * TH] = Dc[d * TH] = 0;
    Nc[0] = Ac[(K - 1) * TH];
    Dc[0] = 1 % p;
    for (int kk = K - 2, s2 = 1; kk >= 0; --kk, ++s2) {
      const uint64_t bk = Ac[kk * TH];
      const uint64_t bkc = shoup_companion(to_mont(bk, k), k);
      const ulonglong2 xk = __ldg(xm + kk);
      for (int d = (s2 + 1) / 2; d >= 0; --d) {  // descending: D[d-1] is still the old one
        const uint64_t Nd = Nc[d * TH], Dd = Dc[d * TH];
        uint64_t v = lazy_canon(shoup_lazy(Nd, bk, bkc, k), p);
        if (d >= 1) v = mod_add(v, Dc[(d - 1) * TH], p);
        v = mod_sub(v, lazy_canon(shoup_lazy(Dd, xk.x, xk.y, k), p), p);
        Dc[d * TH] = Nd;
        Nc[d * TH] = v;
      }
    }
    int dn = (K - 1 + 1) / 2, dd = (K - 1) / 2;
    while (dn >= 0 && Nc[dn * TH] == 0) --dn;
    while (dd >= 0 && Dc[dd * TH] == 0) --dd;
    if (dd < 0) {
      status[i] = (int32_t)ZP_ST_THIELE_DEGENERATE;
      continue;
    }
    const uint64_t sc = mont_inv(to_mont(Dc[dd * TH], k), k);  // (1 / lc D)~: plain x Montgomery -> plain
    for (int d = 0; d <= dn; ++d) num[d * ld + i] = mont_mul(Nc[d * TH], sc, k);
    for (int d = 0; d <= dd; ++d) den[d * ld + i] = mont_mul(Dc[d * TH], sc, k);
    degs[i] = dn;
    degs[ld + i] = dd;
    status[i] = 0;
  }
}

// ------------------------------------------------------------------------------------------------
// (f1) skeleton extension between two lifting steps: the pairs (term i,
// degree d) with a non-zero monomial coefficient become the terms of the next skeleton, in the order i
// ascending, d ascending.  An HBM-bound stream compaction in ONE pass over the coefficient matrix:
//   a CTA takes the next block of ZP_K9_BLOCK consecutive terms (a ticket, so that blocks start in index order), reads their
//   B coefficients (unit-stride rows), keeps a 64-bit mask of the non-zero degrees per term (B <= 64), scans the
//   popcounts inside the block, obtains the number of rows emitted by all earlier blocks by a decoupled look-back
//   over the per-block descriptors {flag, count} (flag 1: the block's own count, 2: the inclusive prefix; one 64-bit
//   word each, so a plain load sees a consistent pair), and writes its rows (exps row, d), coefficients (re-read: the
//   lines are still in L1 / L2), the new offsets of the functions that start inside the block and the per-function
//   maximum degree (the early-termination test).
// desc: [nb + 1] words, zeroed before the launch; desc[nb] is the ticket counter.  stage_rows: rows of the staging buffer in
// dynamic shared memory (stage_rows x (8 + 2 (nv + 1)) bytes, then the block's exponent rows, 2 nv BLOCK bytes + 16); blocks
// that emit more rows than that write them directly.
// ------------------------------------------------------------------------------------------------
#define ZP_K9_THREADS 256
#define ZP_K9_ITEMS 4  // consecutive terms per lane: 32 contiguous bytes of every coefficient row (with 8 the kernel needs 80
                       // registers and three CTAs fill an SM; with 4, five do: 0.262 -> 0.238 ms on C2's output; with 2: 0.278)
#define ZP_K9_BLOCK (ZP_K9_THREADS * ZP_K9_ITEMS)
__global__ void __launch_bounds__(ZP_K9_THREADS, 5)
k_ext_fused(const uint16_t* __restrict__ exps, int nv, const uint64_t* __restrict__ coefs, int64_t T_tot, int B,
            const int64_t* __restrict__ offsets, int F, ZpMod k, unsigned long long* __restrict__ desc, int64_t nb,
            uint16_t* __restrict__ new_exps, uint64_t* __restrict__ new_coefs, int64_t cap, int64_t* __restrict__ new_offsets,
            int32_t* __restrict__ degs, int stage_rows) {
  __shared__ int32_t wsum[ZP_K9_THREADS / 32];
  __shared__ long long s_base;
  __shared__ int s_bid, s_flo, s_fhi;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_bid = (int)atomicAdd(desc + nb, 1ull);
  __syncthreads();
  const int64_t bid = s_bid;
  const int64_t i0 = bid * ZP_K9_BLOCK, i1 = i0 + (int64_t)threadIdx.x * ZP_K9_ITEMS;  // this lane: terms i1 .. i1 + ITEMS - 1
  // ---- the one pass over the coefficients: masks of the non-zero degrees of the lane's terms
  uint64_t m[ZP_K9_ITEMS], c1[ZP_K9_ITEMS];  // c1: the term's first non-zero coefficient (no second read for it)
#pragma unroll
  for (int x = 0; x < ZP_K9_ITEMS; ++x) m[x] = c1[x] = 0;
  if (i1 + ZP_K9_ITEMS <= T_tot && (T_tot & 1) == 0) {  // whole group, rows 16-byte aligned: two 16-byte loads per row
#pragma unroll 4
    for (int d = 0; d < B; ++d) {
      const ulonglong2* src = reinterpret_cast<const ulonglong2*>(coefs + (int64_t)d * T_tot + i1);
      ulonglong2 v[ZP_K9_ITEMS / 2];
#pragma unroll
      for (int x = 0; x < ZP_K9_ITEMS / 2; ++x) v[x] = __ldcs(src + x);
#pragma unroll
      for (int x = 0; x < ZP_K9_ITEMS; ++x) {
        const uint64_t cv = zp_canon((x & 1) ? v[x >> 1].y : v[x >> 1].x, k.p);
        c1[x] = m[x] ? c1[x] : cv;
        m[x] |= (uint64_t)(cv != 0) << d;
      }
    }
  } else {
    for (int d = 0; d < B; ++d)
#pragma unroll
      for (int x = 0; x < ZP_K9_ITEMS; ++x)
        if (i1 + x < T_tot) {
          const uint64_t cv = zp_canon(coefs[(int64_t)d * T_tot + i1 + x], k.p);
          c1[x] = m[x] ? c1[x] : cv;
          m[x] |= (uint64_t)(cv != 0) << d;
        }
  }
  // ---- the block's exponent rows -> shared memory (unit-stride 16-byte loads; in flight during the scan and the look-back)
  extern __shared__ __align__(16) unsigned char ext_smem[];
  uint64_t* sc = reinterpret_cast<uint64_t*>(ext_smem);                               // [stage_rows] coefficients
  uint16_t* sr = reinterpret_cast<uint16_t*>(ext_smem + 8 * (size_t)stage_rows);      // [stage_rows x (nv + 1)] rows
  uint16_t* se = sr + (size_t)stage_rows * (nv + 1) + ((stage_rows * (nv + 1)) & 1 ? 1 : 0) + 0;  // [BLOCK x nv] exponents
  se = reinterpret_cast<uint16_t*>((reinterpret_cast<uintptr_t>(se) + 15) & ~(uintptr_t)15);
  if (stage_rows) {
    const int64_t nterm = (T_tot - i0 < ZP_K9_BLOCK) ? T_tot - i0 : ZP_K9_BLOCK;
    const int n16 = (int)((nterm * nv * 2) / 16), rem0 = n16 * 8;  // 16-byte pieces, then the u16 tail
    const uint4* src = reinterpret_cast<const uint4*>(exps + i0 * nv);  // i0 nv 2 bytes: a multiple of 16
    for (int x = threadIdx.x; x < n16; x += ZP_K9_THREADS) reinterpret_cast<uint4*>(se)[x] = src[x];
    for (int x = rem0 + threadIdx.x; x < nterm * nv; x += ZP_K9_THREADS) se[x] = exps[i0 * nv + x];
  }
  // ---- block scan of the lanes' row counts
  int c = 0;
#pragma unroll
  for (int x = 0; x < ZP_K9_ITEMS; ++x) c += __popcll(m[x]);
  int incl = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  if (lane == 31) wsum[warp] = incl;
  if (threadIdx.x == 0) {  // functions that start inside the block: flo = first f with offsets[f] >= i0, fhi = first beyond
    int lo = 0, hi = F + 1;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (offsets[mid] < i0) lo = mid + 1; else hi = mid;
    }
    s_flo = lo;
    hi = F + 1;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (offsets[mid] < i0 + ZP_K9_BLOCK) lo = mid + 1; else hi = mid;
    }
    s_fhi = lo;
  }
  __syncthreads();
  int base_w = 0, total = 0;
#pragma unroll
  for (int w = 0; w < ZP_K9_THREADS / 32; ++w) {
    if (w < warp) base_w += wsum[w];
    total += wsum[w];
  }
  const int lpos = base_w + incl - c;
  // ---- rows emitted by the earlier blocks: decoupled look-back by the first warp
  if (warp == 0) {
    volatile unsigned long long* vd = desc;
    if (lane == 0) vd[bid] = ((bid == 0 ? 2ull : 1ull) << 62) | (unsigned long long)total;
    long long excl = 0;
    int64_t j = bid - 1;
    while (j >= 0) {
      const int64_t jj = j - lane;
      unsigned long long w = 2ull << 62;  // before the first block: an inclusive prefix of 0
      if (jj >= 0) {
        do {
          w = vd[jj];
        } while ((w >> 62) == 0);
      }
      const unsigned fl = (unsigned)(w >> 62);
      const unsigned done = __ballot_sync(0xffffffffu, fl == 2);
      const int first = done ? __ffs(done) - 1 : 32;  // the nearest block that knows its inclusive prefix
      long long v = (lane <= first) ? (long long)(w & ((1ull << 62) - 1)) : 0;
#pragma unroll
      for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      excl += v;
      if (done) break;
      j -= 32;
    }
    if (lane == 0) {
      if (bid > 0) vd[bid] = (2ull << 62) | (unsigned long long)(excl + total);
      s_base = excl;
    }
  }
  __syncthreads();
  const int64_t base = s_base;
  const int flo = s_flo, fhi = s_fhi;
  // ---- new offsets of the functions that start in this block (the lane that owns the first term writes); the total
  for (int f = flo; f < fhi; ++f) {
    const int64_t o = offsets[f] - i1;
    if (o >= 0 && o < ZP_K9_ITEMS && offsets[f] < T_tot) {
      int before = 0;
#pragma unroll
      for (int x = 0; x < ZP_K9_ITEMS; ++x) before += (x < o) ? __popcll(m[x]) : 0;
      new_offsets[f] = base + lpos + before;
    }
  }
  if (i0 + ZP_K9_BLOCK >= T_tot && threadIdx.x == 0) new_offsets[F] = base + total;
  // ---- per-function maximum degree (the early-termination test): function of a term = the last start at or before
  // it; one atomic per warp when the warp lies inside one function (the usual case), else one per term
  auto fn_of = [&](int64_t i) {
    int lo = flo > 0 ? flo - 1 : 0, hi = fhi;  // offsets[lo] <= i; find the last g < hi with offsets[g] <= i
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (offsets[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
  };
  if (i1 < T_tot) {
    const int64_t ilast = (i1 + ZP_K9_ITEMS <= T_tot ? i1 + ZP_K9_ITEMS : T_tot) - 1;
    const int fa = fn_of(i1), fb = (flo == fhi) ? fa : fn_of(ilast);
    uint64_t all = 0;
#pragma unroll
    for (int x = 0; x < ZP_K9_ITEMS; ++x) all |= m[x];
    const int deg = all ? 63 - __clzll((long long)all) : -1;
    const unsigned act = __activemask();
    const int f0 = __shfl_sync(act, fa, __ffs(act) - 1);
    if (__all_sync(act, fa == f0 && fb == f0)) {
      const int wmax = __reduce_max_sync(act, deg);
      if (lane == __ffs(act) - 1 && wmax >= 0) atomicMax(&degs[f0], wmax);
    } else if (fa == fb) {
      if (deg >= 0) atomicMax(&degs[fa], deg);
    } else {
#pragma unroll
      for (int x = 0; x < ZP_K9_ITEMS; ++x)
        if (m[x]) atomicMax(&degs[fn_of(i1 + x)], 63 - __clzll((long long)m[x]));
    }
  }
  // ---- emit.  Usual case (the block's rows fit the staging buffer): rows and coefficients go to shared memory at
  // their local positions and the block writes its contiguous output range with unit-stride stores
  if (total <= stage_rows && base + total <= cap) {  // uniform
    const int rw = nv + 1;
    if (i1 < T_tot) {
      int lp = lpos;
#pragma unroll
      for (int x = 0; x < ZP_K9_ITEMS; ++x) {
        uint64_t mm = m[x];
        const int64_t i = i1 + x;
        bool first = true;
        while (mm) {
          const int d = __ffsll((long long)mm) - 1;
          mm &= mm - 1;
          uint16_t* row = sr + lp * rw;
          const uint16_t* er = se + (i - i0) * nv;
          for (int j = 0; j < nv; ++j) row[j] = er[j];
          row[nv] = (uint16_t)d;
          sc[lp] = first ? c1[x] : zp_canon(coefs[(int64_t)d * T_tot + i], k.p);
          first = false;
          ++lp;
        }
      }
    }
    __syncthreads();
    for (int x = threadIdx.x; x < total; x += ZP_K9_THREADS) new_coefs[base + x] = sc[x];
    uint16_t* dst = new_exps + base * rw;
    for (int x = threadIdx.x; x < total * rw; x += ZP_K9_THREADS) dst[x] = sr[x];
    return;
  }
  if (i1 >= T_tot) return;
  int64_t pos = base + lpos;
#pragma unroll
  for (int x = 0; x < ZP_K9_ITEMS; ++x) {
    uint64_t mm = m[x];
    const int64_t i = i1 + x;
    bool first = true;
    while (mm && pos < cap) {
      const int d = __ffsll((long long)mm) - 1;
      mm &= mm - 1;
      uint16_t* row = new_exps + pos * (nv + 1);
      for (int j = 0; j < nv; ++j) row[j] = exps[i * nv + j];
      row[nv] = (uint16_t)d;
      new_coefs[pos] = first ? c1[x] : zp_canon(coefs[(int64_t)d * T_tot + i], k.p);
      first = false;
      ++pos;
    }
    pos += __popcll(mm);  // rows beyond cap are counted, not written
  }
}

// ------------------------------------------------------------------------------------------------
// (f4) two-prime CRT + rational reconstruction, one lane per coefficient:
//   x = r1 + p1 ((r2 - r1) p1^-1 mod p2) in [0, m = p1 p2);  extended Euclid on (m, x) down to the first
//   remainder <= N = floor(sqrt((m-1)/2)) (Wang's bounds);  a/b = remainder / cofactor, b > 0, b <= N, gcd 1.
// 128-bit remainders, 64-bit cofactor magnitudes; Euclid's quotients come from a double-precision estimate and one
// correction (no subtraction ladder, no 128-bit division on the usual path).  The number of steps is data-dependent
// (about 37 on average for two 63-bit primes); HBM traffic 32 B/lane.
// ------------------------------------------------------------------------------------------------
#define ZP_ST_NO_RATIONAL 21
typedef unsigned __int128 zp_u128;
typedef __int128 zp_i128;
__global__ void __launch_bounds__(256)
k_crt_rational(const uint64_t* __restrict__ r1, const uint64_t* __restrict__ r2, int64_t n, uint64_t p1, ZpMod k2,
               uint64_t p1inv, uint64_t m_hi, uint64_t m_lo, uint64_t N, int64_t* __restrict__ num,
               int64_t* __restrict__ den, int32_t* __restrict__ status) {
  const zp_u128 m = ((zp_u128)m_hi << 64) | m_lo;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const uint64_t a1 = zp_canon(r1[i], p1), a2 = zp_canon(r2[i], k2.p);
    const uint64_t diff = mod_sub(a2, zp_canon(a1, k2.p), k2.p);
    const uint64_t h = mont_mul(to_mont(diff, k2), p1inv, k2);  // Montgomery x plain -> plain: diff / p1 mod p2
    const zp_u128 x = (zp_u128)a1 + (zp_u128)p1 * h;
    // cofactors: t_i alternates in sign and |t_i| <= m / r_{i-1} < 2^64 while r_{i-1} > N, so the magnitudes fit 64 bits
    // and |t_{i+1}| = |t_{i-1}| + q |t_i| needs no 128-bit product; sign(t_i) = (-1)^(i+1) (t_0 = 0, t_1 = 1)
    zp_u128 ra = m, rb = x;
    uint64_t ta = 0, tb = 1;
    bool tb_neg = false;
    while (rb > N) {
      // quotient: estimate in double precision (relative error about 2^-52, so off by at most one for q < 2^50), then
      // one multiply-subtract and the corrections; the exact 128-bit division only for the quotients beyond that
      // (probability about 2^-50 per step).  Every lane takes the same path: no subtraction ladder, no divergence.
      uint64_t q;
      zp_u128 rn;
      const double da = __ull2double_rn((uint64_t)(ra >> 64)) * 18446744073709551616.0 + __ull2double_rn((uint64_t)ra);
      const double db = __ull2double_rn((uint64_t)(rb >> 64)) * 18446744073709551616.0 + __ull2double_rn((uint64_t)rb);
      const double qd = da / db;
      if (qd < 1125899906842624.0) {  // 2^50
        q = (uint64_t)qd;
        rn = ra - (zp_u128)q * rb;  // modulo 2^128; the true value lies in (-rb, 2 rb)
        if ((zp_i128)rn < 0) {
          rn += rb;
          --q;
        }
        if (rn >= rb) {
          rn -= rb;
          ++q;
        }
      } else {
        q = (uint64_t)(ra / rb);
        rn = ra - (zp_u128)q * rb;
      }
      const uint64_t tn = ta + q * tb;  // q tb <= |t_{i+1}| < 2^64
      ra = rb;
      rb = rn;
      ta = tb;
      tb = tn;
      tb_neg = !tb_neg;
    }
    zp_i128 a = (zp_i128)rb;
    const uint64_t b = tb;
    if (tb_neg) a = -a;
    bool ok = (b > 0) && (b <= N);
    if (ok) {
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
    status[i] = ok ? 0 : ZP_ST_NO_RATIONAL;
  }
}
