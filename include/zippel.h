/*
 * zippel.h -- C-ABI of libzippel.so: one Zippel lifting step k-1 -> k variables over Z/pZ on a
 * B200 (sm_100a).  Method: arXiv 2505.24256, "GPU Implementation of Zippel Method for Feynman
 * Integral Reconstruction" (PAPER.md below = /root/reference/PAPER.md; Gn = readings in DESIGN.md).
 *
 * Conventions for every entry point
 *   - Pointers are DEVICE pointers unless the name starts with h_ (host).  The caller owns every
 *     buffer; the library allocates no device memory and keeps no per-call state.  Scratch comes from
 *     the caller's `workspace` (device, 256-byte aligned, zippel_workspace_bytes() bytes).  Process-wide
 *     state, all of it listed here: the tuning knobs (zippel_set_tuning), the measurement hook and launch
 *     counter (zippel_profile_events, zippel_launch_count), and the two copy streams + events that
 *     zippel_lift_step_host creates per device on first use (zippel_shutdown destroys them).  None of it
 *     is thread-safe: one host thread per process calls the library.
 *   - Calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = default stream).
 *   - Residues are canonical, in [0, p); p is an odd prime, 3 <= p < 2^63 (primality is the caller's
 *     contract; reading G14, G22).  There is no ZP_FLAG_CHECK_RANGE / ZP_ST_RANGE (SURVEY.md 8(b) proposed
 *     them): every kernel canonicalises each input word as it loads it (x < p ? x : x % p), so a residue
 *     >= p gives the result of its canonical representative instead of a status.
 *   - Batch layout: F functions, function f owns the terms [h_offsets[f], h_offsets[f+1]);
 *     T_tot = h_offsets[F] < 2^31.  A "[B x T_tot]" array holds row b at x + b*T_tot; inside a row the
 *     entries of function f start at h_offsets[f].  One function has at most 2^23 - 1 terms (the status
 *     word keeps 23 bits for the index; the NTT engine's longest transform is 2^24).
 *   - Return value: ZP_OK, or an error found on the host before anything was enqueued.
 *     Data-dependent failures are written to status[f] (device int32): 0 = ok, else
 *     (index << 8) | code with the smallest offending index.  Outputs of a failed function are
 *     unspecified; the other functions of the batch are unaffected.  No exceptions, no printing.
 *   - There is no CPU fallback: without a CUDA device every call returns ZP_ERR_CUDA.
 */
#ifndef ZIPPEL_H
#define ZIPPEL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* host return codes */
#define ZP_OK 0
#define ZP_ERR_ARG 1       /* null pointer, size <= 0, p even / < 3 / >= 2^63, nv > ZP_MAX_NV, B > ZP_MAX_B */
#define ZP_ERR_WORKSPACE 2 /* workspace too small or misaligned */
#define ZP_ERR_CUDA 3      /* launch / configuration error, or no device */
#define ZP_ERR_SCRATCH_LIMIT 4 /* zippel_extend_skeleton_static: the batch needs more than ZP_STATIC_SCRATCH_BYTES */

/* per-function status codes (low byte of status[f]) */
#define ZP_ST_DUPLICATE_NODE 16   /* den_i == 0: two terms map to one node (G24); or m_i == 0 with s0 = 1 (G25) */
#define ZP_ST_DUPLICATE_SAMPLE 17 /* c_j == c_j' for some j' < j in Newton (index = j) */
#define ZP_ST_ZERO_PIVOT 18       /* u_{0,s} == 0 in balancing (index = s) */
#define ZP_ST_NO_RATIONAL 21       /* CRT + rational reconstruction: no a/b within Wang's bounds with gcd(a, b) = 1 */
#define ZP_ST_THIELE_DEGENERATE 20 /* Thiele: an inverse difference of level k has a zero denominator at some but
                                      not all of the remaining points (index = k); or the denominator vanished */

#define ZP_MAX_NV 32 /* skeleton variables */
#define ZP_MAX_B 64  /* sample values of x_k (D + 1) */

/* basis of the Newton output */
#define ZP_BASIS_NEWTON 0   /* a_0..a_D of eq. (1): f = a_0 + (x-c_0)[a_1 + (x-c_1)[a_2 + ...]]  (0-based, G16) */
#define ZP_BASIS_MONOMIAL 1 /* coefficients of x_k^0..x_k^D */

const char* zippel_strerror(int code);

/* Scratch needed by an entry point for a batch with these term offsets and B sample values.
 * h_offsets: host [F+1].  flags: ZP_WS_BALANCED adds the [B x T_tot] balanced-value buffer that
 * balanced_zippel_lift_step needs (pass the larger part's offsets).  Returns 0 on bad arguments. */
#define ZP_WS_BALANCED 1
size_t zippel_workspace_bytes(const int64_t* h_offsets, int F, int B, int flags);

/* (a1) Nodes, eq. (3) and L60 (G1, G2): the s-th Zippel probe is (y_1^s .. y_nv^s), so
 * skeleton term i takes the value m_i^s there, with  m_i = prod_j y_j^{e_ij} mod p.
 *   exps    [T_tot x nv] row-major uint16 exponents e_ij
 *   anchors [nv] y_j
 *   nodes   out [T_tot] m_i */
int zippel_eval_nodes(const uint16_t* exps, int64_t T_tot, int nv, const uint64_t* anchors, uint64_t p,
                      uint64_t* nodes, void* stream);

/* (a2)-(a4) Batched transposed Vandermonde solve, PAPER.md L60 and section 2.2:
 * for every function f and every right-hand side b find c with
 *     sum_i c_{b,i} m_i^(s+s0) = v_{b,s},  s = 0 .. t_f-1,
 * by the master polynomial M(z) = prod_i (z - m_i), per-node synthetic division
 * Q_i = M/(z - m_i) (Horner), c_{b,i} = (sum_s q_{i,s} v_{b,s}) / Q_i(m_i) [/ m_i if s0 = 1] (G15).
 *   nodes  [T_tot]; vals [B x T_tot]; coefs out [B x T_tot] (may alias vals: NO);
 *   s0     first power, 0 or 1 (G1);  status out [F]. */
int vandermonde_solve_batch(const uint64_t* nodes, const int64_t* h_offsets, int F, const uint64_t* vals, int B,
                            int s0, uint64_t p, uint64_t* coefs, int32_t* status, void* workspace,
                            size_t workspace_bytes, void* stream);

/* (a5) Batched Newton interpolation in x_k, eq. (1), one lane per coefficient:
 * column i of vals holds the values of coefficient i at samples c_0..c_D (row j at vals + j*ld);
 * column i of out receives its B coefficients in `basis` (row d at out + d*ld).  out may alias vals.
 * The samples are never reordered (G16).  status out [1]. */
int newton_interp_batch(const uint64_t* samples, int B, const uint64_t* vals, int64_t n, int64_t ld, uint64_t p,
                        int basis, uint64_t* out, int32_t* status, void* workspace, size_t workspace_bytes,
                        void* stream);

/* One lifting step = (a1) + (a2)-(a4) + (a5), section 1 L47-60.
 *   vals [B x T_tot] probe values f(y^(s+s0), c_j): row j, function f, entry s;
 *   out  [B x T_tot] row d = coefficient d (in `basis`) of every skeleton coefficient;
 *   nodes_out optional [T_tot] (NULL to skip).
 * status[f]: the solve's code if the solve failed, else DUPLICATE_SAMPLE for every function. */
int zippel_lift_step(const uint16_t* exps, const int64_t* h_offsets, int F, int nv, const uint64_t* anchors,
                     const uint64_t* samples, int B, int s0, const uint64_t* vals, uint64_t p, int basis,
                     uint64_t* out, uint64_t* nodes_out, int32_t* status, void* workspace, size_t workspace_bytes,
                     void* stream);

/* Host-buffer form of zippel_lift_step (the end-to-end call): every data pointer is a HOST pointer
 * (pinned memory makes the copies asynchronous).  Staging is carved from `workspace` (device,
 * zippel_host_workspace_bytes() bytes).  Batches above 8 MB of values (and at least 64 functions) are cut into 6 chunks of whole
 * functions (2, 8, 22, 22, 8, 2 sixty-fourths of the terms: small first and last, each chunk's copy hidden behind
 * its predecessor's kernels; more chunks cost more in partial waves and launches than they hide) (functions are independent): the H2D copy of chunk c+1 and the D2H copy of
 * chunk c-1 run on two copy streams of the library while the kernels of chunk c run on `stream`; the copy
 * streams start after the work already queued on `stream`, and `stream` ends waiting for the last D2H copy.
 * Nothing is synchronised: the caller waits on `stream` before reading h_out / h_status.  The two copy
 * streams and their events are created on first use per device and kept for the process (with the profiling
 * hook the only process-wide state; not thread-safe per device). */
size_t zippel_host_workspace_bytes(const int64_t* h_offsets, int F, int nv, int B);
int zippel_lift_step_host(const uint16_t* h_exps, const int64_t* h_offsets, int F, int nv,
                          const uint64_t* h_anchors, const uint64_t* h_samples, int B, int s0,
                          const uint64_t* h_vals, uint64_t p, int basis, uint64_t* h_out, int32_t* h_status,
                          void* workspace, size_t workspace_bytes, void* stream);

/* (a6) forward evaluation used by the balanced step: power sums
 *     out[b, off_f + s] = sum_i coef[b, off_f + i] * m_i^(s+s0),  s = 0 .. t_f-1
 * (the skeleton evaluated at the Zippel probe points).  coef, out: [B x T_tot]. */
int zippel_power_sums(const uint64_t* nodes, const int64_t* h_offsets, int F, const uint64_t* coef, int B, int s0,
                      uint64_t p, uint64_t* out, void* workspace, size_t workspace_bytes, void* stream);

/* One part (numerator or denominator) of a batch of F rational functions. */
typedef struct {
  const uint16_t* exps;     /* [T_tot x nv] skeleton of this part */
  const int64_t* h_offsets; /* host [F+1] */
  const uint64_t* skel;     /* [T_tot] skeleton coefficients a'_i (the reconstruction at x_k = c_0) */
  const uint64_t* uvals;    /* [B x T_tot] normalised univariate values u_{j,s}, s < t_f */
  uint64_t* out;            /* [B x T_tot] */
} zp_part;

/* (a6) Balanced lifting step for rational functions, eq. (4) (G3, G20): for the
 * numerator and the denominator separately, with R_s = sum_i a'_i m_i^(s+s0) the skeleton's value
 * at probe s,  V_{j,s} = u_{j,s} * R_s / u_{0,s};  then (a2)-(a5) on V.  samples[0] = c_0.
 * workspace must cover the larger part.  status [2F]: numerator codes, then denominator codes;
 * precedence ZERO_PIVOT, then the solve's, then DUPLICATE_SAMPLE. */
int balanced_zippel_lift_step(const zp_part* num, const zp_part* den, int F, int nv, const uint64_t* anchors,
                              const uint64_t* samples, int B, int s0, uint64_t p, int basis, int32_t* status,
                              void* workspace, size_t workspace_bytes, void* stream);

/* (f2, SURVEY.md section 8 "next") Batched univariate Thiele reconstruction, eq. (2): for every
 * column i of values f_i(x_j) at the T pairwise distinct points x_0..x_{T-1} (device, residues), the continued
 * fraction   f(x) = b_0 + (x - x_0) / (b_1 + (x - x_1) / (b_2 + ... ))   with  b_k = phi_k(x_k),
 * phi_0 = f,  phi_k(x_j) = (x_j - x_{k-1}) / (phi_{k-1}(x_j) - phi_{k-1}(x_{k-1}))  (j >= k).  The fraction ends at
 * K = k terms when ALL differences of level k vanish (the function is reproduced at the remaining points);
 * K = T otherwise.  It is then expanded to N(x) / D(x), trimmed to the true degrees and scaled so that D is
 * monic: these are the normalised univariate numerator and denominator whose values at the samples feed
 * balanced_zippel_lift_step (reading G3).  One lane per column.
 *   vals [T x n], leading dimension ld >= n, row j = values at x_j (device);  T <= ZP_MAX_B
 *   num, den [T x n] (ld): row d = coefficient of x^d, zero above the degree
 *   degs [2 x ld] int32: degs[i] = deg N (-1 for the zero function), degs[ld + i] = deg D
 *   cf   [T x n] (ld) or NULL: b_0 .. b_{K-1}, zero above K
 *   status [n]: 0, (k << 8) | ZP_ST_THIELE_DEGENERATE (outputs of that column are zero, degs -1), or
 *               (j << 8) | ZP_ST_DUPLICATE_SAMPLE for every column when x_j repeats an earlier point.
 *   workspace: zippel_workspace_bytes({0,1}, 1, T, 0) bytes. */
int thiele_reconstruct_batch(const uint64_t* points, int T, const uint64_t* vals, int64_t n, int64_t ld, uint64_t p,
                             uint64_t* num, uint64_t* den, int32_t* degs, uint64_t* cf, int32_t* status,
                             void* workspace, size_t workspace_bytes, void* stream);

/* (f1, SURVEY.md section 8 "next") Skeleton extension between two lifting steps (the polynomial in
 * k variables that one step reconstructs is the skeleton of the next).  From the monomial-in-x_k coefficients
 * coefs [B x T_tot] (the `out` of zippel_lift_step with basis = 1) the terms of the new skeleton are the pairs
 * (term i, degree d) with a non-zero coefficient, ordered by i, then d:
 *   new_exps  [cap x (nv+1)] uint16 row-major: (exps row of i, d);   new_coefs [cap]: that coefficient;
 *   new_offsets [F+1] int64 (DEVICE; copy it back to call the next step): term ranges; new_offsets[F] is the
 *   total even when it exceeds cap (then only the first cap terms are written);
 *   degs [F] int32: largest d with a non-zero coefficient in function f, -1 if none (degs[f] < B-1: fewer
 *   samples of x_k would have sufficed -- the early-termination test).
 * nv < ZP_MAX_NV.  workspace: zippel_workspace_bytes(h_offsets, F, B, 0). */
int zippel_extend_skeleton(const uint16_t* exps, const int64_t* h_offsets, int F, int nv, const uint64_t* coefs, int B,
                           uint64_t p, uint16_t* new_exps, uint64_t* new_coefs, int64_t cap, int64_t* new_offsets,
                           int32_t* degs, void* workspace, size_t workspace_bytes, void* stream);

/* The same operation for callers that may not allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc) and so have no workspace to pass: the scratch that zippel_extend_skeleton
 * takes from its workspace (the function offsets and the look-back descriptors of its one-pass scan, k_ext_fused)
 * lies in a file-scope `static __device__` array of ZP_STATIC_SCRATCH_BYTES bytes inside the library (every GPU that
 * loads the library holds it until the process exits).  Same arguments without the workspace, same results bit for
 * bit.  The call allocates nothing: no cudaMalloc / cudaFree / allocating library routine; it enqueues one copy of
 * h_offsets (read before the call returns), one memset of the descriptors and two kernels on `stream`.
 *   Limit: 256-byte-rounded 8 (F + 1) bytes of offsets + 8 (ceil(T_tot / 1024) + 1) bytes of descriptors must fit
 *   ZP_STATIC_SCRATCH_BYTES (e.g. F = 4096 functions of 10^4 terms: 0.35 MB); beyond it the call enqueues nothing and
 *   returns ZP_ERR_SCRATCH_LIMIT (zippel_strerror names the limit).
 *   The array is ONE per device and every call uses it: the call clears what must start at zero (the descriptors), but
 *   two calls that overlap on the GPU (different streams, or threads) race on it -- order them, or give the others
 *   the workspace variant above.  zippel_static_scratch_bytes() returns the limit. */
#define ZP_STATIC_SCRATCH_BYTES (1u << 20)
int zippel_extend_skeleton_static(const uint16_t* exps, const int64_t* h_offsets, int F, int nv, const uint64_t* coefs,
                                  int B, uint64_t p, uint16_t* new_exps, uint64_t* new_coefs, int64_t cap,
                                  int64_t* new_offsets, int32_t* degs, void* stream);
size_t zippel_static_scratch_bytes(void);

/* (f4, SURVEY.md section 8 "next") Second prime + CRT + rational reconstruction (the reduction runs
 * over several large primes "fitting into 2^64" and "the final reconstruction to rational numbers is performed as
 * a final step").  For every coefficient i, from its images r1[i] mod p1 and r2[i] mod p2 (device arrays; p1 != p2
 * odd primes < 2^63, e.g. 2^63 - 25 and 2^63 - 165):  x = CRT(r1, r2) in [0, m = p1 p2), then the extended Euclidean
 * sequence of (m, x) down to the first remainder <= N = floor(sqrt((m-1)/2)) gives a = remainder, b = cofactor
 * (sign moved to a, b > 0); accepted iff b <= N and gcd(|a|, b) = 1 (Wang's bounds; 2 N^2 < m makes a/b unique).
 *   num [n] int64 (signed), den [n] int64 (> 0), status [n]: 0, or ZP_ST_NO_RATIONAL with num = den = 0. */
int crt_rational_reconstruct_batch(const uint64_t* r1, const uint64_t* r2, int64_t n, uint64_t p1, uint64_t p2,
                                   int64_t* num, int64_t* den, int32_t* status, void* stream);

/* Measurement hook (bench.py's roofline leg): when kernel != 0, every later call records the CUDA event
 * `ev_start` on its stream right before the first launch of that kernel and `ev_stop` right after the
 * last one (cudaEvent_t passed as void*; the caller owns them).  kernel: ZP_K_* below in the low byte; 0
 * switches the hook off.  Bits 8.. select an occurrence: 0 = every stage of that kind re-records the
 * events (the last one wins), n >= 1 = only the n-th such stage enqueued after this call (a balanced step
 * runs every stage twice: numerator = 1, denominator = 2).  The only process-wide state in the library;
 * not thread-safe; nothing else changes. */
#define ZP_K_EVAL_NODES 1
#define ZP_K_MASTER_POLY 2
#define ZP_K_NODE_SOLVE 3
#define ZP_K_NEWTON 5
#define ZP_K_POWER_SUMS 6
#define ZP_K_BALANCE 7
#define ZP_K_LEAF_SOLVE 8 /* sub-quadratic route: k_node_solve on the leaves (B + 1 right-hand sides) */
int zippel_profile_events(int kernel, void* ev_start, void* ev_stop);
/* Number of kernels this library has enqueued in this process so far (bench.py's gpu_launches). */
unsigned long long zippel_launch_count(void);

/* Tuning knobs (process-wide; set them before sizing a workspace, not concurrently with other calls).
 *   ZP_TUNE_SUBQ_MIN_T: functions with at least this many terms (and more than 1024) take the sub-quadratic route
 *   (three-prime NTT product tree, tails, leaf solves: csrc/subq.cuh) instead of the quadratic
 *   kernels of PAPER.md section 2.2.  Same results bit for bit.  Default 0 = the measured rule:
 *   960 terms when the batch holds at least 65536 terms in such functions, else 2048 / 4096 / 8192 / 12288 terms for
 *   B >= 16 / >= 6 / >= 2 / = 1 right-hand sides (a single function is bound by the latency of the route's launches).
 *   The route needs more workspace (zippel_workspace_bytes accounts for it: about 1 KB per term and right-hand side
 *   group for the kept transforms and the tails; BASELINE.json configs[1] takes 4 GB instead of 0.3 GB). */
#define ZP_TUNE_SUBQ_MIN_T 1
int zippel_set_tuning(int key, int64_t value);

/* Destroys the copy streams and events that zippel_lift_step_host created (on every device that used it).  The
 * caller makes sure no call of the library is in flight.  A later zippel_lift_step_host creates them again. */
int zippel_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif
