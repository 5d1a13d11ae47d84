#!/usr/bin/env python
"""bench.py -- one JSON line for the driver.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input resident in HBM:
  config 2 (default; BASELINE.json configs[1], the batched 4 -> 5 variable lift: F = 4096 functions,
            t = 1000 terms, B = D+1 = 21 samples): zippel_lift_step = nodes, master polynomials,
            per-node synthetic division + 21 dot products, inversion/scaling, Newton in x_5;
  config 3 / 5: the single large skeletons (eval_nodes + vandermonde_solve_batch [+ Newton]);
  config 4: balanced_zippel_lift_step on F = 1024 rational functions.
metric = Vandermonde terms solved per second = B * T_tot / time, whole job.
N > 1 (torchrun): functions are independent, every rank lifts its own batch of the same shape (weak
scaling, no data-path collective); time = max over ranks.

--impl reference times the CPU oracle (oracle/, as it stands, single thread) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "vandermonde_terms_solved_per_s"
UNIT = "terms/s"
# Multiplier-pipe roofline (profiles/r01_baseline.md): the fma-heavy pipe issues
# 64 lanes/clk/SM of the 32-bit low multiply-add (IMAD) and 32 lanes/clk/SM of anything that needs the
# 64-bit product (IMAD.WIDE, IMAD.HI).  Unit = one lane-cycle of that pipe's 64-lane issue rate:
# IMAD = 1 unit, a 32x32->64 product = 2 units.  peak = 148 SMs x 64 units/clk x 1.965 GHz.
IMAD_PEAK_TOPS = 148 * 64 * 1.965e9 / 1e12  # planning figure; run_ours() re-derives it from the device (imad_peak)
# algorithmic cost of the method's two primitives in those units (cheapest known generic-p forms):
#   modular multiply-add x <- m x + a : 6 wide + 4 low = 16 ; deferred 64x64 MAC : 4 wide = 8
C_MM, C_MAC = 16, 8
# the instruction-count accounting of SURVEY.md 8(d).4 (10 / 4 multiplier instructions), kept as a second figure
C_MM_INSTR, C_MAC_INSTR = 10, 4


def imad_peak(device_index=0, sm_max_mhz=None):
    """T units/s = SMs (cudaDeviceProp) x 64 lanes/clk x max SM clock (nvidia-smi clocks.max.sm as sampled during the
    run, else cudaDeviceProp's clock rate)."""
    import torch

    pr = torch.cuda.get_device_properties(device_index)
    mhz = sm_max_mhz
    src = "nvidia-smi clocks.max.sm"
    if not mhz:
        khz = getattr(pr, "clock_rate", 0)
        mhz, src = (khz / 1e3, "cudaDeviceProp.clockRate") if khz else (1965.0, "B200_PROFILING.md clocks.max.sm")
    return pr.multi_processor_count * 64 * mhz * 1e6 / 1e12, f"{pr.multi_processor_count} SMs x 64 lanes/clk x {mhz:.0f} MHz ({src})"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5, 6, 7, 8, 9],
                    help="1-5: BASELINE.json configs; 6: batched Thiele reconstruction (row f2), C4's input side; "
                         "7: skeleton extension (row f1) on C2's output; 8: two-prime CRT + rational reconstruction (row f4); "
                         "9: one solve at the paper's largest skeleton, t = 4.8e6, B = 1 (PAPER.md L250; row f3)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--F", type=int, default=None, help="override the number of functions (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--subq-min-t", type=int, default=None,
                    help="override the route rule: functions with at least this many terms take the sub-quadratic route (0 = built-in rule)")
    ap.add_argument("--no-extra-legs", action="store_true",
                    help="default config only: skip the C5 and C1 legs attached to the line as \"c5\" and \"c1\"")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 <= t <= t1] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------- workloads
def load_workload(idx: int, seed_shift: int, F_override):
    from paper_2505_24256_b200 import workloads as wl

    kw = {}
    if F_override:
        kw["F"] = F_override
    if idx == 4:
        rw = wl.make_rational_workload("C4", wl.SEED_BASE + 4 + seed_shift, kw.get("F", 1024), 6, 500, 200, 24, 25)
        return rw
    sh = dict(wl.CONFIG_SHAPES[idx])
    sh.update(kw)
    return wl.make_box_workload(f"C{idx}", wl.SEED_BASE + idx + seed_shift, sh["F"], sh["nv"], sh["t"],
                                sh["emax"], sh["B"], with_planted=False)


# the sub-quadratic route (csrc/subq.cuh): constants mirrored from csrc (ZP_SQ_LEAF, ZP_SQ_KB, ZP_SQ_BATCH_T)
SQ_LEAF, SQ_KB, SQ_BATCH_T = 512, 1024, 960


def sq_threshold(ts, B):
    """csrc/zippel_capi.cu sq_threshold: functions with at least this many terms take the sub-quadratic route."""
    if sum(int(t) for t in ts if int(t) >= SQ_BATCH_T) >= 65536:
        return SQ_BATCH_T
    return 2048 if B >= 16 else 4096 if B >= 6 else 8192 if B >= 2 else 12288
C_MONT = 18  # Montgomery product: 8 wide + 2 low


def subq_units(t, B):
    """Algorithmic multiplier-pipe units of the sub-quadratic solve of ONE function of t terms with B right-hand sides,
    counted on the plan csrc/zippel_capi.cu:sq_solve executes: a length-n transform modulo one prime = (n/2) log2 n
    butterflies of one Shoup product (16 units); a pointwise product = 2 Montgomery products per prime (1 in the
    down-tree: the factor 1/n rides on the children's transforms, scaled once when the up-tree keeps them); Garner CRT
    + reduction modulo p = 5 Montgomery products per coefficient; the leaves are the quadratic node solve with B + 1
    right-hand sides.  Returns (total, parts)."""
    from math import ceil, log2

    ntt = lambda n: 3 * (n / 2) * log2(n) * C_MM  # three primes
    pw = lambda n: 3 * n * 2 * C_MONT
    pw1 = lambda n: 3 * n * C_MONT  # one Montgomery product per word and prime
    crt = lambda n: n * 5 * C_MONT
    V = B + 1
    nlev = max(0, ceil(log2(ceil(t / SQ_LEAF))))
    up = down = 0.0
    for l in range(nlev):
        a = SQ_LEAF << l
        n = 2 * a
        pairs, base = [], 0
        while base + a < t:
            pairs.append(min(a, t - base - a))
            base += 2 * a
        P = len(pairs)
        outs = sum(a + b for b in pairs)
        up += P * (3 * ntt(n) + pw(n) + 2 * pw1(n)) + crt(outs)  # both children's transforms are kept, times 2^64 / n
        down += V * (P * (3 * ntt(n) + 2 * pw1(n)) + crt(outs))  # tail x the two kept transforms
    newton = sum(1.5 * k * k * C_MAC for k in (1 << i for i in range(10)))  # schoolbook base case to x^1024
    kk = SQ_KB
    while kk < t:
        n = 2 * kk
        newton += 5 * ntt(n) + 2 * pw(n) + crt(2 * kk)
        kk <<= 1
    nr = 1 << ceil(log2(2 * t))
    root = 3 * ntt(nr) + pw(nr) + crt(t)
    leaf_t2 = sum(min(SQ_LEAF, t - x) ** 2 for x in range(0, t, SQ_LEAF))
    leaves = leaf_t2 * (C_MAC / 2 + C_MM + V * C_MAC)  # in-leaf product tree + node solve with B + 1 right-hand sides
    fin = t * (3 + B + 2) * C_MONT
    parts = {"up_tree": up, "power_sums_of_nodes (Newton inverse + root product)": newton + root, "down_tree": down,
             "leaves": leaves, "final_division": fin}
    return sum(parts.values()), parts


def work_model(ts, B, nv, newton=True, balanced=False, c_mm=C_MM, c_mac=C_MAC):
    """Algorithmic multiplier-pipe units (SURVEY.md 8(d).4 formula), total and for the node-solve kernel."""
    thr = sq_threshold(ts, B) if len(ts) else 0
    long_ts = [int(t) for t in ts if int(t) >= thr]
    if long_ts:  # sub-quadratic route for the long functions, the quadratic formula for the rest
        short = [int(t) for t in ts if int(t) < thr]
        tot_s, ns_s = work_model(short, B, nv, newton, balanced, c_mm, c_mac) if short else (0.0, 0.0)
        T = float(sum(long_ts))
        sq = sum(subq_units(t, B)[0] for t in long_ts)
        total = sq + c_mm * (nv - 1) * T + (c_mm * T * B * (B - 1) / 2 if newton else 0.0)
        if balanced:
            total += c_mac * float(sum(t * t for t in long_ts))
        return tot_s + total, ns_s + sq
    t2 = float(sum(int(t) * int(t) for t in ts))
    T = float(sum(int(t) for t in ts))
    # per (node, stage): one modular multiply-add (the quotient), B deferred MACs, one more MAC for the denominator
    # (k_node_den evaluates M'(m_i) by deferred MACs)
    node_solve = t2 * (c_mm + (B + 1) * c_mac)
    if B == 1 and min(int(t) for t in ts) >= 4096:  # one right-hand side: W = corr(v, M), then W(m_i) and M'(m_i)
        node_solve = t2 * (2 * c_mac + c_mac / 2)  # two polynomial evaluations by deferred MACs + the correlation
    total = node_solve + c_mac * t2 / 2 + c_mm * ((nv - 1) * T + (3 + B) * T)
    if newton:
        total += c_mm * T * B * (B - 1) / 2
    if balanced:
        total += c_mac * t2  # forward evaluation: one deferred MAC per (probe, node) with the strided power tables
    return total, node_solve


# ---------------------------------------------------------------------------------------- ours
def run_leg(idx, K, W, F_override, want_e2e, rank, world, local, sample_clocks=True, latency_leg=False):
    """One configuration: W warm-up steps, K timed steps on resident inputs, then (optionally) the same through the
    host-buffer entry.  Returns the fields of the JSON line (every rank returns; ms is the max over ranks)."""
    import torch

    from paper_2505_24256_b200 import api, sharding

    w = load_workload(idx, sharding.rank_seed_shift(rank), F_override)
    stream = torch.cuda.Stream()
    latency_leg = latency_leg or (idx == 1 and not F_override)  # the one-launch small case: see the timed loop

    # ---- resident inputs and the step closure --------------------------------------------------
    if idx == 4:
        parts = [w.num, w.den]
        B, nv, F = w.num.B, w.num.nv, w.num.F
        ts = [500] * F + [200] * F
        dev = []
        for q in parts:
            dev.append(dict(exps=api.to_dev(q.exps), offsets=q.offsets, skel=api.to_dev(q.meta["skel_standin"]),
                            uvals=api.to_dev(q.vals), out=torch.empty(q.vals.shape, dtype=torch.int64, device="cuda")))
        anchors, samples = api.to_dev(w.num.anchors), api.to_dev(w.num.samples)
        ws = api.alloc_workspace(w.num.offsets, B, api.WS_BALANCED)
        status = torch.empty(2 * F, dtype=torch.int32, device="cuda")
        T_tot = w.num.T_tot + w.den.T_tot
        p = w.num.p

        def step():
            api.balanced_zippel_lift_step(dev[0], dev[1], anchors, samples, p, 0, 1, status=status, workspace=ws,
                                          stream=stream)
        total_ops, _ = work_model(ts, B, nv, True, True)
        _, ns_ops = work_model([500] * F, B, nv, True, True)  # the hook times the numerator part's node solve
        ns_ts = [500] * F
        workload = f"C4 balanced lift 5->6 vars: F={F} rational functions, t_N=500, t_D=200, B=25"
        in_bytes = sum(q.exps.nbytes + q.vals.nbytes + q.meta["skel_standin"].nbytes for q in parts)
        out_bytes = sum(q.vals.nbytes for q in parts)
    else:
        B, nv, F, T_tot, p = w.B, w.nv, w.F, w.T_tot, w.p
        ts = np.diff(w.offsets)
        exps, anchors, samples, vals = (api.to_dev(x) for x in (w.exps, w.anchors, w.samples, w.vals))
        out = torch.empty_like(vals)
        status = torch.empty(F, dtype=torch.int32, device="cuda")
        ws = api.alloc_workspace(w.offsets, B)
        newton = idx not in (5, 9)
        if newton:
            def step():
                api.zippel_lift_step(exps, w.offsets, anchors, samples, vals, p, 0, 1, out=out, status=status,
                                     workspace=ws, stream=stream)
        else:
            nodes = torch.empty(T_tot, dtype=torch.int64, device="cuda")

            def step():
                api.zippel_eval_nodes(exps, anchors, p, out=nodes, stream=stream)
                api.vandermonde_solve_batch(nodes, w.offsets, vals, p, 0, out=out, status=status, workspace=ws,
                                            stream=stream)
        total_ops, ns_ops = work_model(ts, B, nv, newton, False)
        ns_ts = ts
        workload = (f"C{idx} {'lift' if newton else 'solve'}: F={F}, t={int(ts.max())}, nv={nv}, B={B}"
                    + (" (BASELINE.json configs[1])" if idx == 2 and not F_override else "")
                    + (" (PAPER.md L250: the largest skeleton, 4.8m monomials)" if idx == 9 else ""))
        in_bytes = w.exps.nbytes + w.vals.nbytes + w.anchors.nbytes + w.samples.nbytes
        out_bytes = w.vals.nbytes + 4 * F
    subq = int(max(ts)) >= sq_threshold(ts, B)

    def barrier():
        if world > 1:
            import torch.distributed as dist

            dist.barrier()

    # ---- warm-up, then K timed steps (device-resident) ----------------------------------------
    with torch.cuda.stream(stream):
        for _ in range(W):
            step()
        torch.cuda.synchronize()
        st_host = status.cpu().numpy()
        assert not st_host.any(), f"data-dependent failure in the synthetic batch: {st_host[st_host != 0][:4]}"
        ev_k = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        for a, b in ev_k:
            a.record(stream); b.record(stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(local) if (rank == 0 and sample_clocks) else None
        time.sleep(0.3 if sampler else 0.0)
        barrier()
        torch.cuda.synchronize()
        n0 = api.zippel_launch_count()
        t0 = time.perf_counter()
        e0.record(stream)
        for i in range(K):
            # the event hook times one kind of scope per step: the node solve (quadratic route) or the whole
            # sub-quadratic route on even steps, the leaf solve of the sub-quadratic route on odd steps
            kind = api.K_LEAF_SOLVE if (subq and i % 2 == 1) else api.K_NODE_SOLVE
            if not latency_leg:
                api.zippel_profile_events(kind | (1 << 8), ev_k[i][0], ev_k[i][1])  # 1st occurrence in the step
            step()
        e1.record(stream)
        torch.cuda.synchronize()
        barrier()
        t1 = time.perf_counter()
        launches = api.zippel_launch_count() - n0
        if latency_leg:
            # a step of tens of microseconds: the hook's two event records between consecutive launches and its host
            # call are a tenth of it, so the K timed steps above ran without it and the kernel's own time comes from
            # K more steps with it (outside the timed region)
            for i in range(K):
                api.zippel_profile_events(api.K_NODE_SOLVE | (1 << 8), ev_k[i][0], ev_k[i][1])
                step()
            torch.cuda.synchronize()
        api.zippel_profile_events(0)
        clocks = sampler.stop(t0, t1) if sampler else None
        ms = e0.elapsed_time(e1)
        if subq and K >= 2:
            ns_ms = sum(ev_k[i][0].elapsed_time(ev_k[i][1]) for i in range(0, K, 2)) / len(range(0, K, 2))
            leaf_ms = sum(ev_k[i][0].elapsed_time(ev_k[i][1]) for i in range(1, K, 2)) / len(range(1, K, 2))
        else:
            ns_ms = sum(a.elapsed_time(b) for a, b in ev_k) / K
            leaf_ms = None
    ms = sharding.max_over_ranks(ms, "cuda")
    ms_per_step = ms / K
    terms = B * T_tot * world
    value = terms / (ms_per_step * 1e-3)

    # ---- e2e: host (pinned) buffers through the host-buffer C-ABI call ---------------------------
    e2e = None
    if want_e2e and idx not in (4, 5, 9):
        pin = lambda a: torch.from_numpy(a.view(np.int64) if a.dtype == np.uint64 else a.view(np.int16)).pin_memory()
        h_exps, h_anch, h_samp, h_vals = pin(w.exps), pin(w.anchors), pin(w.samples), pin(w.vals)
        h_out = torch.empty(w.vals.shape, dtype=torch.int64).pin_memory()
        h_st = torch.empty(F, dtype=torch.int32).pin_memory()
        hws = torch.empty(api.host_workspace_bytes(w.offsets, nv, B), dtype=torch.uint8, device="cuda")

        def estep():
            api.zippel_lift_step_host(h_exps, w.offsets, h_anch, h_samp, h_vals, p, h_out, h_st, hws, 0, 1, stream=stream)
            stream.synchronize()  # the user reads the result of every step

        for _ in range(max(1, min(W, 2))):
            estep()
        barrier()
        torch.cuda.synchronize()
        ta = time.perf_counter()
        for _ in range(K):
            estep()
        torch.cuda.synchronize()
        tb = time.perf_counter()
        ems = (tb - ta) * 1e3
        ems = sharding.max_over_ranks(ems, "cuda")
        assert not h_st.numpy().any()
        e2e = {"value": terms / (ems / K * 1e-3), "unit": UNIT, "ms_per_step": ems / K,
               "h2d_bytes_per_step": int(in_bytes), "d2h_bytes_per_step": int(out_bytes),
               "call": "zippel_lift_step_host (pinned host buffers; chunked H2D / step / D2H pipeline on 3 streams + stream sync per step)"}

    peak, peak_how = imad_peak(local, clocks.get("sm_max_mhz") if clocks else None)
    achieved = ns_ops / (ns_ms * 1e-3) / 1e12
    ns_ops_instr = float(sum(int(t) ** 2 for t in ns_ts)) * (2 * C_MM_INSTR + B * C_MAC_INSTR)  # SURVEY.md 8(d).4 accounting
    if subq:
        kernel = "sub-quadratic solve (csrc/subq.cuh): leaf trees, up-tree, Newton chain, tails down the tree (k_ntt_mul, k_ntt_pass, CRT), leaf k_node_solve, k_inv_finish"
        cost = ("W_alg of the sub-quadratic route (bench.py subq_units, DESIGN.md section 12): butterfly = one Shoup product = 16 units, "
                "pointwise = 2 Montgomery products (36; 1 in the down-tree, the kept transforms carry 1/n), CRT + reduction = 5 (90), leaves = quadratic node solve with B + 1 right-hand sides")
    elif idx == 5 or (B == 1 and int(min(ts)) >= 4096):
        kernel, cost = "k_corr_w + k_node_eval2", "per (node, stage) 8 (2 + 1/2) units: two evaluations by deferred MACs + the correlation"
    else:
        kernel = "k_node_den + k_node_solve" + (" (numerator part)" if idx == 4 else "")
        cost = "modular multiply-add = 16 units (6 wide + 4 low), deferred 64x64 MAC = 8 units (4 wide); per (node, stage) 16 + 8 (B + 1)"
    quad_equiv = float(sum(int(t) ** 2 for t in ts)) * (C_MM + (B + 1) * C_MAC + C_MAC / 2)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u64", "data": "synthetic",
        "config": {"workload": workload, "p": "2^63-25", "basis": "monomial", "functions_per_gpu": int(F),
                   "terms_per_gpu": int(T_tot), "l2": "inputs larger than L2 (688 MB of values per step)" if idx == 2
                   else "inputs smaller than L2; compute-bound kernels (see DESIGN.md)", "parallelism": f"dp{world}",
                   "route": "sub-quadratic (three-prime NTT product tree)" if subq else "quadratic (PAPER.md section 2.2)"},
        "lift_steps_per_s": F * world / (ms_per_step * 1e-3),
        "credited_modmuls_per_s": B * float(sum(int(t) ** 2 for t in ts)) * world / (ms_per_step * 1e-3),
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {
            "bound": "alu", "kernel": kernel, "achieved": achieved, "peak": peak,
            "unit": "T multiplier-pipe units/s (IMAD = 1, 32x32->64 product = 2)", "frac": achieved / peak,
            # dram__bytes_read.sum + dram__bytes_write.sum of the k_node_solve<21> launch from an ncu --set full capture of
            # the same command; algorithmic 1540 MB.  Only known for the default config; not measured in this run.
            "traffic": 1555.9e6 if (idx == 2 and not F_override) else None,
            "traffic_source": "ncu --set full capture of the same command (profiles/r02_final.md: k_node_solve<21> 895.5 MB read + 660.4 MB "
                              "written), not this run" if (idx == 2 and not F_override) else None,
            "peak_source": "derived (DESIGN.md 5.1): " + peak_how + "; profiles/r01_baseline.md measures IMAD at 63.5 and "
                           "IMAD.WIDE at 31.8 lanes/clk/SM",
            "frac_is": "multiplier-pipe utilisation of the formulation built (the algorithmic operation count in pipe units)",
            "algorithmic_ops_per_launch": ns_ops, "ms_per_launch": ns_ms,
            "algorithmic_cost": cost,
            "whole_step_frac": total_ops / (ms_per_step * 1e-3) / 1e12 / peak,
        },
        "e2e": e2e,
    }
    if subq:
        line["roofline"]["speedup_vs_quadratic_work"] = quad_equiv / total_ops
        line["roofline"]["quadratic_equivalent_frac"] = quad_equiv / (ms_per_step * 1e-3) / 1e12 / peak
        if leaf_ms:
            thr = sq_threshold(ts, B)
            leaf_t2 = float(sum(min(SQ_LEAF, int(t) - x) ** 2 for t in ts if int(t) >= thr for x in range(0, int(t), SQ_LEAF)))
            leaf_ops = leaf_t2 * (C_MM + (B + 1) * C_MAC)
            leaf = {"kernel": f"k_node_solve<{B + 1 if B + 1 <= 25 else 'passes'}> on the {SQ_LEAF}-node leaves (B + 1 right-hand sides)",
                    "ms_per_launch": leaf_ms, "algorithmic_ops_per_launch": leaf_ops, "achieved": leaf_ops / (leaf_ms * 1e-3) / 1e12,
                    "frac": leaf_ops / (leaf_ms * 1e-3) / 1e12 / peak, "share_of_step": leaf_ms / ms_per_step}
            if leaf["share_of_step"] >= 0.5:
                # one kernel holds most of the step: it is the dominant kernel, the route-level figures move aside
                r = line["roofline"]
                r["route"] = {"kernel": r["kernel"], "achieved": r["achieved"], "frac": r["frac"], "ms": r["ms_per_launch"],
                              "algorithmic_ops": r["algorithmic_ops_per_launch"], "algorithmic_cost": r["algorithmic_cost"]}
                r.update(kernel=leaf["kernel"], achieved=leaf["achieved"], frac=leaf["frac"], ms_per_launch=leaf_ms,
                         algorithmic_ops_per_launch=leaf_ops, share_of_step=leaf["share_of_step"],
                         algorithmic_cost="modular multiply-add = 16 units, deferred 64x64 MAC = 8 units; per (node, stage) of a leaf 16 + 8 (B + 1)")
                if idx == 2 and not F_override:
                    # DRAM bytes of this launch from the ncu --set full capture of the same command; algorithmic: the B + 1
                    # tails read and the B + 1 numerator rows written once, 8 (B + 1) T_tot bytes each way (1442 MB)
                    r["traffic"] = 1615.0e6
                    r["traffic_source"] = ("ncu --set full capture of the same command (profiles/r02_final.md: k_node_solve<22> "
                                           "924.0 MB read + 691.0 MB written), not this run")
            else:
                line["roofline"]["leaf_solve"] = leaf
    else:
        line["roofline"]["frac_instr_count_10_4"] = ns_ops_instr / (ns_ms * 1e-3) / 1e12 / peak
    return line


def run_ours(args):
    import torch

    from paper_2505_24256_b200 import api

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist

        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    api.lib()
    if args.subq_min_t is not None:
        api.zippel_set_tuning(api.TUNE_SUBQ_MIN_T, args.subq_min_t)
    idx = args.config
    line = run_leg(idx, args.steps, args.warmup, args.F, not args.no_e2e, rank, world, local)
    # the default line carries the other half of north_star's target (the t = 2^19 solve, configs[4]) and the latency
    # of the small case (configs[0]) as sub-objects; every rank runs them (the barriers inside match), rank 0 prints
    if idx == 2 and not args.F and not args.no_extra_legs:
        c5 = run_leg(5, 10, 3, None, False, rank, world, local)
        line["c5"] = {k: c5[k] for k in ("value", "unit", "ms_per_step", "steps", "warmup", "gpu_launches", "clocks", "roofline")}
        line["c5"]["workload"] = c5["config"]["workload"] + "; " + c5["config"]["route"]
        c1 = run_leg(1, 200, 10, None, True, rank, world, local, latency_leg=True)
        line["c1"] = {"workload": c1["config"]["workload"], "us_per_step": c1["ms_per_step"] * 1e3, "steps": 200, "warmup": 10,
                      "kernel_us": c1["roofline"]["ms_per_launch"] * 1e3,
                      "note": "one fused launch (csrc/small.cuh); us_per_step: 200 back-to-back steps between two CUDA events, no hook; "
                              "kernel_us: the launch between the C-ABI hook's two events, from 200 more steps outside the timed ones",
                      "launches_per_step": c1["gpu_launches"] / 200, "e2e_us_per_step": c1["e2e"]["ms_per_step"] * 1e3,
                      "lift_steps_per_s": c1["lift_steps_per_s"], "clocks": c1["clocks"]}
    if rank != 0:
        if world > 1:
            import torch.distributed as dist

            dist.destroy_process_group()
        return
    # ---- CPU baseline: the oracle on a bounded sample (rank 0, N = 1 only) -------------------------
    line["cpu_baseline"] = oracle_sample(idx, steps=1, all_cores=True) if (world == 1 and not args.no_cpu_baseline) else None
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------- oracle legs
SAMPLE = {1: dict(), 2: dict(F=32), 3: dict(t=6000), 4: dict(F=24), 5: dict(t=1 << 14), 9: dict(t=1 << 14)}


def oracle_step(idx, w):
    from oracle import ref

    if idx == 4:
        parts = {n: dict(exps=q.exps, offsets=q.offsets, skel=q.meta["skel_standin"], uvals=q.vals)
                 for n, q in (("num", w.num), ("den", w.den))}
        ref.balanced_zippel_lift_step(parts["num"], parts["den"], w.num.anchors, w.num.samples, w.num.p, 0, 1)
        return w.num.B * (w.num.T_tot + w.den.T_tot), w.num.F
    if idx in (5, 9):
        nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
        ref.vandermonde_solve_batch(nodes, w.offsets, w.vals, w.p, 0)
    else:
        ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, w.vals, w.p, 0, 1)
    return w.B * w.T_tot, w.F


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_all_cores(idx):
    """The oracle on all the host cores this process may use: the unmodified single-threaded
    routines on independent units from one thread each (ctypes releases the GIL during a call) -- functions for C2 / C4,
    node ranges after one shared master-polynomial build for the single skeletons.  Returns (terms/s at the sample's t,
    cores, seconds, description)."""
    from concurrent.futures import ThreadPoolExecutor

    from oracle import ref
    from paper_2505_24256_b200 import workloads as wl

    cores = host_cores()
    if idx in (2, 4):
        per = 8 if idx == 2 else 6
        F = cores * per
        w = wl.config(idx, F=F)

        def unit(c):
            f0, f1 = c * per, (c + 1) * per
            if idx == 4:
                parts = {}
                for n, q in (("num", w.num), ("den", w.den)):
                    a, b = int(q.offsets[f0]), int(q.offsets[f1])
                    parts[n] = dict(exps=np.ascontiguousarray(q.exps[a:b]), offsets=(q.offsets[f0:f1 + 1] - a).copy(),
                                    skel=np.ascontiguousarray(q.meta["skel_standin"][a:b]), uvals=np.ascontiguousarray(q.vals[:, a:b]))
                ref.balanced_zippel_lift_step(parts["num"], parts["den"], w.num.anchors, w.num.samples, w.num.p, 0, 1)
            else:
                a, b = int(w.offsets[f0]), int(w.offsets[f1])
                ref.zippel_lift_step(np.ascontiguousarray(w.exps[a:b]), (w.offsets[f0:f1 + 1] - a).copy(), w.anchors, w.samples,
                                     np.ascontiguousarray(w.vals[:, a:b]), w.p, 0, 1)

        terms = (w.num.B * (w.num.T_tot + w.den.T_tot)) if idx == 4 else w.B * w.T_tot
        with ThreadPoolExecutor(cores) as ex:
            ta = time.perf_counter()
            list(ex.map(unit, range(cores)))
            dt = time.perf_counter() - ta
        return terms / dt, cores, dt, f"{F} functions, {per} per thread, {cores} threads"
    w = wl.config(idx, **SAMPLE[idx])
    t = w.T_tot
    with ThreadPoolExecutor(cores) as ex:
        ta = time.perf_counter()
        nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
        M = ref.master_poly(nodes, w.p)  # shared, single thread (t^2 / 2 of the (2 + B) t^2 products)
        cuts = [t * c // cores for c in range(cores + 1)]
        list(ex.map(lambda c: ref.node_solve_at(nodes[cuts[c]:cuts[c + 1]], M, w.vals, w.p), range(cores)))
        dt = time.perf_counter() - ta
    return w.B * t / dt, cores, dt, (f"{t}-term prefix: nodes and master polynomial on one thread, then the per-node routine "
                                     f"(PAPER.md L193-195) on {cores} node ranges; the O(t) division and Newton are left out")


def oracle_sample(idx, steps=1, warmup=0, all_cores=False):
    """Time the oracle, as it stands (single thread, unsigned __int128 mulmod), on a bounded sample of the
    bench workload.  The metric is terms/s AT THE SAMPLE'S t; for configs 3 and 5 the sample has a shorter
    skeleton, so the value is also given scaled by (t_sample / t_full) (cost per term is linear in t)."""
    from oracle import ref
    from paper_2505_24256_b200 import workloads as wl

    ref.lib()
    w = wl.config(idx, **SAMPLE[idx])
    for _ in range(warmup):
        oracle_step(idx, w)
    ta = time.perf_counter()
    for _ in range(steps):
        terms, F = oracle_step(idx, w)
    dt = (time.perf_counter() - ta) / steps
    full_t = wl.CONFIG_SHAPES[idx].get("t")
    samp_t = SAMPLE[idx].get("t")
    scale = (samp_t / full_t) if (samp_t and full_t) else 1.0
    desc = {2: "first 32 of the 4096 functions (same t = 1000, B = 21)", 4: "first 24 of the 1024 functions",
            3: "6000-term prefix as a complete problem, value scaled by 6000/100000",
            5: "2^14-term prefix as a complete problem (BASELINE.json), value scaled by 2^14/2^19",
            9: "2^14-term prefix as a complete problem, value scaled by 2^14/4.8e6",
            1: "the whole config"}[idx]
    out = {"value": terms / dt * scale, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
           "seconds_per_sample_step": dt, "lift_steps_per_s": F / dt * (scale * scale if scale != 1.0 else 1.0)}
    if all_cores and idx != 1:
        v, cores, secs, how = oracle_all_cores(idx)
        out["all_cores"] = {"value": v * scale, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": how,
                            "seconds": secs, "speedup_over_one_core": v * scale / out["value"]}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cpu = oracle_sample(args.config, steps=args.steps, warmup=min(args.warmup, 1))
    line = {
        "impl": "reference", "metric": METRIC, "value": cpu["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": cpu["seconds_per_sample_step"] * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": f"C{args.config} via the CPU oracle; each step = {cpu['sample']}", "p": "2^63-25"},
        "cpu_baseline": cpu,
        "e2e": {"value": cpu["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------- (f2) Thiele leg
def thiele_inputs(n, T, seed):
    """Arbitrary residues as values (every column runs the full T levels: the cost model's case) at T distinct
    points; shaped like C4's input side: 1024 functions x 500 probes, degree <= 24 in x_6 -> T = 50 points."""
    from paper_2505_24256_b200 import workloads as wl

    pts = wl.distinct_residues(wl._rng(seed, 40), 2, wl.P63, T)
    vals = wl.uniform_residues(wl._rng(seed, 41), 0, wl.P63, (T, n))
    return pts, vals, wl.P63


def run_thiele(args):
    import torch

    from paper_2505_24256_b200 import api, workloads as wl

    T, n = 50, (args.F or 1024) * 500
    K, W = args.steps, args.warmup
    if args.impl == "reference":
        from oracle import ref

        pts, vals, p = thiele_inputs(4000, T, wl.SEED_BASE + 6)
        ta = time.perf_counter()
        for _ in range(K):
            ref.thiele_reconstruct_batch(pts, vals, p)
        dt = (time.perf_counter() - ta) / K
        cpu = {"value": 4000 / dt, "unit": "reconstructions/s", "cores": 1, "kind": "oracle", "sample": "4000 columns, T = 50"}
        print(json.dumps({"impl": "reference", "metric": "thiele_reconstructions_per_s", "value": 4000 / dt,
                          "unit": "reconstructions/s", "n_gpus": 1, "steps": K, "warmup": 0, "ms_per_step": dt * 1e3,
                          "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
                          "config": {"workload": "Thiele via the CPU oracle; each step = 4000 columns, T = 50"},
                          "cpu_baseline": cpu, "gpu_launches": 0,
                          "e2e": {"value": 4000 / dt, "unit": "reconstructions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return
    torch.cuda.set_device(0)
    api.lib()
    pts, vals, p = thiele_inputs(n, T, wl.SEED_BASE + 6)
    dp, dv = api.to_dev(pts), api.to_dev(vals)
    ws = api.alloc_workspace([0, 1], T)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        for _ in range(W):
            out = api.thiele_reconstruct_batch(dp, dv, p, want_cf=False, workspace=ws, stream=stream)
        torch.cuda.synchronize()
        assert not api.to_host(out[4]).any()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(0)
        time.sleep(0.3)
        n0, t0 = api.zippel_launch_count(), time.perf_counter()
        e0.record(stream)
        for _ in range(K):
            api.thiele_reconstruct_batch(dp, dv, p, want_cf=False, workspace=ws, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        ms = e0.elapsed_time(e1) / K
    clocks = sampler.stop(t0, t1)
    # algorithmic products per column, fraction form.  Shoup products (fixed multiplier, 16 units):
    # 4 per point and level (2T^2 - 2T) and the expansion (T^2/2 + 2T).  Montgomery products (18 units): the companions of
    # the two pivots per level and of b_k per expansion step (3T), one batched inversion of the b_k (4T + 93), the monic
    # scaling (T + 94).
    units = n * (16.0 * (2.5 * T * T) + 18.0 * (8 * T + 187))
    achieved = units / (ms * 1e-3) / 1e12
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import ref

        cp, cv, _ = thiele_inputs(4000, T, wl.SEED_BASE + 6)
        ta = time.perf_counter()
        ref.thiele_reconstruct_batch(cp, cv, p)
        dt = time.perf_counter() - ta
        cpu = {"value": 4000 / dt, "unit": "reconstructions/s", "cores": 1, "kind": "oracle", "sample": "4000 columns, T = 50"}
    print(json.dumps({
        "metric": "thiele_reconstructions_per_s", "value": n / (ms * 1e-3), "unit": "reconstructions/s", "n_gpus": 1,
        "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u64", "data": "synthetic",
        "config": {"workload": f"Thiele batch: n={n} columns (1024 functions x 500 probes), T={T} points, p=2^63-25",
                   "l2": "inputs larger than L2 (205 MB of values per step)"},
        "gpu_launches": int(api.zippel_launch_count() - n0), "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "k_thiele", "achieved": achieved, "peak": IMAD_PEAK_TOPS,
                     "unit": "T multiplier-pipe units/s (IMAD = 1, 32x32->64 product = 2)", "frac": achieved / IMAD_PEAK_TOPS,
                     "traffic": None, "algorithmic_ops_per_launch": units, "ms_per_launch": ms,
                     "algorithmic_cost": "2.5 T^2 Shoup products of 16 units + (8 T + 187) Montgomery products of 18 units per column"},
        "e2e": None, "cpu_baseline": cpu}))


# ---------------------------------------------------------------------------------------- (f1) extension leg
def run_extend(args):
    """zippel_extend_skeleton on the output shape of C2 (4096 functions x 1000 terms, B = 21, the sparse law's one
    non-zero degree per term): HBM-bound stream compaction, reported against the measured copy bandwidth."""
    import torch

    from paper_2505_24256_b200 import api, workloads as wl

    K, W = args.steps, args.warmup
    sh = dict(wl.CONFIG_SHAPES[2])
    F = args.F or (64 if args.impl == "reference" else sh["F"])
    w = wl.make_box_workload("C2out", wl.SEED_BASE + 2, F, sh["nv"], sh["t"], sh["emax"], sh["B"], with_vals=False)
    T_tot, B, nv = w.T_tot, w.B, w.nv
    if args.impl == "reference":
        from oracle import ref

        ta = time.perf_counter()
        for _ in range(K):
            ref.extend_skeleton(w.exps, w.offsets, w.planted, w.p)
        dt = (time.perf_counter() - ta) / K
        cpu = {"value": T_tot / dt, "unit": "terms/s", "cores": 1, "kind": "oracle", "sample": f"{F} functions of C2's shape"}
        print(json.dumps({"impl": "reference", "metric": "skeleton_terms_extended_per_s", "value": T_tot / dt, "unit": "terms/s",
                          "n_gpus": 1, "steps": K, "warmup": 0, "ms_per_step": dt * 1e3, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
                          "config": {"workload": f"skeleton extension via the CPU oracle, {F} functions"}, "cpu_baseline": cpu,
                          "gpu_launches": 0, "e2e": {"value": T_tot / dt, "unit": "terms/s", "h2d_bytes_per_step": 0,
                                                     "d2h_bytes_per_step": 0}}))
        return
    torch.cuda.set_device(0)
    api.lib()
    de, dc = api.to_dev(w.exps), api.to_dev(w.planted)
    ws = api.alloc_workspace(w.offsets, B)
    stream = torch.cuda.Stream()
    cap = T_tot  # one non-zero degree per term
    with torch.cuda.stream(stream):
        for _ in range(W):
            ne, nc, no, dg = api.zippel_extend_skeleton(de, w.offsets, dc, w.p, cap, workspace=ws, stream=stream)
        torch.cuda.synchronize()
        assert int(no.cpu()[-1]) == T_tot
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(0)
        time.sleep(0.3)
        n0, t0 = api.zippel_launch_count(), time.perf_counter()
        e0.record(stream)
        for _ in range(K):
            api.zippel_extend_skeleton(de, w.offsets, dc, w.p, cap, workspace=ws, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        ms = e0.elapsed_time(e1) / K
    clocks = sampler.stop(t0, t1)
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    peak = float(peaks.get("hbm_gbs", 6650.0))
    # algorithmic bytes: the coefficient matrix and the exponent rows in, the new rows and coefficients out
    alg = 8.0 * B * T_tot + 2.0 * nv * T_tot + (2.0 * (nv + 1) + 8.0) * T_tot + 8.0 * (F + 1) + 4.0 * F
    achieved = alg / (ms * 1e-3) / 1e9
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import ref

        ws_ = wl.make_box_workload("C2out", wl.SEED_BASE + 2, 64, sh["nv"], sh["t"], sh["emax"], sh["B"], with_vals=False)
        ta = time.perf_counter()
        ref.extend_skeleton(ws_.exps, ws_.offsets, ws_.planted, ws_.p)
        dt = time.perf_counter() - ta
        cpu = {"value": ws_.T_tot / dt, "unit": "terms/s", "cores": 1, "kind": "oracle", "sample": "first 64 functions"}
    print(json.dumps({
        "metric": "skeleton_terms_extended_per_s", "value": T_tot / (ms * 1e-3), "unit": "terms/s", "n_gpus": 1, "steps": K,
        "warmup": W, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64",
        "data": "synthetic",
        "config": {"workload": f"skeleton extension on C2's output: F={F}, t=1000, nv={nv}, B={B}, one non-zero degree per term",
                   "l2": "inputs larger than L2 (688 MB of coefficients per step)"},
        "gpu_launches": int(api.zippel_launch_count() - n0), "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "k_ext_count + k_ext_emit", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": None, "algorithmic_bytes_per_launch": alg, "ms_per_launch": ms,
                     "peak_source": "MEASURED_PEAKS.json hbm_gbs (measured copy bandwidth)" if peaks else "fallback 6650 GB/s"},
        "e2e": None, "cpu_baseline": cpu}))


# ---------------------------------------------------------------------------------------- (f4) CRT leg
def run_crt(args):
    """crt_rational_reconstruct_batch on as many coefficients as C2 reconstructs (4 096 000), images of random
    fractions a/b with |a|, b < 2^40 (two primes determine them with room to spare)."""
    import torch

    from paper_2505_24256_b200 import api, workloads as wl

    K, W = args.steps, args.warmup
    p1, p2 = wl.P63, (1 << 63) - 165
    n = 4000 if args.impl == "reference" else (args.F or 4096) * 1000
    rng = wl._rng(wl.SEED_BASE + 8, 50)
    a = rng.integers(-(1 << 40), 1 << 40, n, dtype=np.int64)
    bb = rng.integers(1, 1 << 40, n, dtype=np.int64)
    # images mod p by float-free vectorised arithmetic is awkward in numpy; build them from a table of 4096 fractions
    tab = [(int(x), int(y)) for x, y in zip(a[:4096], bb[:4096])]
    t1 = np.array([x * pow(y, -1, p1) % p1 for x, y in tab], dtype=np.uint64)
    t2 = np.array([x * pow(y, -1, p2) % p2 for x, y in tab], dtype=np.uint64)
    idx = rng.integers(0, len(tab), n)
    r1, r2 = t1[idx], t2[idx]
    if args.impl == "reference":
        from oracle import ref

        ta = time.perf_counter()
        for _ in range(K):
            ref.crt_rational_batch(r1, r2, p1, p2)
        dt = (time.perf_counter() - ta) / K
        cpu = {"value": n / dt, "unit": "reconstructions/s", "cores": 1, "kind": "oracle", "sample": f"{n} coefficients"}
        print(json.dumps({"impl": "reference", "metric": "rational_reconstructions_per_s", "value": n / dt,
                          "unit": "reconstructions/s", "n_gpus": 1, "steps": K, "warmup": 0, "ms_per_step": dt * 1e3,
                          "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u128", "data": "synthetic",
                          "config": {"workload": f"CRT + rational reconstruction via the CPU oracle, {n} coefficients"},
                          "cpu_baseline": cpu, "gpu_launches": 0,
                          "e2e": {"value": n / dt, "unit": "reconstructions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return
    torch.cuda.set_device(0)
    api.lib()
    d1, d2 = api.to_dev(r1), api.to_dev(r2)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        for _ in range(W):
            num, den, st = api.crt_rational_reconstruct_batch(d1, d2, p1, p2, stream=stream)
        torch.cuda.synchronize()
        assert not st.any().item()
        hn, hd = num[:1000].cpu().numpy(), den[:1000].cpu().numpy()
        assert all(int(x) * tab[j][1] == tab[j][0] * int(y) for x, y, j in zip(hn, hd, idx[:1000]))  # same fraction
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(0)
        time.sleep(0.3)
        n0, t0 = api.zippel_launch_count(), time.perf_counter()
        e0.record(stream)
        for _ in range(K):
            api.crt_rational_reconstruct_batch(d1, d2, p1, p2, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        t1_ = time.perf_counter()
        ms = e0.elapsed_time(e1) / K
    clocks = sampler.stop(t0, t1_)
    # algorithmic work: about 0.843 ln(sqrt(m)) = 37 Euclid steps per coefficient, each at least
    # two 64 x 64 -> 128 products (q r and q t): 16 units
    units = n * 37.0 * 16.0
    achieved = units / (ms * 1e-3) / 1e12
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import ref

        ta = time.perf_counter()
        ref.crt_rational_batch(r1[:200000], r2[:200000], p1, p2)
        dt = time.perf_counter() - ta
        cpu = {"value": 200000 / dt, "unit": "reconstructions/s", "cores": 1, "kind": "oracle", "sample": "first 200 000 coefficients"}
    print(json.dumps({
        "metric": "rational_reconstructions_per_s", "value": n / (ms * 1e-3), "unit": "reconstructions/s", "n_gpus": 1,
        "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u128", "data": "synthetic",
        "config": {"workload": f"two-prime CRT + rational reconstruction: n={n} coefficients, p1=2^63-25, p2=2^63-165",
                   "l2": "inputs larger than L2 only at 8 M coefficients; the kernel is bound by 128-bit integer arithmetic"},
        "gpu_launches": int(api.zippel_launch_count() - n0), "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "k_crt_rational", "achieved": achieved, "peak": IMAD_PEAK_TOPS,
                     "unit": "T multiplier-pipe units/s (IMAD = 1, 32x32->64 product = 2)", "frac": achieved / IMAD_PEAK_TOPS,
                     "traffic": None, "algorithmic_ops_per_launch": units, "ms_per_launch": ms,
                     "algorithmic_cost": "37 Euclid steps x two 64x64->128 products (16 units) per coefficient; the quotient itself "
                                         "(128-bit division, data-dependent) is not in the multiplier count"},
        "e2e": None, "cpu_baseline": cpu}))


if __name__ == "__main__":
    a = parse()
    if a.config == 8:
        run_crt(a)
    elif a.config == 7:
        run_extend(a)
    elif a.config == 6:
        run_thiele(a)
    elif a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
