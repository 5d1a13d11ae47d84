"""Measure where the sub-quadratic route (csrc/subq.cuh) overtakes the quadratic kernels of PAPER.md section 2.2.

    python -m paper_2505_24256_b200.crossover [--out crossover.json]

For F in {1, 64, 4096} functions of t terms and B right-hand sides, vandermonde_solve_batch is timed (CUDA events on the
launching stream, 3 warm-ups, 10 repetitions) with the route forced either way through zippel_set_tuning, and the
two results are compared for equality.  The built-in rule (sq_threshold in csrc/zippel_capi.cu, include/zippel.h)
was read off this table (profiles/r02_crossover.md).
"""
from __future__ import annotations

import argparse
import json

import numpy as np
import torch

from . import api, workloads as wl


def run(t, B, F, route, reps=10):
    P = wl.P63
    api.zippel_set_tuning(api.TUNE_SUBQ_MIN_T, 513 if route == "subq" else (1 << 22))
    r = np.random.Generator(np.random.Philox(key=[5, t]))
    offs = np.arange(F + 1, dtype=np.int64) * t
    nodes = np.empty(F * t, dtype=np.uint64)
    for f in range(F):
        nodes[f * t:(f + 1) * t] = wl.distinct_residues(r, 1, P, t)
    vals = r.integers(0, P, (B, F * t), dtype=np.uint64)
    dn, dv = api.to_dev(nodes), api.to_dev(vals)
    ws = api.alloc_workspace(offs, B)
    out = torch.empty_like(dv)
    st = torch.empty(F, dtype=torch.int32, device="cuda")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        for _ in range(3):
            api.vandermonde_solve_batch(dn, offs, dv, P, 0, out=out, status=st, workspace=ws, stream=s)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(s)
        for _ in range(reps):
            api.vandermonde_solve_batch(dn, offs, dv, P, 0, out=out, status=st, workspace=ws, stream=s)
        e1.record(s)
        torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps, out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    api.lib()
    res = []
    try:
        cases = [(F, B, t) for F in (1, 64) for B in (1, 3, 9, 21)
                 for t in (1536, 2048, 3072, 4096, 6144, 8192, 12288, 16384, 32768) if F * t * B <= 1 << 26]
        # many short functions (BASELINE.json configs[1] is 4096 functions of 1000 terms): the batch threshold
        cases += [(4096, B, t) for B in (1, 21) for t in (640, 800, 960, 1000, 1280, 1536)]
        for F, B, t in cases:
            reps = 10 if F < 4096 else 3
            q_ms, oq = run(t, B, F, "quad", reps)
            s_ms, os_ = run(t, B, F, "subq", reps)
            same = bool((oq == os_).all())
            res.append(dict(F=F, B=B, t=t, quad_ms=q_ms, subq_ms=s_ms, same=same))
            print(f"F={F} B={B} t={t} quadratic {q_ms:.3f} ms sub-quadratic {s_ms:.3f} ms {'same' if same else 'DIFFERENT'}",
                  flush=True)
    finally:
        api.zippel_set_tuning(api.TUNE_SUBQ_MIN_T, api.SUBQ_MIN_T_DEFAULT)
    if a.out:
        with open(a.out, "w") as fh:
            json.dump(res, fh)


if __name__ == "__main__":
    main()
