"""Roofline micro-benchmarks of the sm_100a integer multiplier pipe (csrc/ubench.cuh).

    python -m paper_2505_24256_b200.ubench [--iters 2000] [--reps 5]

Prints, per kind, lane-statements/s, the multiplier instructions per statement, and the implied
lanes per clock per SM at the SM clock nvidia-smi reports during the run.  DESIGN.md "Roofline" quotes it.
"""
from __future__ import annotations

import argparse
import json
import subprocess

import torch

from . import api, testhooks

P = (1 << 63) - 25
KINDS = [
    (0, "IMAD (mad.lo.u32)", 1), (1, "IMAD.WIDE.U32 (mad.wide.u32)", 1), (2, "IMAD.HI.U32 (mad.hi.u32)", 1),
    (3, "IMAD.WIDE + carry-out + IADD3.X (deferred MAC quarter)", 1), (4, "add + xor (alu)", 2),
    (5, "IMAD.WIDE + IADD3 1:1", 1), (6, "IMAD.WIDE + 2 IMAD", 3), (7, "horner_step (10 mult instr)", 10),
    (8, "mont_mul_v1 (column form, 8 wide + 2 low)", 10), (9, "DFMA (fma.rn.f64)", 1), (10, "DFMA + IMAD.WIDE 1:1", 1),
    (11, "IMAD.WIDE.U32 zero addend (mul.wide.u32)", 1),
    (12, "acc_mac (4 accumulating wide)", 4), (13, "acc_mac2 (2 MACs, 8 accumulating wide)", 8),
    (14, "acc_mac_split (4 bare wide + alu chains)", 4), (15, "acc_mac_hyb (2 accumulating + 2 bare wide)", 4),
    (16, "as 3, one multiplicand in an even register", 1),
    (17, "accumulating IMAD.WIDE, multiplicands even+odd", 1), (18, "accumulating IMAD.WIDE, multiplicands even+even", 1),
    (19, "accumulating IMAD.WIDE, multiplicands odd+odd", 1),
    (20, "mont_mul (64-bit REDC, the form in use)", 10), (21, "mont_mul_v3 (bare products + 32-bit chains)", 10),
]


def sm_clock() -> float:
    try:
        o = subprocess.run(["nvidia-smi", "--query-gpu=clocks.sm", "--format=csv,noheader,nounits", "--id=0"],
                           capture_output=True, text=True, timeout=10).stdout
        return float(o.strip().splitlines()[0])
    except Exception:
        return float("nan")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--iters", type=int, default=2000)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--blocks-per-sm", type=int, default=8)
    a = ap.parse_args()
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    blocks = n_sm * a.blocks_per_sm
    out = torch.zeros(blocks * 256, dtype=torch.int64, device="cuda")
    st = torch.cuda.current_stream()
    rows = []
    for kind, name, mults in KINDS:
        best, clk = None, None
        for r in range(a.reps + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            n = testhooks.zippel_ubench(kind, a.iters, blocks, P, out, stream=st)
            e1.record(st)
            if r == a.reps // 2:
                clk = sm_clock()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            if r and (best is None or ms < best):
                best = ms
        per_s = n / (best * 1e-3)
        rows.append(dict(kind=kind, name=name, ms=best, lane_statements_per_s=per_s,
                         mult_instr_per_statement=mults, lane_mult_instr_per_s=per_s * mults, sm_mhz=clk,
                         statements_per_clk_per_sm=per_s / (n_sm * clk * 1e6) if clk == clk else None))
    for r in rows:
        print(json.dumps(r))


if __name__ == "__main__":
    main()
