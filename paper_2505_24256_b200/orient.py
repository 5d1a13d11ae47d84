"""Derive ZP_K3_ORIENT_MASK (csrc/kernels.cuh) from the SASS that THIS nvcc generates.

    python -m paper_2505_24256_b200.orient [--write profiles/r02_k3_orient.md]

k_node_solve<NB> reads its broadcast value operands as 16-byte records {v_odd.lo, v_even.lo, v_odd.hi, v_even.hi} or
the same with even first (ZP_K3_ORIENT); either way the two limbs of one operand land in registers of the same
parity.  Which order ptxas's register allocation serves with fewer register-bank conflicts differs from template
instance to template instance, so it is read off the SASS: for both orders every instance NB = 1 .. 25 is compiled
(nvcc -cubin, no GPU needed), and among the accumulating wide multiply-adds of its hot loop (IMAD.WIDE.U32 with a
non-zero register addend) the share whose two multiplicand registers have EQUAL parity is counted -- those are the
ones that collide in a register bank (profiles/r01_final.md, register banks).  The mask takes, per NB, the order with
the smaller share.  The table depends on the ptxas version: tests/test_orient_table.py fails when `nvcc --version`
differs from the one recorded in profiles/r02_k3_orient.md, so that a toolchain change forces this to be run again.
"""
from __future__ import annotations

import argparse
import os
import re
import subprocess
import sys
import tempfile

_HERE = os.path.dirname(os.path.abspath(__file__))
_KERNELS = os.path.join(_HERE, "csrc", "kernels.cuh")
NB_MAX = 25

_INST = "#include \"%s\"\n" % _KERNELS + "".join(
    "template __global__ void k_node_solve<%d>(const uint64_t*, const ulonglong4*, const int64_t*, int, const uint64_t*, "
    "int64_t, int, int, ZpMod, const uint64_t*, uint64_t*, int32_t*);\n" % nb for nb in range(1, NB_MAX + 1))

_WIDE = re.compile(r"IMAD\.WIDE\.U32\s+R\d+,\s+(?:P\d,\s+)?R(\d+)(?:\.reuse)?,\s+R(\d+)(?:\.reuse)?,\s+R(\d+)")
_FUNC = re.compile(r"Function : _Z12k_node_solveILi(\d+)E")


def nvcc_version() -> str:
    from . import build

    out = subprocess.run([build._nvcc(), "--version"], stdout=subprocess.PIPE, text=True).stdout
    m = re.search(r"release [^,]+, (V[\d.]+)", out)
    return m.group(1) if m else out.strip().splitlines()[-1]


def equal_parity_shares(orient: int, workdir: str) -> dict:
    """{NB: (accumulating wide multiply-adds with register multiplicands, those of equal parity)}"""
    from . import build

    src = os.path.join(workdir, "inst.cu")
    cubin = os.path.join(workdir, f"o{orient}.cubin")
    with open(src, "w") as fh:
        fh.write(_INST)
    subprocess.run([build._nvcc(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-cubin",
                    f"-DZP_K3_FORCE_ORIENT={orient}", "-o", cubin, src], check=True)
    sass = subprocess.run(["cuobjdump", "-sass", cubin], stdout=subprocess.PIPE, text=True, check=True).stdout
    res, nb = {}, None
    for line in sass.splitlines():
        f = _FUNC.search(line)
        if f:
            nb = int(f.group(1))
            res[nb] = [0, 0]
            continue
        if nb is None:
            continue
        m = _WIDE.search(line)
        if m:  # both multiplicands in registers and a register addend: an accumulating product of the hot loop
            a, b = int(m.group(1)), int(m.group(2))
            res[nb][0] += 1
            res[nb][1] += (a & 1) == (b & 1)
    return {k: tuple(v) for k, v in res.items()}


def derive():
    with tempfile.TemporaryDirectory() as wd:
        s0, s1 = equal_parity_shares(0, wd), equal_parity_shares(1, wd)
    mask, rows = 0, []
    for nb in range(1, NB_MAX + 1):
        f0 = s0[nb][1] / max(1, s0[nb][0])
        f1 = s1[nb][1] / max(1, s1[nb][0])
        pick = 1 if f1 < f0 else 0
        mask |= pick << nb
        rows.append((nb, s0[nb][0], f0, s1[nb][0], f1, pick))
    return mask, rows


def current_mask() -> int:
    m = re.search(r"#define ZP_K3_ORIENT_MASK (0x[0-9a-fA-F]+)u", open(_KERNELS).read())
    return int(m.group(1), 16)


def report(mask, rows) -> str:
    out = ["# Orientation of k_node_solve's value records per template instance (round 2)", "",
           "Command: `python -m paper_2505_24256_b200.orient --write profiles/r02_k3_orient.md` (compiles with nvcc -cubin; no GPU).", "",
           f"nvcc: {nvcc_version()}", f"derived mask: {mask:#x}", f"mask in csrc/kernels.cuh: {current_mask():#x}", "",
           "Share of the accumulating `IMAD.WIDE.U32` (register multiplicands, register addend) whose two multiplicand registers",
           "have equal parity, per order of the 16-byte value record (0: even stage first, 1: odd stage first):", "",
           "| NB | wide MACs (order 0) | equal parity (order 0) | wide MACs (order 1) | equal parity (order 1) | chosen |",
           "|---|---|---|---|---|---|"]
    for nb, n0, f0, n1, f1, pick in rows:
        out.append(f"| {nb} | {n0} | {f0:.3f} | {n1} | {f1:.3f} | {pick} |")
    return "\n".join(out) + "\n"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--write", default=None, help="write the table (markdown) to this path")
    a = ap.parse_args()
    mask, rows = derive()
    txt = report(mask, rows)
    sys.stdout.write(txt)
    if a.write:
        with open(a.write, "w") as fh:
            fh.write(txt)
    if mask != current_mask():
        sys.stderr.write(f"ZP_K3_ORIENT_MASK in csrc/kernels.cuh is {current_mask():#x}; this toolchain gives {mask:#x}\n")


if __name__ == "__main__":
    main()
