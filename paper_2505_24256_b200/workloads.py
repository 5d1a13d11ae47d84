"""Seeded synthetic workloads shaped like BASELINE.json's five configs.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests, so it holds
NONE of the method's arithmetic: no modular multiplication, no evaluation, no solve.  It only
draws random exponent rows, residues, anchors and sample values (numpy, counter-based Philox
generator, fixed seeds) and returns them in the C-ABI layouts of include/zippel.h:

  exps     uint16 [T_tot, nv]   row-major skeleton exponents (eq. (3), reading G2)
  offsets  int64  [F+1]         term range of each function
  anchors  uint64 [nv]          y_j in [2, p)            (reading G1)
  samples  uint64 [B]           c_0..c_D in [2, p), pairwise distinct
  planted  uint64 [B, T_tot]    monomial coefficients in x_k of every skeleton coefficient
                                (row d = coefficient of x_k^d); "sparse": one non-zero per term
  vals     uint64 [B, T_tot]    uniform residues, a stand-in for probe values (the solve's cost and
                                code path do not depend on the values; true probe values of the
                                planted function are computed by the oracle in tests/)

The paper's own datasets (IBP reductions) are private; these stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

P63 = (1 << 63) - 25  # largest prime below 2^63 (pinned by the oracle's Miller-Rabin test)
SEED_BASE = 250524256 * 16


def _rng(seed: int, stream: int) -> np.random.Generator:
    """Independent sub-streams (exponents, coefficients, anchors, samples, ...) of one seed."""
    return np.random.Generator(np.random.Philox(key=[int(seed) & (2**64 - 1), int(stream)]))


def uniform_residues(rng: np.random.Generator, lo: int, p: int, size) -> np.ndarray:
    """Uniform integers in [lo, p) as uint64 (numpy's bounded integers use rejection: exact)."""
    return rng.integers(lo, p, size=size, dtype=np.uint64)


def distinct_residues(rng: np.random.Generator, lo: int, p: int, n: int) -> np.ndarray:
    """n pairwise distinct uniform residues in [lo, p) (redraw on collision)."""
    if p - lo < n:
        raise ValueError("not enough residues")
    out = uniform_residues(rng, lo, p, n)
    while len(np.unique(out)) != n:
        uniq, first = np.unique(out, return_index=True)
        dup = np.setdiff1d(np.arange(n), first)
        out[dup] = uniform_residues(rng, lo, p, len(dup))
    return out


def box_rows(rng: np.random.Generator, t: int, nv: int, emax: int) -> np.ndarray:
    """t distinct exponent rows uniform in [0, emax]^nv (sampling without replacement)."""
    base = emax + 1
    n_cand = base**nv
    if n_cand < t:
        raise ValueError("box too small for t distinct rows")
    if n_cand < 2**62:
        idx = rng.choice(n_cand, size=t, replace=False)
        idx = np.asarray(idx, dtype=np.uint64)
        rows = np.empty((t, nv), dtype=np.uint16)
        for j in range(nv):
            rows[:, j] = (idx % np.uint64(base)).astype(np.uint16)
            idx = idx // np.uint64(base)
        return rows
    rows = rng.integers(0, base, size=(t, nv), dtype=np.uint16)
    while len(np.unique(rows, axis=0)) != t:
        _, first = np.unique(rows, axis=0, return_index=True)
        dup = np.setdiff1d(np.arange(t), first)
        rows[dup] = rng.integers(0, base, size=(len(dup), nv), dtype=np.uint16)
    return rows


def simplex_rows(rng: np.random.Generator, t: int, nvars: int, total: int) -> np.ndarray:
    """t exponent tuples uniform over the integer points of sum_j e_j <= total (stars and bars:
    a uniform nvars-subset of total+nvars slots), redrawn until the projections onto the first
    nvars-1 variables are pairwise distinct (config 4)."""
    slots = total + nvars

    def draw(n):
        keys = rng.random((n, slots))
        bars = np.sort(np.argsort(keys, axis=1)[:, :nvars], axis=1)
        e = np.empty((n, nvars), dtype=np.int64)
        e[:, 0] = bars[:, 0]
        e[:, 1:] = bars[:, 1:] - bars[:, :-1] - 1
        return e.astype(np.uint16)

    rows = draw(t)
    while len(np.unique(rows[:, :-1], axis=0)) != t:
        _, first = np.unique(rows[:, :-1], axis=0, return_index=True)
        dup = np.setdiff1d(np.arange(t), first)
        rows[dup] = draw(len(dup))
    return rows


def lowest_monomial(rows: np.ndarray) -> int:
    """Index of the lowest row in the graded order of reading G19: smaller total degree first,
    ties by lexicographically smaller (e_1, e_2, ...)."""
    deg = rows.astype(np.int64).sum(axis=1)
    keys = [rows[:, j] for j in range(rows.shape[1] - 1, -1, -1)] + [deg]
    return int(np.lexsort(keys)[0])


@dataclass
class Workload:
    """One batch of F functions sharing anchors and samples (one part of a rational batch)."""

    name: str
    p: int
    F: int
    nv: int
    B: int
    s0: int
    exps: np.ndarray
    offsets: np.ndarray
    anchors: np.ndarray
    samples: np.ndarray
    planted: Optional[np.ndarray] = None  # [B, T_tot] monomial-in-x_k coefficients
    xk_exp: Optional[np.ndarray] = None  # [T_tot] g_i of the "sparse" law, else None
    vals: Optional[np.ndarray] = None  # [B, T_tot] uniform stand-in values
    meta: dict = field(default_factory=dict)

    @property
    def T_tot(self) -> int:
        return int(self.offsets[-1])


def _planted(rng, T_tot: int, B: int, p: int, xk_exp: Optional[np.ndarray], dense: bool) -> np.ndarray:
    if dense:
        return uniform_residues(rng, 0, p, (B, T_tot))
    out = np.zeros((B, T_tot), dtype=np.uint64)
    out[xk_exp.astype(np.int64), np.arange(T_tot)] = uniform_residues(rng, 1, p, T_tot)
    return out


def make_box_workload(name: str, seed: int, F: int, nv: int, t, emax: int, B: int, p: int = P63,
                      s0: int = 0, dense: bool = False, with_vals: bool = True,
                      with_planted: bool = True) -> Workload:
    """Polynomial-lift workload: F functions, t terms each (t: int or per-function list), exponent
    rows distinct and uniform in [0, emax]^nv per function, B = D+1 samples of x_k."""
    ts = [int(t)] * F if np.isscalar(t) else [int(x) for x in t]
    assert len(ts) == F
    offsets = np.zeros(F + 1, dtype=np.int64)
    offsets[1:] = np.cumsum(ts)
    T_tot = int(offsets[-1])
    r_exp = _rng(seed, 1)
    exps = np.empty((T_tot, nv), dtype=np.uint16)
    for f in range(F):
        exps[offsets[f]:offsets[f + 1]] = box_rows(r_exp, ts[f], nv, emax)
    anchors = uniform_residues(_rng(seed, 3), 2, p, nv)
    samples = distinct_residues(_rng(seed, 4), 2, p, B)
    xk_exp = _rng(seed, 5).integers(0, B, size=T_tot, dtype=np.int64)
    planted = _planted(_rng(seed, 2), T_tot, B, p, xk_exp, dense) if with_planted else None
    vals = uniform_residues(_rng(seed, 6), 0, p, (B, T_tot)) if with_vals else None
    return Workload(name, p, F, nv, B, s0, exps, offsets, anchors, samples, planted,
                    None if dense else xk_exp, vals, {"emax": emax, "dense": dense, "seed": seed})


@dataclass
class RationalWorkload:
    """Config 4: F rational functions N/D; parts share anchors, samples and the per-probe factors."""

    name: str
    num: Workload
    den: Workload
    low_den: np.ndarray  # [F] index (within the function) of D's lowest monomial (reading G19)
    h: np.ndarray  # [max t] per-probe factors h_s in [1, p)  (reading G3, G20)
    skel: Optional[np.ndarray] = None  # stand-in skeleton coefficients / u values for full-size runs
    meta: dict = field(default_factory=dict)


def make_rational_workload(name: str, seed: int, F: int, nvars: int, t_num, t_den,
                           total: int, B: int, p: int = P63, s0: int = 0,
                           with_vals: bool = True) -> RationalWorkload:
    """t_num, t_den: terms of every numerator / denominator, an int or a per-function list (ragged batches)."""
    nv = nvars - 1
    anchors = uniform_residues(_rng(seed, 3), 2, p, nv)
    samples = distinct_residues(_rng(seed, 4), 2, p, B)
    parts = []
    tmax = 0
    for part, t, stream in (("num", t_num, 10), ("den", t_den, 20)):
        ts = [int(t)] * F if np.isscalar(t) else [int(x) for x in t]
        assert len(ts) == F
        tmax = max(tmax, max(ts))
        offsets = np.zeros(F + 1, dtype=np.int64)
        offsets[1:] = np.cumsum(ts)
        T_tot = int(offsets[-1])
        r_exp = _rng(seed, stream + 1)
        full = np.empty((T_tot, nvars), dtype=np.uint16)
        for f in range(F):
            full[offsets[f]:offsets[f + 1]] = simplex_rows(r_exp, ts[f], nvars, total)
        exps = np.ascontiguousarray(full[:, :nv])
        xk_exp = full[:, nv].astype(np.int64)
        if xk_exp.max() >= B:
            raise ValueError("B must exceed the degree bound in x_k")
        planted = _planted(_rng(seed, stream + 2), T_tot, B, p, xk_exp, False)
        vals = uniform_residues(_rng(seed, stream + 6), 1, p, (B, T_tot)) if with_vals else None
        w = Workload(f"{name}.{part}", p, F, nv, B, s0, exps, offsets, anchors, samples, planted,
                     xk_exp, vals, {"total": total, "seed": seed})
        w.meta["skel_standin"] = uniform_residues(_rng(seed, stream + 7), 1, p, T_tot) if with_vals else None
        parts.append(w)
    num, den = parts
    low = np.array([lowest_monomial(den.exps[den.offsets[f]:den.offsets[f + 1]]) for f in range(F)], dtype=np.int64)
    h = uniform_residues(_rng(seed, 30), 1, p, tmax)
    return RationalWorkload(name, num, den, low, h, None, {"seed": seed})


# ---- the five BASELINE.json configs (index 1..5; BASELINE.json's configs[i-1]) -------------------

CONFIG_SHAPES = {
    1: dict(F=1, nv=2, t=50, emax=10, B=11),
    2: dict(F=4096, nv=4, t=1000, emax=20, B=21),
    3: dict(F=1, nv=7, t=100000, emax=30, B=9),
    4: dict(F=1024, nvars=6, t_num=500, t_den=200, total=24, B=25),
    5: dict(F=1, nv=10, t=524288, emax=40, B=1),
    # not a BASELINE.json config: the paper's largest skeleton (4.8m monomials, reconstructing the 6th
    # variable), one right-hand side -- bench.py --config 9 (row f3)
    9: dict(F=1, nv=5, t=4_800_000, emax=40, B=1),
}


def config(idx: int, F: Optional[int] = None, t: Optional[int] = None, dense: bool = False,
           with_vals: bool = True, with_planted: bool = True):
    """Config idx in 1..5, optionally reduced (fewer functions F, a shorter skeleton t) for the
    oracle-sized parity cases.  Seed = 250524256*16 + idx."""
    seed = SEED_BASE + idx
    sh = dict(CONFIG_SHAPES[idx])
    if F is not None:
        sh["F"] = F
    if idx == 4:
        if t is not None:
            sh["t_num"], sh["t_den"] = t, max(1, (t * 2) // 5)
        return make_rational_workload(f"C4", seed, sh["F"], sh["nvars"], sh["t_num"], sh["t_den"],
                                      sh["total"], sh["B"], with_vals=with_vals)
    if t is not None:
        sh["t"] = t
    return make_box_workload(f"C{idx}", seed, sh["F"], sh["nv"], sh["t"], sh["emax"], sh["B"],
                             dense=dense, with_vals=with_vals, with_planted=with_planted)
