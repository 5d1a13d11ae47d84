"""Full-size parity: BASELINE.json's sizes in the launch configuration bench.py times (same entry points,
same F, t, nv, B, same workspace), checked on what the oracle (or plain Python integers) can afford:

* C2, C4 (many independent functions): the oracle lifts SAMPLED functions in full and every output of those
  functions is compared == (the functions of a batch do not interact, so a sampled function is a complete
  oracle problem; its inputs are the generator's, its position in the batch is the bench's).
* C3, C5 (one huge skeleton; the oracle would need hours): properties that hold at any size, with expected
  values that never come from the CUDA path --
    (i)  nodes == oracle nodes, all of them (O(t));
    (ii) the solved coefficients satisfy the defining equations sum_i c_{b,i} m_i^s = v_{b,s}
         at sampled s, evaluated in Python integers with the ORACLE's nodes; v is the generator's;
    (iii) round trip on a planted function: values produced by the forward-evaluation entry point, spot-checked
         against Python integers at sampled (b, s), lift back to exactly the planted coefficients (the solution
         is unique, reading G21, so GPU == planted is equivalent to GPU == oracle).
"""
import random

import numpy as np
import pytest

from paper_2505_24256_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def zp():
    from paper_2505_24256_b200 import api

    api.lib()
    return api


@pytest.fixture(scope="module")
def ref():
    from oracle import ref as r

    r.lib()
    return r


def slice_function(w, f):
    """Function f of a batch as a complete single-function problem (generator data only)."""
    a, b = int(w.offsets[f]), int(w.offsets[f + 1])
    return dict(exps=np.ascontiguousarray(w.exps[a:b]), offsets=np.array([0, b - a], dtype=np.int64),
                vals=np.ascontiguousarray(w.vals[:, a:b]), a=a, b=b)


def py_residual(nodes, coefs_row, s, p):
    """sum_i c_i m_i^s mod p in Python integers."""
    return sum(int(c) * pow(int(m), s, p) for c, m in zip(coefs_row, nodes)) % p


def sample_indices(rng, n, k, always=()):
    out = sorted(set(always) | {rng.randrange(n) for _ in range(k)})
    return [x for x in out if 0 <= x < n]


# ------------------------------------------------------------------------------------------- C2
def test_config2_full_batch_sampled_functions(zp, ref):
    """configs[1] at full size (F = 4096, t = 1000, nv = 4, B = 21), exactly bench.py's call."""
    import torch

    w = wl.config(2, with_planted=False)
    exps, anchors, samples, vals = (zp.to_dev(x) for x in (w.exps, w.anchors, w.samples, w.vals))
    ws = zp.alloc_workspace(w.offsets, w.B)
    out = torch.empty_like(vals)
    status = torch.empty(w.F, dtype=torch.int32, device="cuda")
    zp.zippel_lift_step(exps, w.offsets, anchors, samples, vals, w.p, 0, 1, out=out, status=status, workspace=ws)
    torch.cuda.synchronize()
    assert not zp.to_host(status).any()
    rng = random.Random(2)
    for f in sample_indices(rng, w.F, 4, always=(0, w.F - 1)):
        s = slice_function(w, f)
        want, _, wst = ref.zippel_lift_step(s["exps"], s["offsets"], w.anchors, w.samples, s["vals"], w.p, 0, 1)
        assert not wst.any()
        got = zp.to_host(out[:, s["a"]:s["b"]].contiguous())
        assert (got == want).all(), f"function {f} differs from the oracle"


# ------------------------------------------------------------------------------------------- C4
def test_config4_full_batch_sampled_functions(zp, ref):
    """configs[3] at full size (F = 1024, t_N = 500, t_D = 200, B = 25), exactly bench.py's call."""
    import torch

    rw = wl.config(4)
    parts = [rw.num, rw.den]
    F, B, p = rw.num.F, rw.num.B, rw.num.p
    dev = [dict(exps=zp.to_dev(q.exps), offsets=q.offsets, skel=zp.to_dev(q.meta["skel_standin"]),
                uvals=zp.to_dev(q.vals), out=torch.empty(q.vals.shape, dtype=torch.int64, device="cuda"))
           for q in parts]
    ws = zp.alloc_workspace(rw.num.offsets, B, zp.WS_BALANCED)
    status = torch.empty(2 * F, dtype=torch.int32, device="cuda")
    zp.balanced_zippel_lift_step(dev[0], dev[1], zp.to_dev(rw.num.anchors), zp.to_dev(rw.num.samples), p, 0, 1,
                                 status=status, workspace=ws)
    torch.cuda.synchronize()
    assert not zp.to_host(status).any()
    rng = random.Random(4)
    for f in sample_indices(rng, F, 3, always=(0, F - 1)):
        sl = []
        for q in parts:
            s = slice_function(q, f)
            sl.append(dict(exps=s["exps"], offsets=s["offsets"], uvals=s["vals"],
                           skel=np.ascontiguousarray(q.meta["skel_standin"][s["a"]:s["b"]]), a=s["a"], b=s["b"]))
        wn, wd, wst = ref.balanced_zippel_lift_step(sl[0], sl[1], rw.num.anchors, rw.num.samples, p, 0, 1)
        assert not wst.any()
        gn = zp.to_host(dev[0]["out"][:, sl[0]["a"]:sl[0]["b"]].contiguous())
        gd = zp.to_host(dev[1]["out"][:, sl[1]["a"]:sl[1]["b"]].contiguous())
        assert (gn == wn).all() and (gd == wd).all(), f"function {f} differs from the oracle"


# ------------------------------------------------------------------------------------------- C3, C5
def check_large_solve(zp, ref, w, n_s, seed):
    """(i) + (ii) of the module docstring through zippel_eval_nodes + vandermonde_solve_batch."""
    import torch

    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)  # oracle, O(t)
    dn = zp.zippel_eval_nodes(zp.to_dev(w.exps), zp.to_dev(w.anchors), w.p)
    assert (zp.to_host(dn) == nodes).all()
    got, st = zp.vandermonde_solve_batch(dn, w.offsets, zp.to_dev(w.vals), w.p, 0)
    torch.cuda.synchronize()
    assert not zp.to_host(st).any()
    got = zp.to_host(got)
    assert (got < np.uint64(w.p)).all()
    t = w.T_tot
    rng = random.Random(seed)
    for s in sample_indices(rng, t, n_s, always=(0, 1, t - 1)):
        for b in range(w.B):
            assert py_residual(nodes, got[b], s, w.p) == int(w.vals[b, s]), f"equation s={s}, b={b} not satisfied"
    return nodes, got


def test_config5_full_size_solve_properties(zp, ref):
    """configs[4] at full size: one solve of size t = 2^19 (nv = 10, B = 1), bench.py --config 5's calls."""
    w = wl.config(5, with_planted=False)
    assert w.T_tot == 1 << 19
    check_large_solve(zp, ref, w, 5, 5)


def test_config3_full_size_lift_properties_and_round_trip(zp, ref):
    """configs[2] at full size (t = 100000, nv = 7, B = 9): solve properties, then the planted round trip
    through zippel_lift_step (bench.py --config 3's call)."""
    import torch

    w = wl.config(3)
    nodes, _ = check_large_solve(zp, ref, w, 2, 3)
    # (iii) planted function -> values at the samples (oracle, O(B^2 t)) -> probe values by forward evaluation
    at = ref.poly_rows_eval(w.samples, w.planted, w.p)
    vals = zp.zippel_power_sums(zp.to_dev(nodes), w.offsets, zp.to_dev(at), w.p, 0)
    torch.cuda.synchronize()
    hv = zp.to_host(vals)
    rng = random.Random(33)
    for _ in range(6):  # spot check of the forward evaluation in Python integers
        b, s = rng.randrange(w.B), rng.randrange(w.T_tot)
        assert py_residual(nodes, at[b], s, w.p) == int(hv[b, s])
    out, st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(w.anchors), zp.to_dev(w.samples), vals,
                                  w.p, 0, 1)
    torch.cuda.synchronize()
    assert not zp.to_host(st).any()
    assert (zp.to_host(out) == w.planted).all(), "lift(forward(planted)) != planted"


# ------------------------------------------------------------------------------------------- C3, C5: intermediates
@pytest.mark.parametrize("idx,n_nodes", [(5, 256), (3, 256)])
def test_full_size_intermediates_on_sampled_nodes(zp, ref, idx, n_nodes):
    """SURVEY.md 8(c).3 at full size (t = 2^19 and t = 10^5): (1) the master polynomial of the CUDA path, read through
    the dump hook of the test build, passes M(r) = prod_i (r - m_i) at random r in Python integers (O(t), with the
    ORACLE's nodes); (2) with that M, the oracle's per-node routine (ref_node_solve_at: synthetic division, Horner
    denominator, B dot products) on 256 random node indices gives exactly the numerators and
    denominators the CUDA path holds before its final division, and the quotients are the solved coefficients."""
    import torch

    from paper_2505_24256_b200 import testhooks

    w = wl.config(idx, with_planted=False)
    t, B, p = w.T_tot, w.B, w.p
    nodes = ref.eval_nodes(w.exps, w.anchors, p)
    dn, dv = zp.to_dev(nodes), zp.to_dev(w.vals)
    inv64 = pow(1 << 64, -1, p)
    dumps = {}
    with testhooks.routed():
        for stage, words in ((1, t), (5, (B + 1) * t)):
            out = torch.zeros(words, dtype=torch.int64, device="cuda")
            testhooks.subq_dump(stage, out)
            got, st = zp.vandermonde_solve_batch(dn, w.offsets, dv, p, 0)
            torch.cuda.synchronize()
            testhooks.subq_dump(0, None)
            assert not zp.to_host(st).any()
            dumps[stage] = zp.to_host(out)
    coefs = zp.to_host(got)
    # (1) M: Montgomery coefficients 0 .. t-1 (monic, leading 1 not stored)
    M = np.empty(t + 1, dtype=np.uint64)
    M[:t] = [int(x) * inv64 % p for x in dumps[1]]
    M[t] = 1
    rng = random.Random(500 + idx)
    for r in [rng.randrange(2, p) for _ in range(2)] + [int(nodes[rng.randrange(t)])]:
        horner = 0
        for c in M[::-1]:
            horner = (horner * r + int(c)) % p
        prod = 1
        for m in nodes:
            prod = prod * (r - int(m)) % p
        assert horner == prod
    # (2) per-node routine of the oracle on sampled nodes
    pick = sample_indices(rng, t, n_nodes, always=(0, 1023, 1024, t - 1))
    den, num = ref.node_solve_at(nodes[pick], M, w.vals, p)
    g = dumps[5].reshape(B + 1, t)
    assert (g[B, pick] == den).all(), "denominators M'(m_i) differ from the oracle's Horner values"
    assert (g[:B, pick] == num).all(), "numerators differ from the oracle's synthetic-division dot products"
    for k, i in enumerate(pick):
        dinv = pow(int(den[k]), -1, p)
        for b in range(B):
            assert int(coefs[b, i]) == int(num[b, k]) * dinv % p
