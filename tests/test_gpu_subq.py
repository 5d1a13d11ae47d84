"""The sub-quadratic route for long skeletons (csrc/subq.cuh) against the CPU oracle: the answer is
the unique solution of the transposed Vandermonde system (reading G21), so every comparison is == with
oracle.vandermonde_solve_batch -- the quadratic textbook route of PAPER.md section 2.2.  The switch-over length is
forced down (zippel_set_tuning) so that the oracle finishes in seconds while the skeletons still cross every
structural boundary: one and several 1024-node leaves, ragged last leaves (down to a single node), one-, two- and
three-level trees, transform lengths above 4096 (two-pass NTT), batches that mix both routes, s0 = 1, statuses."""
import numpy as np
import pytest
import torch

from paper_2505_24256_b200 import workloads as wl

pytestmark = pytest.mark.gpu
P63 = wl.P63


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


@pytest.fixture()
def low(zp):
    zp.zippel_set_tuning(zp.TUNE_SUBQ_MIN_T, 1025)
    yield
    zp.zippel_set_tuning(zp.TUNE_SUBQ_MIN_T, zp.SUBQ_MIN_T_DEFAULT)


def make(ts, B, seed, p=P63, nv=4, emax=40):
    w = wl.make_box_workload("subq", seed, len(ts), nv, ts, emax, B, p=p)
    return w


def solve_both(zp, ref, w, nodes, vals, s0):
    want, wst = ref.vandermonde_solve_batch(nodes, w.offsets, vals, w.p, s0)
    got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), w.offsets, zp.to_dev(vals), w.p, s0)
    torch.cuda.synchronize()
    return zp.to_host(got), zp.to_host(st), want, wst


@pytest.mark.parametrize("t", [1025, 1500, 2047, 2048, 2049, 3000, 3073, 4097, 5000, 9001])
@pytest.mark.parametrize("B,s0", [(1, 0), (3, 1)])
def test_single_long_function(zp, ref, low, t, B, s0):
    w = make([t], B, 9100 + t)
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    got, st, want, wst = solve_both(zp, ref, w, nodes, w.vals, s0)
    assert not wst.any() and (st == wst).all()
    assert (got == want).all()


def test_planted_coefficients_come_back(zp, ref, low):
    """The values are the power sums of planted coefficients (made by the oracle): the solve returns them."""
    t, B = 4500, 2
    w = make([t], B, 9201)
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    planted = wl.uniform_residues(wl._rng(9201, 77), 0, w.p, (B, t))
    vals = ref.power_sums(nodes, w.offsets, planted, w.p, 0)
    got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), w.offsets, zp.to_dev(vals), w.p, 0)
    torch.cuda.synchronize()
    assert not zp.to_host(st).any()
    assert (zp.to_host(got) == planted).all()


@pytest.mark.parametrize("ts", [[1100, 2500], [300, 2100, 700, 1026, 5000, 1024], [2000, 2000, 2000], [4097, 50]])
@pytest.mark.parametrize("B", [1, 9])
def test_batches_mixing_both_routes(zp, ref, low, ts, B):
    w = make(ts, B, 9300 + len(ts) + B)
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    got, st, want, wst = solve_both(zp, ref, w, nodes, w.vals, 0)
    assert not wst.any() and (st == wst).all()
    assert (got == want).all()


@pytest.mark.parametrize("B", [26, 64])
def test_many_right_hand_sides(zp, ref, low, B):
    """B + 1 rows go through the leaf solve in passes of at most 25."""
    w = make([2300], B, 9400 + B)
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    got, st, want, wst = solve_both(zp, ref, w, nodes, w.vals, 0)
    assert (st == wst).all() and (got == want).all()


@pytest.mark.parametrize("p", [65537, (1 << 31) - 1, (1 << 61) - 1])
def test_other_primes(zp, ref, low, p):
    t = 2600
    w = make([t], 2, 9500, p=p, nv=3, emax=60)
    nodes = wl.distinct_residues(wl._rng(9500, p & 0xFFFF), 1, p, t)  # exponent rows collide modulo a small p
    got, st, want, wst = solve_both(zp, ref, w, nodes, w.vals, 1)
    assert not wst.any() and (st == wst).all()
    assert (got == want).all()


def test_duplicate_and_zero_nodes(zp, ref, low):
    """A repeated node makes M'(m_i) vanish at both copies: status DUPLICATE_NODE with the smaller index, like the
    oracle; a zero node is legal for s0 = 0 and an error for s0 = 1 (readings G24, G25).  The second, healthy
    function of the batch is unaffected."""
    ts = [2200, 1300]
    w = make(ts, 2, 9600)
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    nodes[1700] = nodes[40]
    got, st, want, wst = solve_both(zp, ref, w, nodes, w.vals, 0)
    assert wst[0] == (40 << 8 | 16) and (st == wst).all()
    assert (got[:, 2200:] == want[:, 2200:]).all()
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    nodes[2200 + 7] = 0
    got, st, want, wst = solve_both(zp, ref, w, nodes, w.vals, 0)
    assert not wst.any() and (st == wst).all() and (got == want).all()
    got, st, want, wst = solve_both(zp, ref, w, nodes, w.vals, 1)
    assert wst[1] == (7 << 8 | 16) and (st == wst).all()
    assert (got[:, :2200] == want[:, :2200]).all()


def test_lift_step_takes_the_route_too(zp, ref, low):
    """zippel_lift_step = nodes + solve + Newton: a long function in the batch changes nothing in the result."""
    w = make([1500, 600], 4, 9700)
    want, _, wst = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, w.vals, w.p, 0, 1)
    got, st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(w.anchors), zp.to_dev(w.samples), zp.to_dev(w.vals),
                                  w.p, 0, 1)
    torch.cuda.synchronize()
    assert (zp.to_host(st) == wst).all() and (zp.to_host(got) == want).all()


def test_intermediates_master_polynomial_and_power_sums(zp, ref):
    """Two intermediates of the route have oracle counterparts: the top-level master polynomial (ref.master_poly,
    pinned by Vieta and the roots) and the root tail of M', which is the power-sum sequence of the nodes
    (ref.power_sums with unit coefficients).  Read through the dump hook of the test build."""
    from paper_2505_24256_b200 import testhooks

    t, B, p = 3500, 1, P63
    w = make([t], B, 9800)
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    inv64 = pow(1 << 64, -1, p)
    with testhooks.routed():
        zp.zippel_set_tuning(zp.TUNE_SUBQ_MIN_T, 1025)
        try:
            for stage, words in ((1, t), (3, 2 * t)):
                out = torch.zeros(words, dtype=torch.int64, device="cuda")
                testhooks.subq_dump(stage, out)
                zp.vandermonde_solve_batch(zp.to_dev(nodes), w.offsets, zp.to_dev(w.vals), p, 0)
                torch.cuda.synchronize()
                testhooks.subq_dump(0, None)
                got = zp.to_host(out)
                if stage == 1:
                    M = ref.master_poly(nodes, p)
                    assert [int(x) * inv64 % p for x in got] == [int(x) for x in M[:t]]
                else:
                    assert (got[:t] == w.vals[0]).all()
                    ones = np.ones((1, t), dtype=np.uint64)
                    assert (got[t:] == ref.power_sums(nodes, w.offsets, ones, p, 0)[0]).all()
        finally:
            zp.zippel_set_tuning(zp.TUNE_SUBQ_MIN_T, zp.SUBQ_MIN_T_DEFAULT)
