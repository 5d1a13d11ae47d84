"""Bit-exact parity of zippel_extend_skeleton (C-ABI) with the CPU oracle, and a two-step chain
lift -> extend -> lift on the GPU that recovers a planted polynomial (expected values: the generator's)."""
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


def both(zp, ref, w, coefs, cap=None):
    import torch

    we, wc, wo, wd = ref.extend_skeleton(w.exps, w.offsets, coefs, w.p, cap)
    ge, gc, go, gd = zp.zippel_extend_skeleton(zp.to_dev(w.exps), w.offsets, zp.to_dev(coefs), w.p, cap)
    torch.cuda.synchronize()
    go, gd = go.cpu().numpy(), gd.cpu().numpy()
    assert (go == wo).all() and (gd == wd).all()
    n = len(wc)
    assert (zp.to_host(gc[:n]) == wc).all()
    assert (zp.to_host(ge[:n]) == we).all()
    return we, wc, wo


@pytest.mark.parametrize("dense", [False, True])
def test_extend_parity_ragged_batch_with_holes(zp, ref, dense):
    w = wl.make_box_workload("ext", wl.SEED_BASE + 93, 6, 3, [300, 1, 257, 256, 2, 1000], 9, 7, dense=dense)
    coefs = w.planted.copy()
    coefs[:, 5] = 0          # a vanished term
    coefs[:, 300] = 0        # the whole one-term function vanishes
    coefs[4:, 301:558] = 0   # function 2 has degree 3 < B - 1
    coefs[0, ::3] = w.p      # a non-canonical zero
    both(zp, ref, w, coefs)
    both(zp, ref, w, coefs, cap=100)  # truncated output, full count


def test_extend_parity_config2_shape_and_many_blocks(zp, ref):
    w = wl.config(2, F=64)  # 64 000 terms: 250 blocks, B = 21, one non-zero degree per term
    both(zp, ref, w, w.planted)
    w3 = wl.config(3, t=20000, dense=True)  # one function, every coefficient non-zero: 180 000 new terms
    both(zp, ref, w3, w3.planted)


def test_two_step_chain_on_the_gpu(zp, ref):
    """planted sparse f(x1..x4): lift 2 -> 3 variables, extend, lift 3 -> 4; the result equals the planted
    polynomial.  Probe values: the oracle's forward evaluation of the planted polynomial."""
    import itertools
    import random
    import torch

    p = wl.P63
    rng = random.Random(12)
    terms = {}
    while len(terms) < 120:
        terms[(rng.randrange(6), rng.randrange(6), rng.randrange(4), rng.randrange(3))] = rng.randrange(1, p)
    full_exps = np.array(list(terms.keys()), dtype=np.uint16)
    full_coef = np.array(list(terms.values()), dtype=np.uint64)
    anchors = np.array([rng.randrange(2, p) for _ in range(3)], dtype=np.uint64)
    c3 = np.array(rng.sample(range(2, p), 4), dtype=np.uint64)
    c4 = np.array(rng.sample(range(2, p), 3), dtype=np.uint64)

    def probes(nv, t, cs, fixed_tail):
        """values f(y_1^s, .., y_nv^s, c_j, fixed_tail...) for s < t, j < len(cs) via the oracle's sparse evaluation"""
        out = np.empty((len(cs), t), dtype=np.uint64)
        for j, cj in enumerate(cs):
            for s in range(t):
                pt = [pow(int(a), s, p) for a in anchors[:nv]] + [int(cj)] + fixed_tail
                out[j, s] = ref.eval_sparse(full_exps, full_coef, np.array(pt, dtype=np.uint64), p)
        return out

    skel2 = sorted({(k[0], k[1]) for k in terms})
    exps = np.array(skel2, dtype=np.uint16)
    offsets = np.array([0, len(skel2)], dtype=np.int64)
    vals = probes(2, len(skel2), c3, [int(c4[0])])
    out, st = zp.zippel_lift_step(zp.to_dev(exps), offsets, zp.to_dev(anchors[:2]), zp.to_dev(c3), zp.to_dev(vals), p, 0, 1)
    ne, nc, no, degs = zp.zippel_extend_skeleton(zp.to_dev(exps), offsets, out, p)
    torch.cuda.synchronize()
    assert not zp.to_host(st).any()
    no = no.cpu().numpy()
    t3 = int(no[-1])
    ne3 = ne[:t3].contiguous()
    assert {tuple(r) for r in zp.to_host(ne3).tolist()} == {(k[0], k[1], k[2]) for k in terms}
    vals2 = probes(3, t3, c4, [])
    out2, st2 = zp.zippel_lift_step(ne3, no, zp.to_dev(anchors), zp.to_dev(c4), zp.to_dev(vals2), p, 0, 1)
    ne4, nc4, no4, degs4 = zp.zippel_extend_skeleton(ne3, no, out2, p)
    torch.cuda.synchronize()
    assert not zp.to_host(st2).any()
    t4 = int(no4.cpu().numpy()[-1])
    got = {tuple(r): int(c) for r, c in zip(zp.to_host(ne4[:t4].contiguous()).tolist(), zp.to_host(nc4[:t4]).tolist())}
    assert got == terms
    assert int(degs4.cpu().numpy()[0]) == max(k[3] for k in terms)


@pytest.mark.parametrize("nv,ts", [(12, [700, 3, 2049, 1]),              # wide rows: the staging buffer is off
                                   (2, [5, 4096, 1, 1, 2047, 3]),         # odd total: the scalar load path
                                   (3, None)])                            # thousands of tiny functions per block
def test_extend_block_boundaries_wide_rows_and_tiny_functions(zp, ref, nv, ts):
    """The single-pass kernel's corners: functions that start at, just before and just after a 2048-term block, more
    function starts in one block than lanes, rows too wide for the shared-memory staging, an odd number of terms (rows
    not 16-byte aligned), sparse and dense coefficients."""
    if ts is None:
        r = np.random.Generator(np.random.Philox(key=[10, 977]))
        ts = [int(x) for x in r.integers(1, 4, 6000)]
    for dense in (False, True):
        w = wl.make_box_workload("extb", wl.SEED_BASE + 95 + nv, len(ts), nv, ts, 80, 5, dense=dense)
        coefs = w.planted.copy()
        coefs[:, ::7] = 0  # vanished terms scattered over the batch
        both(zp, ref, w, coefs)
