"""Bit-exact parity of the CUDA Thiele reconstruction (thiele_reconstruct_batch through the C-ABI) with the CPU
oracle (oracle/zippel_ref.c, pinned by tests/test_thiele_oracle_pins.py) on the same seeded inputs: planted
rational functions of mixed degrees in one batch (columns end at different K: lanes diverge), arbitrary values
(K = T), several CTAs and a ragged tail, small and large primes, degenerate columns, duplicate points."""
import random

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

P63 = (1 << 63) - 25


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


def peval(c, x, p):
    r = 0
    for a in reversed(c):
        r = (r * x + a) % p
    return r


def planted_columns(rng, T, n, p, max_deg):
    """Columns of values of random rational functions with degrees up to max_deg (generator data only: Python
    integers; no oracle, no CUDA)."""
    pts = rng.sample(range(p), T)
    cols = []
    while len(cols) < n:
        dn, dd = rng.randrange(-1, max_deg + 1), rng.randrange(0, max_deg + 1)
        P = [rng.randrange(p) for _ in range(dn)] + [rng.randrange(1, p)] if dn >= 0 else []
        Q = [rng.randrange(p) for _ in range(dd)] + [1]
        if any(peval(Q, x, p) == 0 for x in pts):
            continue
        cols.append([(peval(P, x, p) * pow(peval(Q, x, p), -1, p)) % p for x in pts])
    return np.array(pts, dtype=np.uint64), np.array(cols, dtype=np.uint64).T.copy()


def both(zp, ref, pts, vals, p):
    wn, wd, wdeg, wcf, wst = ref.thiele_reconstruct_batch(pts, vals, p)
    gn, gd, gdeg, gcf, gst = zp.thiele_reconstruct_batch(zp.to_dev(pts), zp.to_dev(vals), p)
    assert (zp.to_host(gst) == wst).all()
    assert (gdeg.cpu().numpy() == wdeg).all()
    assert (zp.to_host(gn.contiguous()) == wn).all() and (zp.to_host(gd.contiguous()) == wd).all()
    assert (zp.to_host(gcf.contiguous()) == wcf).all()
    return wst, wdeg


@pytest.mark.parametrize("p", [101, (1 << 31) - 1, P63])
@pytest.mark.parametrize("T,max_deg", [(1, 0), (2, 0), (3, 1), (8, 3), (9, 4), (33, 12), (64, 31)])
def test_thiele_parity_planted_mixed_degrees(zp, ref, p, T, max_deg):
    if p == 101 and T > 33:
        pytest.skip("mod 101 has too few points")
    rng = random.Random(T * 7 + p % 11)
    pts, vals = planted_columns(rng, T, 64 * 3 + 17, p, max_deg)
    st, deg = both(zp, ref, pts, vals, p)
    if p > 101:
        assert not st.any() and len(set(deg[1].tolist())) > (1 if max_deg else 0)


@pytest.mark.parametrize("T", [5, 24, 50])
def test_thiele_parity_arbitrary_values_full_length(zp, ref, T):
    """no low-degree function behind the values: K = T in every column (the cost model's case)"""
    p = P63
    r = np.random.Generator(np.random.Philox(key=[77, T]))
    pts = np.array(random.Random(T).sample(range(p), T), dtype=np.uint64)
    vals = r.integers(0, p, (T, 1000), dtype=np.uint64)
    st, deg = both(zp, ref, pts, vals, p)
    assert not st.any() and (deg[0] == T // 2).all() and (deg[1] == (T - 1) // 2).all()


def test_thiele_status_degenerate_duplicate_and_strided_input(zp, ref):
    import torch

    p = P63
    pts = np.array([1, 2, 3, 4], dtype=np.uint64)
    vals = np.array([[5, 5, 0], [5, 6, 0], [9, 7, 0], [11, 8, 0]], dtype=np.uint64)
    st, _ = both(zp, ref, pts, vals, p)
    assert st[0] == ((1 << 8) | zp.ST_THIELE_DEGENERATE) and st[1] == 0 and st[2] == 0
    st, _ = both(zp, ref, np.array([1, 2, 1, 4], dtype=np.uint64), vals, p)
    assert (st == ((2 << 8) | zp.ST_DUPLICATE_SAMPLE)).all()
    # a view with leading dimension > n
    rng = random.Random(9)
    pts, full = planted_columns(rng, 7, 40, p, 3)
    dv = zp.to_dev(full)[:, :29]
    gn, gd, gdeg, gcf, gst = zp.thiele_reconstruct_batch(zp.to_dev(pts), dv, p)
    wn, wd, wdeg, wcf, wst = ref.thiele_reconstruct_batch(pts, np.ascontiguousarray(full[:, :29]), p)
    torch.cuda.synchronize()
    assert (zp.to_host(gn.contiguous()) == wn).all() and (zp.to_host(gd.contiguous()) == wd).all()
    assert (gdeg.cpu().numpy() == wdeg).all() and (zp.to_host(gst) == wst).all()
