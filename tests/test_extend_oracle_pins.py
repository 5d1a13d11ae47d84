"""Pins of the oracle's skeleton extension against things other than itself:
numpy's nonzero, the polynomial identity  sum_d x_k^d sum_i c_{d,i} mono_i(x) == sum_new c' mono'(x, x_k)  in Python
integers, and a two-step chain 1 -> 2 -> 3 variables that recovers a planted sparse polynomial exactly."""
import random

import numpy as np

from oracle import ref
from paper_2505_24256_b200 import workloads as wl

P63 = wl.P63


def sparse_eval(exps, coef, point, p):
    tot = 0
    for row, c in zip(exps, coef):
        term = int(c)
        for e, z in zip(row, point):
            term = term * pow(int(z), int(e), p) % p
        tot += term
    return tot % p


def test_extend_matches_numpy_nonzero_and_is_the_same_polynomial():
    w = wl.make_box_workload("ext", wl.SEED_BASE + 91, 4, 3, [17, 1, 40, 9], 5, 6)  # sparse law: one d per term
    dense = wl.make_box_workload("ext", wl.SEED_BASE + 92, 4, 3, [17, 1, 40, 9], 5, 6, dense=True)
    for ww in (w, dense):
        coefs = ww.planted.copy()
        coefs[3, 5] = 0
        coefs[:, 20] = 0  # a term that vanishes altogether disappears from the skeleton
        coefs[5, :17] = 0  # function 0 has degree < B - 1
        ne, nc, no, degs = ref.extend_skeleton(ww.exps, ww.offsets, coefs, ww.p)
        nz_d, nz_i = np.nonzero(coefs.T.T)  # rows d, columns i
        order = np.lexsort((nz_d, nz_i))  # i ascending, then d ascending
        assert len(nc) == len(order) == no[-1]
        assert (nc == coefs[nz_d[order], nz_i[order]]).all()
        assert (ne[:, :-1] == ww.exps[nz_i[order]]).all() and (ne[:, -1] == nz_d[order]).all()
        for f in range(ww.F):
            a, b = ww.offsets[f], ww.offsets[f + 1]
            assert no[f] == np.count_nonzero(coefs[:, :a])
            rows = np.nonzero(coefs[:, a:b].any(axis=1))[0]
            assert degs[f] == (rows.max() if len(rows) else -1)
        rng = random.Random(3)
        z = [rng.randrange(2, ww.p) for _ in range(ww.nv + 1)]
        for f in range(ww.F):
            a, b = ww.offsets[f], ww.offsets[f + 1]
            old = sum(pow(z[-1], d, ww.p) * sparse_eval(ww.exps[a:b], coefs[d, a:b], z[:-1], ww.p) for d in range(ww.B))
            new = sparse_eval(ne[no[f]:no[f + 1]], nc[no[f]:no[f + 1]], z, ww.p)
            assert old % ww.p == new
    # capacity: the count is still reported, nothing is written past cap
    ne, nc, no, _ = ref.extend_skeleton(w.exps, w.offsets, w.planted, w.p, cap=5)
    assert no[-1] == np.count_nonzero(w.planted) and len(nc) == 5


def test_two_step_chain_recovers_a_planted_polynomial():
    """f(x1, x2, x3) sparse, planted.  Step 1 lifts the x1-skeleton to (x1, x2); its extension is the skeleton of
    step 2, which lifts to (x1, x2, x3).  Probe values come from Python integers only."""
    p = P63
    rng = random.Random(8)
    terms = {}
    while len(terms) < 30:
        terms[(rng.randrange(5), rng.randrange(4), rng.randrange(4))] = rng.randrange(1, p)
    full_exps = np.array(list(terms.keys()), dtype=np.uint16)
    full_coef = np.array(list(terms.values()), dtype=np.uint64)
    f = lambda pt: sparse_eval(full_exps, full_coef, pt, p)
    y1 = rng.randrange(2, p)
    c2 = [rng.randrange(2, p) for _ in range(4)]  # samples of x2 (degree <= 3), c2[0] = the skeleton's value
    c3 = [rng.randrange(2, p) for _ in range(4)]
    # step 0: the univariate skeleton in x1 at (x2, x3) = (c2[0], c3[0]): exponents of x1 that occur
    e1 = sorted({k[0] for k in terms})
    exps = np.array([[e] for e in e1], dtype=np.uint16)
    offsets = np.array([0, len(e1)], dtype=np.int64)
    # step 1: lift x2.  probes at x1 = y1^s, x2 = c2[j], x3 = c3[0]
    vals = np.array([[f([pow(y1, s, p), cj, c3[0]]) for s in range(len(e1))] for cj in c2], dtype=np.uint64)
    out, _, st = ref.zippel_lift_step(exps, offsets, np.array([y1], dtype=np.uint64), np.array(c2, dtype=np.uint64), vals, p, 0, 1)
    assert not st.any()
    ne, nc, no, degs = ref.extend_skeleton(exps, offsets, out, p)
    assert {tuple(r) for r in ne.tolist()} == {(k[0], k[1]) for k in terms}  # generic c3[0]: no accidental cancellation
    # step 2: lift x3 with the extended skeleton; anchors (y1, y2)
    y2 = rng.randrange(2, p)
    t2 = len(nc)
    vals2 = np.array([[f([pow(y1, s, p), pow(y2, s, p), cj]) for s in range(t2)] for cj in c3], dtype=np.uint64)
    out2, _, st2 = ref.zippel_lift_step(ne, no, np.array([y1, y2], dtype=np.uint64), np.array(c3, dtype=np.uint64), vals2, p, 0, 1)
    assert not st2.any()
    ne3, nc3, no3, _ = ref.extend_skeleton(ne, no, out2, p)
    got = {tuple(r): int(c) for r, c in zip(ne3.tolist(), nc3.tolist())}
    assert got == {k: v for k, v in terms.items()}
