"""Pins of the oracle's Thiele reconstruction (eq. (2)) against things other
than itself: planted rational functions recovered exactly, the interpolation property, cross-multiplied fresh
probes, closed forms over Q, and an independent continued-fraction EVALUATION in Python integers (the oracle's
b_k are plugged into eq. (2) as printed in the paper and must reproduce the inputs)."""
import random
from fractions import Fraction

import numpy as np
import pytest

from oracle import ref

P63 = (1 << 63) - 25
ST_DUP, ST_DEG = 17, 20


def peval(c, x, p):
    r = 0
    for a in reversed([int(v) for v in c]):
        r = (r * x + a) % p
    return r


def planted(rng, dn, dd, p):
    """P of degree exactly dn (dn = -1: zero), Q monic of degree dd, random coefficients."""
    P = [rng.randrange(p) for _ in range(dn)] + [rng.randrange(1, p)] if dn >= 0 else []
    Q = [rng.randrange(p) for _ in range(dd)] + [1]
    return P, Q


def values(P, Q, pts, p):
    return [(peval(P, x, p) * pow(peval(Q, x, p), -1, p)) % p for x in pts]


def thiele_eval_eq2(b, pts, x, p):
    """eq. (2) as printed: b_0 + (x - x_0)[b_1 + (x - x_1)[b_2 + ...]^-1]^-1, evaluated from the tail."""
    K = len(b)
    r = b[K - 1]
    for k in range(K - 2, -1, -1):
        r = (b[k] + (x - pts[k]) * pow(r, -1, p)) % p
    return r


@pytest.mark.parametrize("p", [101, (1 << 31) - 1, P63])
@pytest.mark.parametrize("dn,dd", [(0, 0), (3, 0), (0, 1), (1, 1), (2, 3), (5, 2), (4, 4), (-1, 0)])
def test_thiele_recovers_planted_rational_functions(p, dn, dd):
    rng = random.Random(1000 * dn + 10 * dd + p % 7)
    n = 6
    T = 2 * max(dn, dd, 0) + 2 + (dn + dd) % 3  # enough points to see the fraction terminate, sometimes more
    if p == 101 and T > 12:
        pytest.skip("not enough room for generic points mod 101")
    cols, truth = [], []
    pts = None
    for _ in range(400):  # points at which no planted denominator vanishes and no accidental degeneracy occurs
        pts = rng.sample(range(p), T)
        cols, truth = [], []
        ok = True
        for _ in range(n):
            P, Q = planted(rng, dn, dd, p)
            if any(peval(Q, x, p) == 0 for x in pts):
                ok = False
                break
            truth.append((P, Q))
            cols.append(values(P, Q, pts, p))
        if not ok:
            continue
        vals = np.array(cols, dtype=np.uint64).T.copy()
        num, den, degs, cf, st = ref.thiele_reconstruct_batch(np.array(pts, dtype=np.uint64), vals, p)
        if not st.any():
            break
    assert not st.any()
    for i, (P, Q) in enumerate(truth):
        # a planted pair may share a factor by accident only with negligible probability at these sizes mod 2^31, 2^63;
        # mod 101 compare as functions instead
        N = [int(v) for v in num[:, i]]
        D = [int(v) for v in den[:, i]]
        dN, dD = int(degs[0, i]), int(degs[1, i])
        assert dD >= 0 and D[dD] == 1 and all(v == 0 for v in D[dD + 1:]) and all(v == 0 for v in N[dN + 1:])
        if p > 101:
            assert dN == dn and dD == dd
            assert N[:dn + 1] == P and D[:dd + 1] == Q
        for _ in range(5):  # fresh probes, cross-multiplied
            z = rng.randrange(p)
            assert (peval(N, z, p) * peval(Q, z, p) - peval(P, z, p) * peval(D, z, p)) % p == 0


def test_thiele_interpolates_and_matches_eq2_as_printed():
    """Arbitrary values (no underlying low-degree function): K = T, the expanded N/D and eq. (2) evaluated in
    Python integers with the oracle's b_k both reproduce every input value."""
    p = P63
    rng = random.Random(5)
    T, n = 9, 8
    pts = rng.sample(range(p), T)
    vals = np.array([[rng.randrange(p) for _ in range(n)] for _ in range(T)], dtype=np.uint64)
    num, den, degs, cf, st = ref.thiele_reconstruct_batch(np.array(pts, dtype=np.uint64), vals, p)
    assert not st.any()
    for i in range(n):
        b = [int(v) for v in cf[:, i]]
        assert degs[0, i] == T // 2 and degs[1, i] == (T - 1) // 2
        for j in range(T):
            f = int(vals[j, i])
            assert (peval(num[:, i], pts[j], p) - f * peval(den[:, i], pts[j], p)) % p == 0
            if j >= 1:  # at x = x_k the tail below level k is multiplied by zero; avoid 0 * inverse-of-0 in the check
                continue
        for _ in range(3):
            z = rng.randrange(p)
            lhs = thiele_eval_eq2(b, pts, z, p)
            assert (lhs * peval(den[:, i], z, p) - peval(num[:, i], z, p)) % p == 0


def test_thiele_closed_forms_over_Q():
    """f = 1/(x - a) and f = (x + 1)/(x + 2) at small integer points: continued-fraction coefficients computed
    with exact rationals, reduced mod p, equal the oracle's."""
    p = P63
    for f, pts in ((lambda x: Fraction(1, x - 20), [1, 2, 3, 4]), (lambda x: Fraction(x + 1, x + 2), [0, 1, 3, 7, 8])):
        T = len(pts)
        phi = [f(x) for x in pts]
        b = [phi[0]]
        K = T
        for k in range(1, T):
            if all(phi[j] == phi[k - 1] for j in range(k, T)):
                K = k
                break
            for j in range(T - 1, k - 1, -1):
                phi[j] = Fraction(pts[j] - pts[k - 1]) / (phi[j] - phi[k - 1])
            b.append(phi[k])
        modp = lambda q: (q.numerator % p) * pow(q.denominator % p, -1, p) % p
        vals = np.array([[modp(f(x))] for x in pts], dtype=np.uint64)
        num, den, degs, cf, st = ref.thiele_reconstruct_batch(np.array(pts, dtype=np.uint64), vals, p)
        assert st[0] == 0
        assert [int(v) for v in cf[:K, 0]] == [modp(x) for x in b[:K]] and not cf[K:, 0].any()
        assert degs[0, 0] <= 1 and degs[1, 0] == 1
    # 1/(x - 20): N = 1, D = x - 20
    vals = np.array([[pow((x - 20) % p, -1, p)] for x in [1, 2, 3, 4]], dtype=np.uint64)
    num, den, degs, cf, st = ref.thiele_reconstruct_batch(np.array([1, 2, 3, 4], dtype=np.uint64), vals, p)
    assert [int(v) for v in num[:, 0]] == [1, 0, 0, 0] and [int(v) for v in den[:, 0]] == [p - 20, 1, 0, 0]


def test_thiele_single_point_and_status_codes():
    p = P63
    num, den, degs, cf, st = ref.thiele_reconstruct_batch(np.array([7], dtype=np.uint64), np.array([[42, 0]], dtype=np.uint64), p)
    assert [int(num[0, 0]), int(den[0, 0]), int(degs[0, 0]), int(degs[1, 0])] == [42, 1, 0, 0]
    assert [int(num[0, 1]), int(den[0, 1]), int(degs[0, 1]), int(degs[1, 1])] == [0, 1, -1, 0] and not st.any()
    # f(x_0) = f(x_1) != f(x_2): the first inverse difference has a zero denominator at one point only
    vals = np.array([[5, 5], [5, 6], [9, 7], [11, 8]], dtype=np.uint64)
    _, _, _, _, st = ref.thiele_reconstruct_batch(np.array([1, 2, 3, 4], dtype=np.uint64), vals, p)
    assert st[0] == ((1 << 8) | ST_DEG) and st[1] == 0
    _, _, _, _, st = ref.thiele_reconstruct_batch(np.array([1, 2, 1, 4], dtype=np.uint64), vals, p)
    assert (st == ((2 << 8) | ST_DUP)).all()
