"""Pins of the CPU oracle (oracle/zippel_ref.c) against things other than itself: Python big
integers, closed forms, Vieta, exact interpolation over Q, an independent Python Gauss-Jordan,
planted recovery, fresh probes, and the golden worked example (tests/golden/worked_example.json,
written by tests/golden/make_worked_example.py with Python big integers only).

Every check is chosen so that a plausible slip in the oracle (dropped term, wrong sign or index,
transposed operand, off-by-one in a loop bound) fails at least one of them.  CPU only.
"""
import itertools
import json
import math
import os
import random
from fractions import Fraction

import numpy as np
import pytest

from oracle import ref
from paper_2505_24256_b200 import workloads as wl

P63 = (1 << 63) - 25
PRIMES = [101, 65537, (1 << 31) - 1, (1 << 61) - 1, P63]
GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_example.json")


def rnd(p, n, seed, lo=0):
    r = random.Random(seed)
    return [r.randrange(lo, p) for _ in range(n)]


# ---------------------------------------------------------------------------- prime (north_star)
def test_prime_is_2_63_minus_25():
    assert ref.largest_prime_below(1 << 63) == P63 == 9223372036854775783 == 0x7FFFFFFFFFFFFFE7
    assert P63 % 8 == 7
    for c in range(1, 25):  # everything between is composite: find a factor or fail Fermat base 2
        n = (1 << 63) - c
        assert not ref.is_prime(n)
        assert pow(2, n - 1, n) != 1 or any(n % q == 0 for q in range(2, 10000))


def test_miller_rabin_vs_sieve_and_pseudoprimes():
    N = 20000
    sieve = bytearray([1]) * N
    sieve[0] = sieve[1] = 0
    for i in range(2, int(N**0.5) + 1):
        if sieve[i]:
            sieve[i * i::i] = bytearray(len(sieve[i * i::i]))
    for n in range(N):
        assert ref.is_prime(n) == bool(sieve[n]), n
    # Carmichael numbers and strong pseudoprimes to small base sets must be rejected
    for n in (561, 1105, 1729, 2047, 3215031751, 3474749660383, 341550071728321, 3825123056546413051):
        assert not ref.is_prime(n), n
    for n in ((1 << 61) - 1, (1 << 31) - 1, 18446744073709551557, 2305843009213693951):
        assert ref.is_prime(n), n
    # p - 1 factorisation quoted in SURVEY.md appendix (no 2-power NTT modulo p)
    assert P63 - 1 == 2 * 3**4 * 17 * 23 * 319279 * 456065899


# ---------------------------------------------------------------------------- arithmetic (L88-100)
@pytest.mark.parametrize("p", PRIMES)
def test_modular_arithmetic_vs_python(p):
    edge = [0, 1, 2, p - 1, p - 2, p // 2, p // 2 + 1, (1 << 32) - 1, 1 << 32, (1 << 32) + 1, 0xFFFFFFFF00000000,
            0x00000000FFFFFFFF, 0x7FFFFFFF7FFFFFFF]
    edge = sorted({e % p for e in edge})
    vals = edge + rnd(p, 200, 1)
    for a, b in itertools.product(edge, edge):
        assert ref.mulmod(a, b, p) == a * b % p
    r = random.Random(2)
    for _ in range(3000):
        a, b = r.choice(vals), r.choice(vals)
        assert ref.mulmod(a, b, p) == a * b % p
        assert ref.addmod(a, b, p) == (a + b) % p
        assert ref.submod(a, b, p) == (a - b) % p
    for a in vals[:60]:
        e = r.randrange(0, 1 << 63)
        assert ref.powmod(a, e, p) == pow(a, e, p)
        assert ref.powmod(a, 0, p) == 1
        if a:
            assert ref.invmod(a, p) == pow(a, -1, p)
            assert ref.powmod(a, p - 1, p) == 1  # Fermat
    assert ref.mulmod(p - 1, p - 1, p) == 1


def test_montgomery_constants_quoted_in_survey():
    # constants the CUDA side's tests use; derived here with Python only
    p = P63
    assert pow(2, 64, p) == 50 and pow(2, 128, p) == 2500
    assert (-pow(p, -1, 1 << 64)) % (1 << 64) == 1106804644422573097
    assert (-pow(p, -1, 1 << 32)) % (1 << 32) == 3264175145


# ---------------------------------------------------------------------------- nodes (eq. 3)
@pytest.mark.parametrize("p", [101, P63])
def test_nodes_vs_python_pow(p):
    r = np.random.default_rng(3)
    nv, T = 5, 300
    exps = r.integers(0, 41, size=(T, nv)).astype(np.uint16)
    exps[0] = 0
    exps[1] = 65535 if p == P63 else 40
    anchors = np.array(rnd(p, nv, 4, lo=2), dtype=np.uint64)
    got = ref.eval_nodes(exps, anchors, p)
    for i in range(T):
        want = 1
        for j in range(nv):
            want = want * pow(int(anchors[j]), int(exps[i, j]), p) % p
        assert int(got[i]) == want
    assert int(got[0]) == 1


# ---------------------------------------------------------------------------- master polynomial (L191)
@pytest.mark.parametrize("p,t", [(101, 7), (P63, 1), (P63, 2), (P63, 33), ((1 << 61) - 1, 64)])
def test_master_poly_vieta_roots_and_random_point(p, t):
    m = rnd(p, t, 5)
    M = [int(x) for x in ref.master_poly(m, p)]
    assert len(M) == t + 1 and M[t] == 1
    assert M[t - 1] == (-sum(m)) % p
    assert M[0] == (-1) ** t * math.prod(m) % p
    if t >= 2:  # second elementary symmetric function
        e2 = sum(a * b for a, b in itertools.combinations(m, 2))
        assert M[t - 2] == e2 % p
    ev = lambda z: sum(c * pow(z, l, p) for l, c in enumerate(M)) % p
    for mi in m:
        assert ev(mi) == 0
    for z in rnd(p, 5, 6):
        assert ev(z) == math.prod((z - mi) for mi in m) % p


# ---------------------------------------------------------------------------- quotient, den (L193-196, G15)
@pytest.mark.parametrize("p,t", [(101, 6), (P63, 1), (P63, 17)])
def test_quotient_times_linear_factor_is_master_and_den_is_product(p, t):
    m = random.Random(7).sample(range(2, min(p, 1 << 62)), t) if p > 200 else random.Random(7).sample(range(1, p), t)
    M = ref.master_poly(m, p)
    Mi = [int(x) for x in M]
    vals = np.array([rnd(p, t, 8), rnd(p, t, 9)], dtype=np.uint64)
    den, num = ref.node_solve(m, M, vals, p)
    for i, mi in enumerate(m):
        q = [int(x) for x in ref.node_quotient(M, mi, p)]
        assert q[t - 1] == 1
        prod = [0] * (t + 1)  # Q_i(z) (z - m_i), big integers
        for l, c in enumerate(q):
            prod[l + 1] += c
            prod[l] -= c * mi
        assert [x % p for x in prod] == Mi
        want_den = math.prod((mi - mj) for j, mj in enumerate(m) if j != i) % p
        assert int(den[i]) == want_den
        for b in range(2):
            assert int(num[b, i]) == sum(q[s] * int(vals[b, s]) for s in range(t)) % p


@pytest.mark.parametrize("p,t", [(101, 7), (P63, 1), (P63, 23)])
def test_node_solve_at_sampled_nodes_and_arbitrary_points(p, t):
    """ref_node_solve_at (the per-node routine on caller-chosen node values) against Python
    integers: at a root m_i of M, den = prod_{j != i}(m_i - m_j) and num_b = sum_s q_{i,s} v_{b,s} with the quotient
    defined by Q_i(z)(z - m_i) = M(z); at a non-root x the quotient of the division with remainder."""
    rr = random.Random(70 + t)
    m = rr.sample(range(1, p), t) if p < 200 else rr.sample(range(2, 1 << 62), t)
    M = ref.master_poly(m, p)
    Mi = [int(x) for x in M]
    vals = np.array([rnd(p, t, 18), rnd(p, t, 19), rnd(p, t, 20)], dtype=np.uint64)
    pick = [t - 1, 0, t // 2][: min(t, 3)]
    extra = [x for x in rnd(p, 3, 71) if x not in m]
    xs = [m[i] for i in pick] + extra
    den, num = ref.node_solve_at(xs, M, vals, p)
    assert den.shape == (len(xs),) and num.shape == (3, len(xs))
    for k, x in enumerate(xs):
        q = [0] * t  # synthetic division of M by (z - x) in big integers: q_{t-1} = 1, q_{l-1} = M_l + x q_l
        q[t - 1] = 1
        for l in range(t - 1, 0, -1):
            q[l - 1] = Mi[l] + x * q[l]
        rem = Mi[0] + x * q[0]
        assert (rem % p == 0) == (x in m)
        if x in m:
            assert int(den[k]) == math.prod((x - mj) for mj in m if mj != x) % p
        assert int(den[k]) == sum(c * pow(x, l, p) for l, c in enumerate(q)) % p  # Q_x(x)
        for b in range(3):
            assert int(num[b, k]) == sum(q[s] * int(vals[b, s]) for s in range(t)) % p
    if t > 1:  # on all the nodes it is ref_node_solve's answer
        d_all, n_all = ref.node_solve(m, M, vals, p)
        d_at, n_at = ref.node_solve_at(m, M, vals, p)
        assert (d_all == d_at).all() and (n_all == n_at).all()


# ---------------------------------------------------------------------------- solve (L60, L191-197)
def py_gauss(A, b, p):
    n = len(A)
    A = [row[:] + [bi] for row, bi in zip(A, b)]
    for c in range(n):
        piv = next(r for r in range(c, n) if A[r][c] % p)
        A[c], A[piv] = A[piv], A[c]
        inv = pow(A[c][c], -1, p)
        A[c] = [x * inv % p for x in A[c]]
        for r in range(n):
            if r != c and A[r][c]:
                f = A[r][c]
                A[r] = [(x - f * y) % p for x, y in zip(A[r], A[c])]
    return [A[i][n] for i in range(n)]


@pytest.mark.parametrize("s0", [0, 1])
@pytest.mark.parametrize("p,ts", [(101, [5, 1, 9]), (P63, [1, 2, 13, 40]), (65537, [24])])
def test_solve_vs_python_gauss_residual_and_oracle_gauss(p, ts, s0):
    r = random.Random(10 + s0)
    offsets = np.concatenate([[0], np.cumsum(ts)]).astype(np.int64)
    nodes = []
    for t in ts:
        nodes += r.sample(range(1, p if p < 1 << 40 else 1 << 62), t)
    B = 3
    vals = np.array([[r.randrange(p) for _ in range(offsets[-1])] for _ in range(B)], dtype=np.uint64)
    coefs, status = ref.vandermonde_solve_batch(nodes, offsets, vals, p, s0)
    assert not status.any()
    for f, t in enumerate(ts):
        o = int(offsets[f])
        m = nodes[o:o + t]
        A = [[pow(mi, s + s0, p) for mi in m] for s in range(t)]
        for b in range(B):
            v = [int(x) for x in vals[b, o:o + t]]
            c = [int(x) for x in coefs[b, o:o + t]]
            assert c == py_gauss(A, v, p)  # independent Python elimination
            for s in range(t):  # residual: sum_i c_i m_i^(s+s0) = v_s
                assert sum(ci * A[s][i] for i, ci in enumerate(c)) % p == v[s]
            g = ref.gauss_solve(m, v, p, s0)  # the oracle's own O(t^3) route
            assert [int(x) for x in g] == c


def test_solve_closed_forms_t1_t2():
    p = P63
    m1, m2, v0, v1 = rnd(p, 4, 11, lo=2)
    c, st = ref.vandermonde_solve_batch([m1], [0, 1], [[v0]], p)
    assert int(c[0, 0]) == v0 and st[0] == 0
    c, st = ref.vandermonde_solve_batch([m1, m2], [0, 2], [[v0, v1]], p)
    c1 = (v1 - m2 * v0) * pow(m1 - m2, -1, p) % p
    assert [int(c[0, 0]), int(c[0, 1])] == [c1, (v0 - c1) % p]
    c, st = ref.vandermonde_solve_batch([m1], [0, 1], [[v0]], p, s0=1)
    assert int(c[0, 0]) == v0 * pow(m1, -1, p) % p


def test_solve_t64_gauss_crosscheck():
    # north_star: "a naive O(t^3) Gaussian-elimination Vandermonde solver for t <= 64 as a brute-force cross-check"
    p = P63
    m = random.Random(12).sample(range(2, 1 << 62), 64)
    v = rnd(p, 64, 13)
    c, st = ref.vandermonde_solve_batch(m, [0, 64], [v], p)
    g = ref.gauss_solve(m, v, p)
    assert st[0] == 0 and (c[0] == g).all()
    assert all(sum(int(ci) * pow(mi, s, p) for ci, mi in zip(c[0], m)) % p == v[s] for s in (0, 1, 31, 63))


def test_solve_status_duplicate_and_zero_node():
    p = P63
    c, st = ref.vandermonde_solve_batch([5, 7, 5, 9, 11, 12], [0, 4, 6], [[1, 2, 3, 4, 5, 6]], p)
    assert st[0] & 0xFF == ref.ST_DUPLICATE_NODE and (st[0] >> 8) in (0, 2) and st[1] == 0
    c, st = ref.vandermonde_solve_batch([0, 7], [0, 2], [[1, 2]], p, s0=0)
    assert st[0] == 0  # one zero node is fine with s0 = 0 (reading G25)
    c, st = ref.vandermonde_solve_batch([7, 0], [0, 2], [[1, 2]], p, s0=1)
    assert st[0] == ((1 << 8) | ref.ST_DUPLICATE_NODE)
    assert ref.gauss_solve([5, 7, 5], [1, 2, 3], p) is None


def test_deferred_reduction_identity_L208():
    # reducing every product and partial sum == one reduction of the integer sum
    p = P63
    a, b = rnd(p, 1000, 14), rnd(p, 1000, 15)
    step = 0
    for x, y in zip(a, b):
        step = ref.addmod(step, ref.mulmod(x, y, p), p)
    total = sum(x * y for x, y in zip(a, b))
    assert total < 1 << 192 and step == total % p


# ---------------------------------------------------------------------------- Newton (eq. 1)
def newton_eval(a, xs, x, p):
    r = 0
    for j in range(len(a) - 1, -1, -1):
        r = (r * (x - xs[j]) + a[j]) % p
    return r


@pytest.mark.parametrize("p,B", [(101, 4), (P63, 1), (P63, 2), (P63, 9), (P63, 26)])
def test_newton_reproduces_inputs_and_is_exact_on_planted(p, B):
    r = random.Random(16)
    xs = r.sample(range(2, p), B)
    n = 7
    planted = [[r.randrange(p) for _ in range(n)] for _ in range(B)]  # row d: coefficient of x^d
    vals = [[sum(planted[d][i] * pow(x, d, p) for d in range(B)) % p for i in range(n)] for x in xs]
    assert (ref.poly_rows_eval(xs, planted, p) == np.array(vals, dtype=np.uint64)).all()
    a, st = ref.newton_interp_batch(xs, vals, p, basis=0)
    mono, st1 = ref.newton_interp_batch(xs, vals, p, basis=1)
    assert st == 0 and st1 == 0
    assert (mono == np.array(planted, dtype=np.uint64)).all()  # exact on a degree-D polynomial
    for i in range(n):
        ai = [int(a[j, i]) for j in range(B)]
        assert ai[0] == vals[0][i]  # a_0 = f(c_0)
        for j, x in enumerate(xs):  # eq. (1) reproduces every input
            assert newton_eval(ai, xs, x, p) == vals[j][i]
        z = r.randrange(p)  # and agrees with the planted polynomial at a fresh point
        assert newton_eval(ai, xs, z, p) == sum(planted[d][i] * pow(z, d, p) for d in range(B)) % p
        if B >= 2:  # D = 1 closed form for the first divided difference
            assert ai[1] == (vals[1][i] - vals[0][i]) * pow(xs[1] - xs[0], -1, p) % p


def test_newton_vs_exact_lagrange_over_Q():
    # small integer data: interpolate exactly over Q with Fractions, then map to Z/pZ
    p = P63
    xs = [2, 3, 5, 7, 11]
    ys = [4, -9, 25, 3, 8]
    B = len(xs)
    coeffs = [Fraction(0)] * B
    for j in range(B):
        basis = [Fraction(1)]
        den = Fraction(1)
        for k in range(B):
            if k != j:
                basis = [Fraction(0)] + basis
                for d in range(len(basis) - 1):
                    basis[d] -= xs[k] * basis[d + 1]
                den *= xs[j] - xs[k]
        for d in range(B):
            coeffs[d] += ys[j] * basis[d] / den
    want = [c.numerator * pow(c.denominator, -1, p) % p for c in coeffs]
    mono, st = ref.newton_interp_batch(xs, [[y % p] for y in ys], p, basis=1)
    assert st == 0 and [int(mono[d, 0]) for d in range(B)] == want


def test_newton_duplicate_sample_status_and_order_dependence():
    p = P63
    out, st = ref.newton_interp_batch([3, 5, 3], [[1], [2], [3]], p)
    assert st == ((2 << 8) | ref.ST_DUPLICATE_SAMPLE)
    xs, ys = [2, 9, 4], [[10], [20], [33]]
    a, _ = ref.newton_interp_batch(xs, ys, p, basis=0)
    perm = [2, 0, 1]
    a2, _ = ref.newton_interp_batch([xs[k] for k in perm], [ys[k] for k in perm], p, basis=0)
    m1, _ = ref.newton_interp_batch(xs, ys, p, basis=1)
    m2, _ = ref.newton_interp_batch([xs[k] for k in perm], [ys[k] for k in perm], p, basis=1)
    assert (m1 == m2).all() and not (a == a2).all()  # reading G16


# ---------------------------------------------------------------------------- power sums (L60, L219)
@pytest.mark.parametrize("s0", [0, 1])
def test_power_sums_vs_python(s0):
    p = P63
    ts = [3, 8]
    offsets = [0, 3, 11]
    nodes = rnd(p, 11, 17, lo=1)
    coef = np.array([rnd(p, 11, 18), rnd(p, 11, 19)], dtype=np.uint64)
    out = ref.power_sums(nodes, offsets, coef, p, s0)
    for f, t in enumerate(ts):
        o = offsets[f]
        for b in range(2):
            for s in range(t):
                want = sum(int(coef[b, o + i]) * pow(nodes[o + i], s + s0, p) for i in range(t)) % p
                assert int(out[b, o + s]) == want


# ---------------------------------------------------------------------------- end to end: planted recovery
def probe_values(w, planted=None):
    """Probe values of the planted function, v_{j,s} = f(y^(s+s0), c_j), through the oracle."""
    planted = w.planted if planted is None else planted
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    at = ref.poly_rows_eval(w.samples, planted, w.p)
    return ref.power_sums(nodes, w.offsets, at, w.p, w.s0), nodes


def eval_planted(w, planted, f, point):
    """f(z_1..z_nv, z_k) in Python big integers."""
    p = w.p
    o, e = int(w.offsets[f]), int(w.offsets[f + 1])
    tot = 0
    for i in range(o, e):
        ci = sum(int(planted[d, i]) * pow(point[-1], d, p) for d in range(planted.shape[0]))
        term = ci
        for j in range(w.nv):
            term = term * pow(point[j], int(w.exps[i, j]), p) % p
        tot += term
    return tot % p


@pytest.mark.parametrize("dense", [False, True])
@pytest.mark.parametrize("s0", [0, 1])
def test_config1_planted_recovery_and_fresh_probes(dense, s0):
    w = wl.config(1, dense=dense)
    w.s0 = s0
    assert w.T_tot == 50 and w.B == 11 and w.nv == 2
    vals, nodes = probe_values(w)
    out, nodes2, status = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, vals, w.p, s0, basis=1)
    assert not status.any() and (nodes == nodes2).all()
    assert (out == w.planted).all()  # exact recovery of every coefficient polynomial
    r = random.Random(20)
    for _ in range(5):  # 5 fresh probes at points not used in the reconstruction
        z = [r.randrange(2, w.p) for _ in range(w.nv + 1)]
        assert eval_planted(w, out, 0, z) == eval_planted(w, w.planted, 0, z)
    a, _, _ = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, vals, w.p, s0, basis=0)
    assert (a[0] == ref.poly_rows_eval(w.samples, w.planted, w.p)[0]).all()


def test_batched_planted_recovery_ragged():
    w = wl.make_box_workload("rag", 99, F=5, nv=3, t=[1, 2, 17, 33, 8], emax=6, B=4, dense=True)
    vals, _ = probe_values(w)
    out, _, status = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, vals, w.p, 0, basis=1)
    assert not status.any() and (out == w.planted).all()


# ---------------------------------------------------------------------------- balanced (eq. 4)
def ragged_rational(s0):
    """Three rational functions of different sizes (numerators 30 / 7 / 19 terms, denominators 12 / 1 / 9)."""
    return wl.make_rational_workload("rag4", wl.SEED_BASE + 44, 3, 6, [30, 7, 19], [12, 1, 9], 24, 25, s0=s0)


@pytest.mark.parametrize("s0", [0, 1])
@pytest.mark.parametrize("ragged", [False, True])
def test_balanced_recovers_C_times_planted_and_cross_multiplied_probes(s0, ragged):
    """eq. (4) (readings G3, G20) with probes at the powers s0 .. s0 + t - 1 (reading G1: s0 = 1
    divides by m_i at the end) and with functions of different lengths in one batch (the per-probe factor h_s is
    shared by numerator and denominator: the numerator uses s < t_N, the denominator s < t_D)."""
    rw = ragged_rational(s0) if ragged else wl.config(4, F=3, t=30)  # t_num = 30, t_den = 12
    rw.num.s0 = rw.den.s0 = s0
    p = rw.num.p
    c0 = int(rw.num.samples[0])
    parts, Cs = {}, None
    f_scale = []
    for f in range(rw.num.F):  # C = 1 / (skeleton-level coefficient of D's lowest monomial), per function
        i = int(rw.den.offsets[f]) + int(rw.low_den[f])
        a_low = sum(int(rw.den.planted[d, i]) * pow(c0, d, p) for d in range(rw.den.B)) % p
        f_scale.append(pow(a_low, -1, p))
    for name, w in (("num", rw.num), ("den", rw.den)):
        true_vals, nodes = probe_values(w)  # n(y^s, c_j)
        skel = ref.poly_rows_eval(w.samples, w.planted, p)[0].copy()  # coefficients at x_k = c_0 ...
        u = true_vals.copy()
        for f in range(w.F):
            o, e = int(w.offsets[f]), int(w.offsets[f + 1])
            for i in range(o, e):  # ... times the unknown constant C of this function
                skel[i] = int(skel[i]) * f_scale[f] % p
            for s in range(e - o):  # u_{j,s} = true value times the unknown per-probe factor h_s
                for j in range(w.B):
                    u[j, o + s] = int(true_vals[j, o + s]) * int(rw.h[s]) % p
        parts[name] = dict(exps=w.exps, offsets=w.offsets, skel=skel, uvals=u)
    on, od, status = ref.balanced_zippel_lift_step(parts["num"], parts["den"], rw.num.anchors, rw.num.samples, p,
                                                   s0, basis=1)
    assert not status.any()
    for name, w, out in (("num", rw.num, on), ("den", rw.den, od)):
        a0 = ref.poly_rows_eval(w.samples, out, p)[0]
        assert (a0 == parts[name]["skel"]).all()  # the j = 0 solve returns the skeleton
        for f in range(w.F):
            o, e = int(w.offsets[f]), int(w.offsets[f + 1])
            for i in range(o, e):
                for d in range(w.B):
                    assert int(out[d, i]) == int(w.planted[d, i]) * f_scale[f] % p  # = C x planted
    for f in range(rw.den.F):  # normalisation: D's lowest monomial has coefficient 1 at x_k = c_0
        i = int(rw.den.offsets[f]) + int(rw.low_den[f])
        assert int(parts["den"]["skel"][i]) == 1
    r = random.Random(21)
    for f in range(rw.num.F):  # cross-multiplied fresh probes, independent of C
        z = [r.randrange(2, p) for _ in range(rw.num.nv + 1)]
        lhs = eval_planted(rw.num, on, f, z) * eval_planted(rw.den, rw.den.planted, f, z) % p
        rhs = eval_planted(rw.num, rw.num.planted, f, z) * eval_planted(rw.den, od, f, z) % p
        assert lhs == rhs


def test_eval_sparse_vs_python():
    """ref_eval_sparse (the fresh-probe evaluator) against Python integers: random rows, a zero
    exponent row, the largest exponent 65535, a zero coordinate, one term, and a small prime."""
    r = random.Random(31)
    for p in (101, 65537, P63):
        for t, nv in ((1, 1), (7, 3), (40, 6)):
            exps = np.array([[r.choice([0, 1, 2, 5, 40, 65535]) for _ in range(nv)] for _ in range(t)], dtype=np.uint16)
            exps[0, :] = 0  # the constant term
            coef = np.array([r.randrange(p) for _ in range(t)], dtype=np.uint64)
            for point in ([r.randrange(p) for _ in range(nv)], [0] * nv, [p - 1] * nv, [1] + [r.randrange(p) for _ in range(nv - 1)]):
                want = 0
                for row, c in zip(exps, coef):
                    term = int(c)
                    for e, z in zip(row, point):
                        term = term * pow(int(z), int(e), p) % p  # Python: 0 ** 0 == 1, as in the polynomial ring
                    want += term
                assert ref.eval_sparse(exps, coef, np.array(point, dtype=np.uint64), p) == want % p


def test_balanced_zero_pivot_status():
    p = 101
    part = dict(exps=[[0], [1], [2]], offsets=[0, 3], skel=[1, 2, 3], uvals=[[5, 0, 7], [1, 2, 3]])
    on, od, st = ref.balanced_zippel_lift_step(part, part, [2], [3, 4], p)
    assert st[0] == ((1 << 8) | ref.ST_ZERO_PIVOT) and st[1] == st[0]


# ---------------------------------------------------------------------------- golden worked example
def test_golden_worked_example():
    gold = json.load(open(GOLD))
    for c in gold["cases"]:
        p = c["p"]
        exps = np.array(c["exps"], dtype=np.uint16)
        nodes = ref.eval_nodes(exps, c["anchors"], p)
        assert [int(x) for x in nodes] == c["nodes"]
        M = ref.master_poly(nodes, p)
        assert [int(x) for x in M] == c["master"]
        planted = np.array(c["planted"], dtype=np.uint64).T.copy()  # [B, t]
        at = ref.poly_rows_eval(c["samples"], planted, p)
        vals = ref.power_sums(nodes, [0, 4], at, p)
        assert vals.tolist() == c["vals"]
        den, num = ref.node_solve(nodes, M, vals, p)
        assert [int(x) for x in den] == c["den"]
        coefs, st = ref.vandermonde_solve_batch(nodes, [0, 4], vals, p)
        assert st[0] == 0 and coefs.tolist() == c["solved"]
        a, st = ref.newton_interp_batch(c["samples"], coefs, p, basis=0)
        assert a.T.tolist() == c["newton"]
        mono, st = ref.newton_interp_batch(c["samples"], coefs, p, basis=1)
        assert mono.T.tolist() == c["planted"]
        out, _, st = ref.zippel_lift_step(exps, [0, 4], c["anchors"], c["samples"], vals, p, 0, 1)
        assert out.T.tolist() == c["planted"] and st[0] == 0
