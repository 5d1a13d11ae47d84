"""Bit-exact parity of crt_rational_reconstruct_batch (C-ABI) with the CPU oracle: planted fractions
(recovered exactly: expected values are the generator's), arbitrary residue pairs (accepted and rejected ones),
small primes, several CTAs and a ragged tail."""
import math
import random

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

P1, P2 = (1 << 63) - 25, (1 << 63) - 165


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


def both(zp, ref, r1, r2, p1, p2):
    wn, wd, ws = ref.crt_rational_batch(r1, r2, p1, p2)
    gn, gd, gs = zp.crt_rational_reconstruct_batch(zp.to_dev(r1), zp.to_dev(r2), p1, p2)
    gn, gd, gs = gn.cpu().numpy(), gd.cpu().numpy(), gs.cpu().numpy()
    assert (gs == ws).all() and (gn == wn).all() and (gd == wd).all()
    return gn, gd, gs


def test_crt_parity_planted_fractions(zp, ref):
    N = math.isqrt((P1 * P2 - 1) // 2)
    rng = random.Random(21)
    planted = [(0, 1), (1, 1), (-1, 1), (N, 1), (-N, 1), (1, N), (N, N - 1)]
    while len(planted) < 256 * 40 + 77:
        a = rng.randrange(-min(N, 1 << rng.randrange(1, 64)), min(N, 1 << rng.randrange(1, 64)) + 1)
        b = rng.randrange(1, min(N, 1 << rng.randrange(1, 64)) + 1)
        if math.gcd(a, b) == 1:
            planted.append((a, b))
    r1 = np.array([a * pow(b, -1, P1) % P1 for a, b in planted], dtype=np.uint64)
    r2 = np.array([a * pow(b, -1, P2) % P2 for a, b in planted], dtype=np.uint64)
    gn, gd, gs = both(zp, ref, r1, r2, P1, P2)
    assert not gs.any()
    assert [(int(a), int(b)) for a, b in zip(gn, gd)] == planted


@pytest.mark.parametrize("p1,p2", [(P1, P2), (P2, P1), ((1 << 61) - 1, (1 << 31) - 1), (101, 103), (65537, 3)])
def test_crt_parity_arbitrary_residues(zp, ref, p1, p2):
    r = np.random.Generator(np.random.Philox(key=[31, p1 % 1000]))
    n = 256 * 9 + 5
    r1 = r.integers(0, p1, n, dtype=np.uint64)
    r2 = r.integers(0, p2, n, dtype=np.uint64)
    r1[:3] = [0, 1, p1 - 1]
    r2[:3] = [0, 1, p2 - 1]
    gn, gd, gs = both(zp, ref, r1, r2, p1, p2)
    assert (gs == 0).any()
    assert int(gn[0]) == 0 and int(gd[0]) == 1 and int(gn[1]) == 1 and int(gn[2]) == -1


def test_crt_huge_and_borderline_quotients(zp, ref):
    """The kernel estimates Euclid's quotients in double precision and takes the exact 128-bit division only beyond 2^50:
    combined values x chosen so that the first quotients m / x are huge (x just above N), sit at the 2^50 switch, or at
    powers of two where a rounded estimate is off by one -- followed by arbitrary continuations.  == the oracle."""
    m = P1 * P2
    N = math.isqrt((m - 1) // 2)
    xs = [N + 1, N + 2, N + 12345, (1 << 63), (1 << 64) - 1, (1 << 64), (1 << 64) + 1, (1 << 70) + 3, m - 1, m - 2, m // 2, m // 2 + 1,
          m // 3, m // 3 + 1]
    for e in (49, 50, 51, 52, 53):  # first quotient about 2^e
        for d in (-2, -1, 0, 1, 2):
            xs.append(m // ((1 << e) + d))
            xs.append(m // ((1 << e) + d) + 1)
    rng = random.Random(77)
    for _ in range(300):  # second and later quotients large: x = (m + r) / q-ish with a tiny remainder
        q = rng.randrange(1 << 40, 1 << 62)
        xs.append(m // q + rng.randrange(0, 3))
    xs = [x for x in xs if 0 < x < m]
    r1 = np.array([x % P1 for x in xs], dtype=np.uint64)
    r2 = np.array([x % P2 for x in xs], dtype=np.uint64)
    both(zp, ref, r1, r2, P1, P2)
