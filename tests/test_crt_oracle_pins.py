"""Pins of the oracle's two-prime CRT + rational reconstruction: planted
rationals a/b with |a|, b <= floor(sqrt((m-1)/2)) are recovered exactly from their images mod p1 and p2
(uniqueness: 2 N D < m), integers and zero included; the defining congruence a = b x (mod m) holds for every
accepted output (Python integers); the primes are the two largest below 2^63 (the oracle's Miller-Rabin)."""
import math
import random

import numpy as np

from oracle import ref

P1 = (1 << 63) - 25


def test_second_prime_is_the_next_one_below_p1():
    p2 = ref.largest_prime_below(P1)
    assert p2 == (1 << 63) - 165 and ref.is_prime(p2) and not any(ref.is_prime(x) for x in range(p2 + 1, P1))


def test_crt_rational_recovers_planted_fractions():
    p1, p2 = P1, ref.largest_prime_below(P1)
    m = p1 * p2
    N = math.isqrt((m - 1) // 2)
    rng = random.Random(4)
    planted = [(0, 1), (1, 1), (-1, 1), (N, 1), (-N, 1), (1, N), (-1, N), (N, N - 1), (2**31, 3), (-7, 2**40 + 1)]
    while len(planted) < 400:
        bits = rng.randrange(1, 63)
        a, b = rng.randrange(-min(N, 1 << bits), min(N, 1 << bits) + 1), rng.randrange(1, min(N, 1 << rng.randrange(1, 63)) + 1)
        if math.gcd(a, b) == 1 and b % p1 and b % p2:
            planted.append((a, b))
    r1 = np.array([a * pow(b, -1, p1) % p1 for a, b in planted], dtype=np.uint64)
    r2 = np.array([a * pow(b, -1, p2) % p2 for a, b in planted], dtype=np.uint64)
    num, den, st = ref.crt_rational_batch(r1, r2, p1, p2)
    assert not st.any()
    assert [(int(a), int(b)) for a, b in zip(num, den)] == planted


def test_crt_rational_outputs_satisfy_the_congruence_or_are_rejected():
    p1, p2 = P1, ref.largest_prime_below(P1)
    m = p1 * p2
    N = math.isqrt((m - 1) // 2)
    rng = random.Random(6)
    r1 = np.array([rng.randrange(p1) for _ in range(300)], dtype=np.uint64)
    r2 = np.array([rng.randrange(p2) for _ in range(300)], dtype=np.uint64)
    num, den, st = ref.crt_rational_batch(r1, r2, p1, p2)
    assert (st == 0).any() and set(st.tolist()) <= {0, 21}
    for a1, a2, a, b, s in zip(r1.tolist(), r2.tolist(), num.tolist(), den.tolist(), st.tolist()):
        if s == 0:
            assert 0 < b <= N and abs(a) <= N and math.gcd(a, b) == 1
            assert (a - b * a1) % p1 == 0 and (a - b * a2) % p2 == 0
        else:
            assert a == 0 and b == 0
    # small primes: every residue pair, against exhaustive search for the unique fraction within the bounds
    p1s, p2s = 101, 103
    ms = p1s * p2s
    Ns = math.isqrt((ms - 1) // 2)
    pairs = [(x % p1s, x % p2s) for x in range(0, ms, 7)]
    num, den, st = ref.crt_rational_batch(np.array([a for a, _ in pairs], dtype=np.uint64),
                                          np.array([b for _, b in pairs], dtype=np.uint64), p1s, p2s)
    for k, x in enumerate(range(0, ms, 7)):
        sols = [(a, b) for b in range(1, Ns + 1) for a in range(-Ns, Ns + 1) if (a - b * x) % ms == 0 and math.gcd(a, b) == 1]
        if st[k] == 0:
            assert sols == [(int(num[k]), int(den[k]))]
        else:
            assert sols == []
