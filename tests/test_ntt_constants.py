"""CPU-only pins of the constants of the three-prime NTT engine (csrc/ntt.cuh), read back from the
test build through zippel_test_ntt_constants() and checked with Python integers and the oracle's Miller-Rabin test
(which is itself pinned in test_oracle_pins.py): a wrong prime, a root of the wrong order or too small a product
would make every long-skeleton result wrong in a way only a GPU run could show."""
import pytest


@pytest.fixture(scope="module")
def consts():
    from paper_2505_24256_b200 import testhooks

    return testhooks.ntt_constants()


def test_primes_are_prime_and_ntt_friendly(consts):
    from oracle import ref

    q = consts["q"]
    assert q[0] > q[1] > q[2]
    for x in q:
        assert ref.is_prime(x)
        assert x < 1 << 62  # lazy butterflies keep values below 4q < 2^64
        assert (x - 1) % (1 << consts["log_order"]) == 0
        assert all(x % s for s in (3, 5, 7, 11, 13))  # a second, trivial opinion


def test_roots_have_order_2_24(consts):
    k = consts["log_order"]
    assert k == 24
    for q, w in zip(consts["q"], consts["w"]):
        assert 1 < w < q
        assert pow(w, 1 << (k - 1), q) == q - 1  # w^(2^23) = -1: the order is exactly 2^24


def test_product_covers_the_convolution_bound(consts):
    """A coefficient of the integer product of two polynomials with coefficients below 2^63 and at most 2^23 terms
    is below 2^23 * 2^126 = 2^149; the CRT recovers it only if q1 q2 q3 exceeds that."""
    q = consts["q"]
    assert q[0] * q[1] * q[2] > 1 << 149
    # the Garner step reduces k1 < q1 modulo q2 and k2 < q2 modulo q3 by ONE conditional subtraction
    assert q[0] < 2 * q[1] and q[1] < 2 * q[2] and q[0] < 2 * q[2]
    # inputs < 2^63 enter the forward transform unreduced: they must be below 4q
    assert all(4 * x > 1 << 63 for x in q)
