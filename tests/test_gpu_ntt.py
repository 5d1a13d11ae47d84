"""The three-prime NTT engine (csrc/ntt.cuh) against Python integers, through the hooks of the test
build (include/zippel_test.h): forward/inverse round trips and polynomial products modulo p at lengths that take one,
two and three passes, with ragged operand lengths, the extreme coefficient bound, and small primes."""
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
def hooks():
    from paper_2505_24256_b200 import testhooks

    testhooks.lib()
    return testhooks


def rnd(seed, n, p):
    return np.random.Generator(np.random.Philox(key=[seed, n & 0xFFFFFFFF])).integers(0, p, n, dtype=np.uint64)


# transform lengths: 2 .. 4096 one pass; 2^13 .. 2^21 two passes (1 .. 9 strided stages); 2^22 .. 2^24 three
@pytest.mark.parametrize("na,nb", [(1, 2), (3, 3), (40, 25), (2048, 2049), (4096, 4097), (5000, 60000), (1 << 16, 1 << 16),
                                   (1 << 20, (1 << 20) + 1), (1 << 21, (1 << 21) + 5), (1 << 22, (1 << 22) + 1)])
def test_forward_inverse_round_trip(zp, hooks, na, nb):
    a, b = rnd(1, na, P63), rnd(2, nb, P63)
    got = hooks.polymul(zp.to_dev(a), zp.to_dev(b), P63, roundtrip=True)
    torch.cuda.synchronize()
    n = got.numel() // 6
    q = hooks.ntt_constants()["q"]
    x = torch.zeros(2 * n, dtype=torch.int64, device="cuda")
    x[:na] = zp.to_dev(a)
    x[n:n + nb] = zp.to_dev(b)
    for j in range(3):
        assert torch.equal(got[2 * n * j:2 * n * (j + 1)], x % q[j]), f"prime {j}, n = {n}"


@pytest.mark.parametrize("p", [101, 65537, (1 << 61) - 1, P63])
@pytest.mark.parametrize("na,nb", [(1, 1), (2, 1), (7, 9), (64, 64), (100, 157), (300, 213)])
def test_small_products_vs_python(zp, hooks, p, na, nb):
    a, b = rnd(3, na, p), rnd(4, nb, p)
    a[-1] = p - 1
    b[0] = p - 1
    got = zp.to_host(hooks.polymul(zp.to_dev(a), zp.to_dev(b), p))
    want = [0] * (na + nb - 1)
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            want[i + j] = (want[i + j] + int(x) * int(y)) % p
    assert [int(x) for x in got] == want


@pytest.mark.parametrize("na,nb", [(4096, 4097), (9000, 7000), (1 << 17, 3), ((1 << 19) + 11, 1 << 19), (1 << 21, (1 << 21) + 1)])
def test_large_products_sparse_operand(zp, hooks, na, nb):
    """a has six non-zero coefficients (both ends included): the product is six shifted copies of b, exact for every
    output coefficient, in vectorised Python integers."""
    p = P63
    b = rnd(5, nb, p)
    a = np.zeros(na, dtype=np.uint64)
    pos = sorted({0, na - 1, na // 2, na // 3, min(na - 1, 4095), min(na - 1, 4096)})
    for k, i in enumerate(pos):
        a[i] = (p - 1 - k) if k % 2 == 0 else (123456789 + k)
    got = zp.to_host(hooks.polymul(zp.to_dev(a), zp.to_dev(b), p))
    want = np.zeros(na + nb - 1, dtype=object)
    bo = b.astype(object)
    for i in pos:
        want[i:i + nb] += int(a[i]) * bo
    want %= p
    assert (got.astype(object) == want).all()


@pytest.mark.parametrize("logn", [12, 20, 24])
def test_extreme_coefficients_reach_the_crt_bound(zp, hooks, logn):
    """All coefficients p - 1 with 2^(logn-1) terms per operand: the integer product peaks at 2^(logn-1) (p-1)^2
    (2^149 at the longest transform: the bound the three primes were sized for) and equals, modulo p, the number of
    terms that meet in each coefficient, because (p-1)^2 = 1."""
    p = P63
    n = 1 << (logn - 1)
    a = torch.full((n,), p - 1, dtype=torch.int64, device="cuda")
    got = hooks.polymul(a, a, p)
    torch.cuda.synchronize()
    k = torch.arange(2 * n - 1, dtype=torch.int64, device="cuda")
    want = torch.minimum(k + 1, 2 * n - 1 - k)
    assert torch.equal(got, want)
