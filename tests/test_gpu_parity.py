"""Bit-exact parity of the CUDA path (through the C-ABI, paper_2505_24256_b200.api) with the CPU
oracle (oracle/ref.py) on the same seeded inputs.  All work is integer: every comparison is ==.

Sizes are chosen so the oracle finishes in seconds yet several tiles and a ragged tail are covered
(K3 tile = 64 coefficients, 128 nodes per CTA; product-tree leaf = 1024 nodes).  Full-size cases
(BASELINE.json sizes, bench.py's launch configuration) are in test_gpu_fullsize.py.
"""
import random

import numpy as np
import pytest

from paper_2505_24256_b200 import workloads as wl

pytestmark = pytest.mark.gpu

P63 = wl.P63
PRIMES = [101, 65537, (1 << 31) - 1, (1 << 61) - 1, P63]


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


@pytest.fixture(scope="module")
def ref():
    from oracle import ref as r

    r.lib()
    return r


def u64(xs):
    return np.array(xs, dtype=np.uint64)


# ------------------------------------------------------------------------------ (a0) substrate
def edge_values(p):
    cand = [0, 1, 2, p - 1, p - 2, (p - 1) // 2, (p + 1) // 2, (1 << 32) - 1, 1 << 32, (1 << 32) + 1,
            0xFFFFFFFF00000000, 0x00000000FFFFFFFF, 0x7FFFFFFF7FFFFFFF, 0x7FFFFFFFFFFFFFFF, (1 << 62) - 1, 1 << 62,
            0x5555555555555555, 0x2AAAAAAAAAAAAAAA]
    return sorted({c % p for c in cand})


@pytest.mark.parametrize("p", PRIMES)
def test_modarith_fuzz_vs_python(zp, hooks, p):
    """PAPER.md section 2.1: the paper's own test of mul_mod is 10^7 iterations; here 10^7 random pairs
    for p = 2^63 - 25 (2*10^5 for the other primes) plus all pairs of edge values, against Python big integers
    (a third opinion)."""
    r = np.random.Generator(np.random.Philox(key=[7, p & 0xFFFF]))
    n = 10_000_000 if p == P63 else 200_000
    ev = edge_values(p)
    ea = [a for a in ev for _ in ev]
    eb = [b for _ in ev for b in ev]
    a = np.concatenate([u64(ea), r.integers(0, p, n, dtype=np.uint64)])
    b = np.concatenate([u64(eb), r.integers(0, p, n, dtype=np.uint64)])
    da, db = zp.to_dev(a), zp.to_dev(b)
    ao, bo = a.astype(object), b.astype(object)
    got = zp.to_host(hooks.zippel_modarith_selftest(0, da, db, p))
    assert (got.astype(object) == (ao * bo) % p).all()
    got = zp.to_host(hooks.zippel_modarith_selftest(1, da, db, p))
    assert (got.astype(object) == (ao + bo) % p).all()
    got = zp.to_host(hooks.zippel_modarith_selftest(2, da, db, p))
    assert (got.astype(object) == (ao - bo) % p).all()
    m = 2000
    got = zp.to_host(hooks.zippel_modarith_selftest(3, da[:m].contiguous(), db[:m].contiguous(), p))
    assert [int(x) for x in got] == [pow(int(x), int(e), p) for x, e in zip(a[:m], b[:m])]
    got = zp.to_host(hooks.zippel_modarith_selftest(4, da[:m].contiguous(), None, p))
    assert [int(x) for x in got] == [pow(int(x), p - 2, p) for x in a[:m]]


@pytest.mark.parametrize("p", PRIMES)
def test_horner_step_lazy_operand_vs_python(zp, hooks, p):
    """The hot recurrence x <- m x + a of (a3) (PAPER.md L193 Horner / synthetic division), with x a LAZY
    value: any 64-bit number, in particular the extremes 2p-1, 2^64-1, and m, a at 0, 1, p-1."""
    r = np.random.Generator(np.random.Philox(key=[11, p & 0xFFFF]))
    n = 500_000
    ex = sorted({0, 1, p - 1, p, p + 1, 2 * p - 1, 2 * p, (1 << 64) - 1, (1 << 64) - 2, 1 << 63, (1 << 63) - 1,
                 (1 << 32) - 1, 1 << 32, 0xFFFFFFFF00000000, 0x00000000FFFFFFFF})
    ev = edge_values(p)
    xs = [x for x in ex for _ in ev]
    ms = [m for _ in ex for m in ev]
    x = np.concatenate([u64(xs), r.integers(0, 1 << 64, n, dtype=np.uint64)])
    m = np.concatenate([u64(ms), r.integers(0, p, n, dtype=np.uint64)])
    x[-8:] = u64([p - 1, 0, 1, p - 1, (1 << 64) - 1, p - 1, 2 * p - 1, p - 1])  # addend a[(i+1) % n] at its extremes too
    m[-8:] = p - 1
    got = zp.to_host(hooks.zippel_modarith_selftest(6, zp.to_dev(x), zp.to_dev(m), p))
    xo, mo = x.astype(object), m.astype(object)
    ao = np.roll(xo, -1) % p
    assert (got.astype(object) == (mo * xo + ao) % p).all()


@pytest.mark.parametrize("p", [65537, P63])
@pytest.mark.parametrize("n", [1, 255, 100_000])
def test_deferred_dot_identity_L208(zp, hooks, p, n):
    """the deferred (wide accumulator) sum equals the step-wise reduced sum."""
    r = np.random.Generator(np.random.Philox(key=[8, n]))
    a = r.integers(0, p, n, dtype=np.uint64)
    b = r.integers(0, p, n, dtype=np.uint64)
    a[: min(n, 4)] = p - 1
    b[: min(n, 4)] = p - 1
    got = int(zp.to_host(hooks.zippel_modarith_selftest(5, zp.to_dev(a), zp.to_dev(b), p))[0])
    assert got == int((a.astype(object) * b.astype(object)).sum() % p)


# ------------------------------------------------------------------------------ (a1) nodes
@pytest.mark.parametrize("idx,kw", [(1, {}), (2, dict(F=64)), (3, {}), (5, {})])
def test_eval_nodes_parity(zp, ref, idx, kw):
    w = wl.config(idx, with_vals=False, with_planted=False, **kw)
    want = ref.eval_nodes(w.exps, w.anchors, w.p)
    got = zp.to_host(zp.zippel_eval_nodes(zp.to_dev(w.exps), zp.to_dev(w.anchors), w.p))
    assert (got == want).all()


def test_eval_nodes_edge_exponents(zp, ref):
    """exponent 0 rows -> 1; maximal uint16 exponents; nv = 1 and nv = ZP_MAX_NV; small primes."""
    r = np.random.Generator(np.random.Philox(key=[9, 0]))
    for p in PRIMES:
        for nv in (1, 5, 32):
            exps = r.integers(0, 65536, (777, nv), dtype=np.uint16)
            exps[0] = 0
            exps[1] = 65535
            anchors = r.integers(0, p, nv, dtype=np.uint64)
            anchors[0] = p - 1
            want = ref.eval_nodes(exps, anchors, p)
            got = zp.to_host(zp.zippel_eval_nodes(zp.to_dev(exps), zp.to_dev(anchors), p))
            assert (got == want).all()
            assert got[0] == 1


# ------------------------------------------------------------------------------ (a2)-(a4) solve
def random_solve_case(seed, ts, B, p):
    r = np.random.Generator(np.random.Philox(key=[10, seed]))
    offsets = np.zeros(len(ts) + 1, dtype=np.int64)
    offsets[1:] = np.cumsum(ts)
    T = int(offsets[-1])
    nodes = np.empty(T, dtype=np.uint64)
    for f, t in enumerate(ts):
        nodes[offsets[f]:offsets[f + 1]] = wl.distinct_residues(r, 1, p, t)
    vals = r.integers(0, p, (B, T), dtype=np.uint64)
    return nodes, offsets, vals


@pytest.mark.parametrize("p", [101, (1 << 31) - 1, P63])
@pytest.mark.parametrize("s0", [0, 1])
def test_solve_small_ragged_batch(zp, ref, p, s0):
    ts = [1, 2, 3, 7, 50, 63, 64, 65] if p > 101 else [1, 2, 3, 7, 50, 63, 64, 65, 100]
    nodes, offsets, vals = random_solve_case(1, ts, 5, p)
    want, wst = ref.vandermonde_solve_batch(nodes, offsets, vals, p, s0)
    got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), offsets, zp.to_dev(vals), p, s0)
    assert not wst.any() and not zp.to_host(st).any()
    assert (zp.to_host(got) == want).all()


@pytest.mark.parametrize("B", list(range(1, 28)) + [33, 52, 53, 64])
def test_solve_every_rhs_count_path(zp, ref, B):
    """each B exercises another template instance / pass split of the node-solve kernel"""
    nodes, offsets, vals = random_solve_case(100 + B, [63, 64, 65, 129, 200], B, P63)
    want, _ = ref.vandermonde_solve_batch(nodes, offsets, vals, P63, 0)
    got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), offsets, zp.to_dev(vals), P63, 0)
    assert not zp.to_host(st).any()
    assert (zp.to_host(got) == want).all()


@pytest.mark.parametrize("ts,B", [([1000, 1023, 1024, 1025], 3), ([2049, 1, 4097], 2), ([9001], 1), ([3000] * 3, 9)])
def test_solve_tree_levels_and_tails(zp, ref, ts, B):
    """t around the product-tree leaf size (1024) and across 1-3 merge levels, ragged tails"""
    nodes, offsets, vals = random_solve_case(sum(ts), ts, B, P63)
    want, _ = ref.vandermonde_solve_batch(nodes, offsets, vals, P63, 0)
    got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), offsets, zp.to_dev(vals), P63, 0)
    assert not zp.to_host(st).any()
    assert (zp.to_host(got) == want).all()


@pytest.mark.parametrize("ts", [[4095], [4096], [4097, 5000, 300], [1, 4200, 2, 33]])
@pytest.mark.parametrize("s0", [0, 1])
def test_solve_single_rhs_both_paths(zp, ref, ts, s0):
    """B = 1: below t = 4096 the per-node quotient form, from 4096 on W = corr(v, M) and two Horner chains per node
    (k_corr_w, k_node_eval2); a batch mixes functions of both lengths under the longer one's path"""
    nodes, offsets, vals = random_solve_case(40 + len(ts), ts, 1, P63)
    want, wst = ref.vandermonde_solve_batch(nodes, offsets, vals, P63, s0)
    got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), offsets, zp.to_dev(vals), P63, s0)
    assert not wst.any() and not zp.to_host(st).any()
    assert (zp.to_host(got) == want).all()


def test_solve_residual_property_large(zp, ref):
    """size the oracle cannot finish in seconds: t = 40000; the unique solution is checked by the residual
    sum_i c_i m_i^s = v_s on sampled s through the oracle's power sums (one s costs O(t log s))."""
    t = 40000
    nodes, offsets, vals = random_solve_case(5, [t], 2, P63)
    got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), offsets, zp.to_dev(vals), P63, 0)
    got = zp.to_host(got)
    assert not zp.to_host(st).any()
    rr = random.Random(3)
    for s in [0, 1, t - 1] + [rr.randrange(t) for _ in range(5)]:
        for b in range(2):
            acc = 0
            pw = [ref.powmod(int(m), s, P63) for m in nodes[:t]]
            acc = sum(int(c) * q for c, q in zip(got[b], pw)) % P63
            assert acc == int(vals[b, s])


def test_solve_status_duplicate_and_zero_node(zp, ref):
    p = P63
    nodes, offsets, vals = random_solve_case(6, [40, 200, 30], 3, p)
    nodes[offsets[1] + 150] = nodes[offsets[1] + 20]  # duplicate inside function 1
    want, wst = ref.vandermonde_solve_batch(nodes, offsets, vals, p, 0)
    got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), offsets, zp.to_dev(vals), p, 0)
    st = zp.to_host(st)
    assert (st == wst).all() and st[1] == ((20 << 8) | zp.ST_DUPLICATE_NODE) and st[0] == 0 and st[2] == 0
    got = zp.to_host(got)
    for f in (0, 2):  # other functions unaffected
        sl = slice(offsets[f], offsets[f + 1])
        assert (got[:, sl] == want[:, sl]).all()
    # zero node: fine for s0 = 0, flagged for s0 = 1 (G25)
    nodes, offsets, vals = random_solve_case(7, [33], 2, p)
    nodes[5] = 0
    for s0 in (0, 1):
        want, wst = ref.vandermonde_solve_batch(nodes, offsets, vals, p, s0)
        got, st = zp.vandermonde_solve_batch(zp.to_dev(nodes), offsets, zp.to_dev(vals), p, s0)
        assert (zp.to_host(st) == wst).all()
        if s0 == 0:
            assert wst[0] == 0 and (zp.to_host(got) == want).all()
        else:
            assert wst[0] == ((5 << 8) | zp.ST_DUPLICATE_NODE)


# ------------------------------------------------------------------------------ (a5) Newton
@pytest.mark.parametrize("B", [1, 2, 3, 9, 16, 17, 21, 25, 32, 33, 64])
@pytest.mark.parametrize("basis", [0, 1])
@pytest.mark.parametrize("n", [5, 1000 + 37])  # few coefficients: per-column recurrences; many: the matrix form L x vals
def test_newton_parity(zp, ref, B, basis, n):
    p = P63
    r = np.random.Generator(np.random.Philox(key=[11, B]))
    samples = wl.distinct_residues(r, 0, p, B)
    vals = r.integers(0, p, (B, n), dtype=np.uint64)
    want, wst = ref.newton_interp_batch(samples, vals, p, basis)
    got, st = zp.newton_interp_batch(zp.to_dev(samples), zp.to_dev(vals), p, basis)
    assert wst == 0 and int(zp.to_host(st)[0]) == 0
    assert (zp.to_host(got) == want).all()


def test_newton_small_prime_inplace_and_duplicate(zp, ref):
    p = 101
    r = np.random.Generator(np.random.Philox(key=[12, 0]))
    samples = wl.distinct_residues(r, 0, p, 7)
    vals = r.integers(0, p, (7, 300), dtype=np.uint64)
    want, _ = ref.newton_interp_batch(samples, vals, p, 1)
    dv = zp.to_dev(vals)
    got, st = zp.newton_interp_batch(zp.to_dev(samples), dv, p, 1, out=dv)  # in place
    assert (zp.to_host(got) == want).all()
    samples[5] = samples[2]
    _, wst = ref.newton_interp_batch(samples, vals, p, 0)
    _, st = zp.newton_interp_batch(zp.to_dev(samples), zp.to_dev(vals), p, 0)
    assert int(zp.to_host(st)[0]) == wst == ((5 << 8) | zp.ST_DUPLICATE_SAMPLE)


# ------------------------------------------------------------------------------ (a6) power sums
@pytest.mark.parametrize("s0", [0, 1])
@pytest.mark.parametrize("ts,p", [([1, 130, 257, 700], P63),
                                  # around k_power_sums's blocks: 512 probes per CTA, 64 nodes per tile, 32 probes per lane group
                                  ([511, 512, 513, 64, 65, 31, 33, 1024, 1537, 2], P63),
                                  ([100, 600, 3], (1 << 61) - 1), ([40, 529], 65537)])
def test_power_sums_parity(zp, ref, s0, ts, p):
    nodes, offsets, coef = random_solve_case(13, ts, 3, p)
    want = ref.power_sums(nodes, offsets, coef, p, s0)
    got = zp.zippel_power_sums(zp.to_dev(nodes), offsets, zp.to_dev(coef), p, s0)
    assert (zp.to_host(got) == want).all()


# ------------------------------------------------------------------------------ lifting step, configs 1-3, 5
def probe_values(ref, w, planted=None):
    planted = w.planted if planted is None else planted
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    at = ref.poly_rows_eval(w.samples, planted, w.p)
    return ref.power_sums(nodes, w.offsets, at, w.p, w.s0), nodes


def lift_both(zp, ref, w, vals, basis):
    want, wnodes, wst = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, vals, w.p, w.s0, basis)
    import torch

    dn = torch.empty(w.T_tot, dtype=torch.int64, device="cuda")
    got, st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(w.anchors), zp.to_dev(w.samples),
                                  zp.to_dev(vals), w.p, w.s0, basis, nodes_out=dn)
    assert (zp.to_host(dn) == wnodes).all()
    assert (zp.to_host(st) == wst).all()
    got = zp.to_host(got)
    assert (got == want).all()
    return got


@pytest.mark.parametrize("dense", [False, True])
@pytest.mark.parametrize("s0", [0, 1])
def test_config1_lift_parity_planted_and_fresh_probes(zp, ref, dense, s0):
    """BASELINE.json configs[0] in full: t = 50, D = 10, 2 -> 3 variables, 5 fresh probes."""
    w = wl.config(1, dense=dense)
    w.s0 = s0
    vals, _ = probe_values(ref, w)
    lift_both(zp, ref, w, vals, 0)
    got = lift_both(zp, ref, w, vals, 1)
    assert (got == w.planted).all()
    r = random.Random(20)
    for _ in range(5):
        z = u64([r.randrange(2, w.p) for _ in range(w.nv + 1)])
        full_exps = np.concatenate([w.exps, np.zeros((w.T_tot, 1), np.uint16)], axis=1)
        tot_got = tot_true = 0
        for d in range(w.B):
            full_exps[:, -1] = d
            tot_got += ref.eval_sparse(full_exps, got[d], z, w.p)
            tot_true += ref.eval_sparse(full_exps, w.planted[d], z, w.p)
        assert tot_got % w.p == tot_true % w.p


@pytest.mark.parametrize("dense", [False, True])
def test_config2_lift_parity_first_functions(zp, ref, dense):
    """configs[1] shape (t = 1000, nv = 4, B = 21), first 8 functions as a complete problem."""
    w = wl.config(2, F=8, dense=dense)
    vals, _ = probe_values(ref, w)
    got = lift_both(zp, ref, w, vals, 1)
    assert (got == w.planted).all()


def test_config3_lift_parity_prefix(zp, ref):
    """configs[2] shape (nv = 7, B = 9) on a 10^4-term skeleton as a complete problem."""
    w = wl.config(3, t=10000)
    lift_both(zp, ref, w, w.vals, 0)


def test_config5_solve_parity_prefix(zp, ref):
    """configs[4] shape (nv = 10, B = 1) on the 2^14-term prefix problem BASELINE.json names."""
    w = wl.config(5, t=1 << 14)
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    want, wst = ref.vandermonde_solve_batch(nodes, w.offsets, w.vals, w.p, 0)
    dn = zp.zippel_eval_nodes(zp.to_dev(w.exps), zp.to_dev(w.anchors), w.p)
    got, st = zp.vandermonde_solve_batch(dn, w.offsets, zp.to_dev(w.vals), w.p, 0)
    assert (zp.to_host(dn) == nodes).all()
    assert not wst.any() and not zp.to_host(st).any()
    assert (zp.to_host(got) == want).all()


def test_lift_ragged_batch_and_status_precedence(zp, ref):
    w = wl.make_box_workload("rag", 99, F=6, nv=3, t=[1, 2, 17, 133, 8, 260], emax=6, B=4, dense=True)
    vals, _ = probe_values(ref, w)
    got = lift_both(zp, ref, w, vals, 1)
    assert (got == w.planted).all()
    w.exps[w.offsets[3] + 9] = w.exps[w.offsets[3] + 4]  # duplicate node in function 3
    w.samples[3] = w.samples[1]  # and a duplicate sample for everybody
    want, _, wst = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, vals, w.p, 0, 0)
    _, st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(w.anchors), zp.to_dev(w.samples),
                                zp.to_dev(vals), w.p, 0, 0)
    assert (zp.to_host(st) == wst).all()
    assert wst[3] == ((4 << 8) | zp.ST_DUPLICATE_NODE) and wst[0] == ((3 << 8) | zp.ST_DUPLICATE_SAMPLE)


def test_lift_host_entry_matches_device_entry(zp, ref):
    """zippel_lift_step_host = H2D + zippel_lift_step + D2H (the bench's e2e call)."""
    import torch

    w = wl.config(2, F=3)
    want, _, wst = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, w.vals, w.p, 0, 1)
    pin = lambda a: torch.from_numpy(a.view(np.int64) if a.dtype == np.uint64 else a.view(np.int16)).pin_memory()
    h_out = torch.empty(w.vals.shape, dtype=torch.int64).pin_memory()
    h_st = torch.empty(w.F, dtype=torch.int32).pin_memory()
    ws = torch.empty(zp.host_workspace_bytes(w.offsets, w.nv, w.B), dtype=torch.uint8, device="cuda")
    zp.zippel_lift_step_host(pin(w.exps), w.offsets, pin(w.anchors), pin(w.samples), pin(w.vals), w.p, h_out, h_st,
                             ws, 0, 1)
    torch.cuda.synchronize()
    assert (h_out.numpy().view(np.uint64) == want).all() and (h_st.numpy() == wst).all()


def test_lift_host_entry_chunked_pipeline(zp, ref):
    """above 8 MB of values and 64 functions the host entry cuts the batch into 6 chunks of whole functions and
    pipelines H2D / kernels / D2H: every output equals the device entry's (itself checked against the oracle on
    sampled functions here); ragged function lengths, status of a planted duplicate node in one chunk"""
    import torch

    r = np.random.Generator(np.random.Philox(key=[77, 1]))
    ts = [int(x) for x in r.integers(200, 700, 160)]
    w = wl.make_box_workload("chunks", wl.SEED_BASE + 55, len(ts), 4, ts, 20, 21, with_planted=False)
    assert w.vals.nbytes >= (8 << 20)
    w.exps[int(w.offsets[100]) + 5] = w.exps[int(w.offsets[100]) + 17]  # duplicate node in function 100
    dev_out, dev_st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(w.anchors), zp.to_dev(w.samples),
                                          zp.to_dev(w.vals), w.p, 0, 1)
    pin = lambda a: torch.from_numpy(a.view(np.int64) if a.dtype == np.uint64 else a.view(np.int16)).pin_memory()
    h_out = torch.empty(w.vals.shape, dtype=torch.int64).pin_memory()
    h_st = torch.empty(w.F, dtype=torch.int32).pin_memory()
    ws = torch.empty(zp.host_workspace_bytes(w.offsets, w.nv, w.B), dtype=torch.uint8, device="cuda")
    for _ in range(2):  # twice: the copy streams and events are reused across calls
        zp.zippel_lift_step_host(pin(w.exps), w.offsets, pin(w.anchors), pin(w.samples), pin(w.vals), w.p, h_out, h_st,
                                 ws, 0, 1)
        torch.cuda.synchronize()
    st = h_st.numpy()
    assert (st == zp.to_host(dev_st)).all() and st[100] != 0 and np.count_nonzero(st) == 1
    got = h_out.numpy().view(np.uint64)
    ok = np.ones(w.T_tot, dtype=bool)
    ok[int(w.offsets[100]):int(w.offsets[101])] = False  # outputs of the failed function are unspecified
    assert (got[:, ok] == zp.to_host(dev_out)[:, ok]).all()
    for f in (0, 63, 159):
        a, b = int(w.offsets[f]), int(w.offsets[f + 1])
        want, _, wst = ref.zippel_lift_step(np.ascontiguousarray(w.exps[a:b]), np.array([0, b - a], dtype=np.int64), w.anchors,
                                            w.samples, np.ascontiguousarray(w.vals[:, a:b]), w.p, 0, 1)
        assert not wst.any() and (got[:, a:b] == want).all()


# ------------------------------------------------------------------------------ balanced step, config 4
def balanced_inputs(ref, rw):
    """u_{j,s} = true value x per-probe factor h_s; skel = C x coefficients at c_0 (readings G3, G19, G20)."""
    p = rw.num.p
    c0 = int(rw.num.samples[0])
    f_scale = []
    for f in range(rw.num.F):
        i = int(rw.den.offsets[f]) + int(rw.low_den[f])
        a_low = sum(int(rw.den.planted[d, i]) * pow(c0, d, p) for d in range(rw.den.B)) % p
        f_scale.append(pow(a_low, -1, p))
    parts = {}
    for name, w in (("num", rw.num), ("den", rw.den)):
        true_vals, _ = probe_values(ref, w)
        skel = ref.poly_rows_eval(w.samples, w.planted, p)[0].astype(object)
        u = true_vals.astype(object)
        for f in range(w.F):
            o, e = int(w.offsets[f]), int(w.offsets[f + 1])
            skel[o:e] = skel[o:e] * f_scale[f] % p
            u[:, o:e] = u[:, o:e] * rw.h[: e - o].astype(object)[None, :] % p
        parts[name] = dict(exps=w.exps, offsets=w.offsets, skel=skel.astype(np.uint64), uvals=u.astype(np.uint64))
    return parts, f_scale


@pytest.mark.parametrize("basis", [0, 1])
def test_config4_balanced_parity_first_functions(zp, ref, basis):
    """configs[3] shape (nv = 5, t_N = 500, t_D = 200, B = 25), first 6 functions as a complete problem."""
    rw = wl.config(4, F=6)
    p = rw.num.p
    parts, f_scale = balanced_inputs(ref, rw)
    wn, wd, wst = ref.balanced_zippel_lift_step(parts["num"], parts["den"], rw.num.anchors, rw.num.samples, p, 0, basis)
    dev = {k: dict(exps=zp.to_dev(v["exps"]), offsets=v["offsets"], skel=zp.to_dev(v["skel"]),
                   uvals=zp.to_dev(v["uvals"])) for k, v in parts.items()}
    gn, gd, st = zp.balanced_zippel_lift_step(dev["num"], dev["den"], zp.to_dev(rw.num.anchors),
                                              zp.to_dev(rw.num.samples), p, 0, basis)
    assert not wst.any() and (zp.to_host(st) == wst).all()
    gn, gd = zp.to_host(gn), zp.to_host(gd)
    assert (gn == wn).all() and (gd == wd).all()
    if basis == 1:  # = C x planted, per function
        for w, g in ((rw.num, gn), (rw.den, gd)):
            for f in range(w.F):
                sl = slice(int(w.offsets[f]), int(w.offsets[f + 1]))
                assert (g[:, sl].astype(object) == w.planted[:, sl].astype(object) * f_scale[f] % p).all()


def test_balanced_zero_pivot_status(zp, ref):
    rw = wl.config(4, F=3, t=30)
    p = rw.num.p
    parts, _ = balanced_inputs(ref, rw)
    parts["num"]["uvals"][0, int(rw.num.offsets[1]) + 7] = 0  # u_{0,7} of function 1's numerator
    wn, wd, wst = ref.balanced_zippel_lift_step(parts["num"], parts["den"], rw.num.anchors, rw.num.samples, p, 0, 1)
    dev = {k: dict(exps=zp.to_dev(v["exps"]), offsets=v["offsets"], skel=zp.to_dev(v["skel"]),
                   uvals=zp.to_dev(v["uvals"])) for k, v in parts.items()}
    gn, gd, st = zp.balanced_zippel_lift_step(dev["num"], dev["den"], zp.to_dev(rw.num.anchors),
                                              zp.to_dev(rw.num.samples), p, 0, 1)
    st = zp.to_host(st)
    assert (st == wst).all() and st[1] == ((7 << 8) | zp.ST_ZERO_PIVOT)
    gn, gd = zp.to_host(gn), zp.to_host(gd)
    assert (gd == wd).all()
    for f in (0, 2):
        sl = slice(int(rw.num.offsets[f]), int(rw.num.offsets[f + 1]))
        assert (gn[:, sl] == wn[:, sl]).all()


def run_balanced_both(zp, ref, rw, parts, s0, basis):
    p = rw.num.p
    wn, wd, wst = ref.balanced_zippel_lift_step(parts["num"], parts["den"], rw.num.anchors, rw.num.samples, p, s0, basis)
    dev = {k: dict(exps=zp.to_dev(v["exps"]), offsets=v["offsets"], skel=zp.to_dev(v["skel"]),
                   uvals=zp.to_dev(v["uvals"])) for k, v in parts.items()}
    gn, gd, st = zp.balanced_zippel_lift_step(dev["num"], dev["den"], zp.to_dev(rw.num.anchors),
                                              zp.to_dev(rw.num.samples), p, s0, basis)
    return (wn, wd, wst), (zp.to_host(gn), zp.to_host(gd), zp.to_host(st))


@pytest.mark.parametrize("s0", [0, 1])
@pytest.mark.parametrize("ragged", [False, True])
def test_balanced_probe_offset_and_ragged_lengths(zp, ref, s0, ragged):
    """eq. (4) (readings G1, G3, G20) with probes at the powers s0 .. s0 + t - 1 and with functions
    of different lengths in one batch (k_balance's search over ragged offsets, the division by m_i of s0 = 1)."""
    if ragged:  # lengths around the CTA, warp and batched-inversion group sizes
        rw = wl.make_rational_workload("rag4g", wl.SEED_BASE + 45, 7, 6, [300, 7, 129, 1, 513, 64, 31], [12, 1, 90, 1, 257, 33, 128],
                                       24, 25, s0=s0)
    else:
        rw = wl.config(4, F=3, t=140)
    rw.num.s0 = rw.den.s0 = s0
    parts, f_scale = balanced_inputs(ref, rw)
    (wn, wd, wst), (gn, gd, st) = run_balanced_both(zp, ref, rw, parts, s0, 1)
    assert not wst.any() and (st == wst).all()
    assert (gn == wn).all() and (gd == wd).all()
    p = rw.num.p
    for w, g in ((rw.num, gn), (rw.den, gd)):  # = C x planted, per function
        for f in range(w.F):
            sl = slice(int(w.offsets[f]), int(w.offsets[f + 1]))
            assert (g[:, sl].astype(object) == w.planted[:, sl].astype(object) * f_scale[f] % p).all()


@pytest.mark.parametrize("s0", [0, 1])
def test_balanced_long_functions_cross_the_power_sum_blocks(zp, ref, s0):
    """Functions of more than 512 terms: k_power_sums takes the probes s in blocks of 512 (the table of a later block
    starts at m^(sb0 + s0)), the nodes in tiles of 64, and splits the nodes of a tile among lane groups where the last
    block is short; k_balance_apply's grid has several slot blocks and row blocks (B = 25 > ZP_BAL_ROWS)."""
    rw = wl.make_rational_workload("rag4l", wl.SEED_BASE + 47, 4, 6, [1100, 40, 1024, 577], [515, 1025, 3, 640], 24, 25, s0=s0)
    rw.num.s0 = rw.den.s0 = s0
    parts, f_scale = balanced_inputs(ref, rw)
    (wn, wd, wst), (gn, gd, st) = run_balanced_both(zp, ref, rw, parts, s0, 0)
    assert not wst.any() and (st == wst).all()
    assert (gn == wn).all() and (gd == wd).all()


def test_balanced_zero_pivots_in_a_ragged_batch(zp, ref):
    """Zero pivots u_{0,s} in several functions of a ragged batch, inside and at the ends of a warp's group of the
    batched inversion: status word (smallest probe index) and every other function's output as the oracle's."""
    rw = wl.make_rational_workload("rag4z", wl.SEED_BASE + 46, 5, 6, [140, 3, 129, 40, 260], [50, 2, 9, 33, 100], 24, 25)
    parts, _ = balanced_inputs(ref, rw)
    o = rw.num.offsets
    for f, ss in ((1, [2]), (2, [128, 5, 77]), (4, [0, 259])):
        for s in ss:
            parts["num"]["uvals"][0, int(o[f]) + s] = 0
    parts["den"]["uvals"][0, int(rw.den.offsets[3]) + 32] = 0
    (wn, wd, wst), (gn, gd, st) = run_balanced_both(zp, ref, rw, parts, 0, 0)
    assert (st == wst).all()
    F = rw.num.F
    assert st[1] == ((2 << 8) | zp.ST_ZERO_PIVOT) and st[2] == ((5 << 8) | zp.ST_ZERO_PIVOT) and st[4] == zp.ST_ZERO_PIVOT
    assert st[F + 3] == ((32 << 8) | zp.ST_ZERO_PIVOT) and st[0] == 0 and st[3] == 0
    for w, want, got, base in ((rw.num, wn, gn, 0), (rw.den, wd, gd, F)):
        for f in range(F):
            if st[base + f] == 0:
                sl = slice(int(w.offsets[f]), int(w.offsets[f + 1]))
                assert (got[:, sl] == want[:, sl]).all()


# ------------------------------------------------------------------------------ many tiny functions (F > 65535)
def test_more_functions_than_grid_rows(zp, ref):
    """F = 70 001 functions of 1 .. 3 terms: every kernel walks the functions with blockIdx.y strides of at most 65 535
    (grid_y in csrc/zippel_capi.cu); the polynomial and the balanced step, == the oracle."""
    F = 70_001
    r = np.random.Generator(np.random.Philox(key=[10, 4242]))
    ts = r.integers(1, 4, F)
    w = wl.make_box_workload("tiny", wl.SEED_BASE + 77, F, 3, ts, 6, 3, dense=True)
    vals, _ = probe_values(ref, w)
    got = lift_both(zp, ref, w, vals, 1)  # == the oracle inside
    assert (got == w.planted).all()
    # balanced: arbitrary residues as u and skel (parity with the oracle does not need a planted function)
    td = r.integers(1, 3, F)
    rw = wl.make_rational_workload("tinyr", wl.SEED_BASE + 78, F, 4, ts, td, 6, 7)
    parts = {n: dict(exps=q.exps, offsets=q.offsets, skel=q.meta["skel_standin"], uvals=q.vals)
             for n, q in (("num", rw.num), ("den", rw.den))}
    (wn, wd, wst), (gn, gd, st) = run_balanced_both(zp, ref, rw, parts, 1, 1)
    assert (st == wst).all() and (gn == wn).all() and (gd == wd).all()


# ------------------------------------------------------------------------------ non-canonical inputs (reading G22)
def test_inputs_offset_by_p_give_the_canonical_answer(zp, ref):
    """Anchors, samples and values passed as x + p (still below 2^64): same outputs as for the canonical residues, on
    the quadratic route, the B = 1 evaluation route and the sub-quadratic route, and for the balanced step."""
    import torch

    for ts, B in (([300, 41], 3), ([4200], 1), ([9000, 100], 2)):
        w = wl.make_box_workload("nc", wl.SEED_BASE + 90 + B, len(ts), 3, ts, 30, B)
        want, wnodes, wst = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, w.vals, w.p, 1, 1)
        up = lambda a: (a.astype(np.uint64) + np.uint64(w.p))
        got, st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(up(w.anchors)), zp.to_dev(up(w.samples)),
                                      zp.to_dev(up(w.vals)), w.p, 1, 1)
        assert not wst.any() and not zp.to_host(st).any() and (zp.to_host(got) == want).all()
        nodes = zp.to_dev(up(wnodes))
        c, st = zp.vandermonde_solve_batch(nodes, w.offsets, zp.to_dev(up(w.vals)), w.p, 0)
        wc, wst = ref.vandermonde_solve_batch(wnodes, w.offsets, w.vals, w.p, 0)
        assert (zp.to_host(c) == wc).all()
    rw = wl.config(4, F=2, t=70)
    parts = {n: dict(exps=q.exps, offsets=q.offsets, skel=q.meta["skel_standin"], uvals=q.vals)
             for n, q in (("num", rw.num), ("den", rw.den))}
    p = rw.num.p
    wn, wd, wst = ref.balanced_zippel_lift_step(parts["num"], parts["den"], rw.num.anchors, rw.num.samples, p, 0, 1)
    dev = {k: dict(exps=zp.to_dev(v["exps"]), offsets=v["offsets"], skel=zp.to_dev(v["skel"] + np.uint64(p)),
                   uvals=zp.to_dev(v["uvals"] + np.uint64(p))) for k, v in parts.items()}
    gn, gd, st = zp.balanced_zippel_lift_step(dev["num"], dev["den"], zp.to_dev(rw.num.anchors + np.uint64(p)),
                                              zp.to_dev(rw.num.samples + np.uint64(p)), p, 0, 1)
    assert (zp.to_host(st) == wst).all() and (zp.to_host(gn) == wn).all() and (zp.to_host(gd) == wd).all()


# ------------------------------------------------------------------------------ bindings on a non-current stream
def test_bindings_on_a_side_stream_without_a_workspace(zp, ref):
    """Every binding that allocates its own workspace and outputs does so on the stream the kernels are enqueued on
    (api._on): calls on a side stream, while the current stream keeps allocating and overwriting blocks, still give
    the oracle's numbers."""
    import torch

    w = wl.config(2, F=40)
    want, _, _ = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, w.vals, w.p, 0, 1)
    side = torch.cuda.Stream()
    de, da, ds, dv = (zp.to_dev(x) for x in (w.exps, w.anchors, w.samples, w.vals))
    torch.cuda.synchronize()
    outs = []
    for _ in range(4):
        got, st = zp.zippel_lift_step(de, w.offsets, da, ds, dv, w.p, 0, 1, stream=side)
        outs.append((got, st))
        for _ in range(8):  # churn on the current stream: blocks freed by the binding must not be handed out early
            junk = torch.full((1 << 20,), -1, dtype=torch.int64, device="cuda")
            del junk
    side.synchronize()
    torch.cuda.synchronize()
    for got, st in outs:
        assert not zp.to_host(st).any() and (zp.to_host(got) == want).all()


# ------------------------------------------------------------------------------ host-side argument checks
def test_argument_errors_are_reported_not_launched(zp):
    import torch

    d = torch.zeros(8, dtype=torch.int64, device="cuda")
    e = torch.zeros((8, 1), dtype=torch.int16, device="cuda")
    with pytest.raises(zp.ZippelError):
        zp.zippel_eval_nodes(e, d, 1 << 63)  # p >= 2^63
    with pytest.raises(zp.ZippelError):
        zp.zippel_eval_nodes(e, d, 100)  # p even
    with pytest.raises(zp.ZippelError):
        zp.vandermonde_solve_batch(d, [0, 8], d[None, :], P63, s0=2)
    with pytest.raises(zp.ZippelError):
        zp.vandermonde_solve_batch(d, [0, 8], d[None, :], P63, workspace=torch.empty(256, dtype=torch.uint8, device="cuda"))
