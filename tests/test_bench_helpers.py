"""Host-side helpers of bench.py (no GPU): the algorithmic-work model behind roofline.frac and the clock sampler's
fallback when nvidia-smi is absent."""
import importlib.util
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def load_bench():
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    sys.modules["bench_mod"] = mod
    spec.loader.exec_module(mod)
    return mod


def test_work_model_matches_design_md():
    b = load_bench()
    ts = [900] * 4096  # below the batch threshold of the sub-quadratic route: the quadratic kernels
    total, ns = b.work_model(ts, 21, 4, True, False)
    assert ns == 4096 * 900 * 900 * (16 + 8 * 22)  # one multiply-add + (B + 1) MACs per (node, stage)
    assert total > ns and (total - ns) / ns < 0.05  # tree, Newton, nodes: a few per cent
    # BASELINE.json configs[1] (t = 1000, 4096 functions) is above it: two 512-node leaves and one tree level per function
    tot2, ns2 = b.work_model([1000] * 4096, 21, 4, True, False)
    assert b.sq_threshold([1000] * 4096, 21) == 960 and b.sq_threshold([1000] * 60, 21) == 2048
    assert ns2 == 4096 * b.subq_units(1000, 21)[0] and ns2 < 0.75 * 4096 * 1000 * 1000 * (16 + 8 * 22)
    _, ns5 = b.work_model([4096], 1, 10, False, False)
    assert ns5 == (1 << 24) * 20  # B = 1 route below the sub-quadratic threshold: two evaluations by MACs + the correlation
    _, ns_small = b.work_model([1000], 1, 10, False, False)
    assert ns_small == 1000 * 1000 * (16 + 8 * 2)  # below t = 4096 the general path
    tb, _ = b.work_model([500] * 4, 25, 5, True, True)
    tn, _ = b.work_model([500] * 4, 25, 5, True, False)
    assert tb - tn == 8 * 4 * 500 * 500  # balanced: one MAC per (probe, node) of the forward evaluation
    assert abs(b.IMAD_PEAK_TOPS - 148 * 64 * 1.965e-3) < 1e-9


def test_work_model_of_the_subquadratic_route():
    """bench.py subq_units counts the plan of csrc/zippel_capi.cu:sq_solve; checked here against the counts written
    out by hand for t = 4096 (three levels above the 512-node leaves), B = 1, and for its growth (t log^2 t)."""
    from math import log2

    b = load_bench()
    ntt = lambda n: 3 * (n / 2) * log2(n) * 16
    pw = lambda n: 3 * n * 36
    crt = lambda n: n * 90
    tot, parts = b.subq_units(4096, 1)  # three levels above the 512-node leaves: (pairs, n) = (4, 1024), (2, 2048), (1, 4096)
    levels = ((4, 1024), (2, 2048), (1, 4096))
    pw1 = lambda n: 3 * n * 18  # one Montgomery product per word: scaling a kept transform; the down-tree's pointwise product
    up = sum(P * (3 * ntt(n) + pw(n) + 2 * pw1(n)) + crt(4096) for P, n in levels)
    assert parts["up_tree"] == up
    V = 2
    down = sum(V * (P * (3 * ntt(n) + 2 * pw1(n)) + crt(4096)) for P, n in levels)  # the siblings' transforms are kept
    assert parts["down_tree"] == down
    assert parts["leaves"] == 8 * 512 * 512 * (4 + 16 + 2 * 8)
    t19, _ = b.subq_units(1 << 19, 1)
    t20, _ = b.subq_units(1 << 20, 1)
    assert 2.0 < t20 / t19 < 2.3  # quasi-linear
    total, ns = b.work_model([1 << 19], 1, 10, False, False)
    assert ns == t19 and total == t19 + 16 * 9 * (1 << 19)  # + the node evaluation
    quad = (1 << 38) * 20
    assert quad / t19 > 100  # the quadratic B = 1 route does over 100 x the multiplier work at t = 2^19


def test_clock_sampler_without_nvidia_smi(monkeypatch):
    b = load_bench()
    monkeypatch.setenv("PATH", "/nonexistent")
    s = b.ClockSampler(0)
    out = s.stop(time.perf_counter() - 1, time.perf_counter())
    assert "reasons" in out and out["sm_mhz"] is None
