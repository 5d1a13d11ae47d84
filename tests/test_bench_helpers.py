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
    ts = [1000] * 4096
    total, ns = b.work_model(ts, 21, 4, True, False)
    assert ns == 4096 * 1000 * 1000 * (16 + 8 * 22)  # one multiply-add + (B + 1) MACs per (node, stage)
    assert total > ns and (total - ns) / ns < 0.05  # tree, Newton, nodes: a few per cent
    _, ns5 = b.work_model([1 << 19], 1, 10, False, False)
    assert ns5 == (1 << 38) * 20  # B = 1 route: two evaluations by MACs + the correlation
    _, ns_small = b.work_model([1000], 1, 10, False, False)
    assert ns_small == 1000 * 1000 * (16 + 8 * 2)  # below t = 4096 the general path
    tb, _ = b.work_model([500] * 4, 25, 5, True, True)
    tn, _ = b.work_model([500] * 4, 25, 5, True, False)
    assert tb - tn == 8 * 4 * 500 * 500  # balanced: one MAC per (probe, node) of the forward evaluation
    assert abs(b.IMAD_PEAK_TOPS - 148 * 64 * 1.965e-3) < 1e-9


def test_clock_sampler_without_nvidia_smi(monkeypatch):
    b = load_bench()
    monkeypatch.setenv("PATH", "/nonexistent")
    s = b.ClockSampler(0)
    out = s.stop(time.perf_counter() - 1, time.perf_counter())
    assert "reasons" in out and out["sm_mhz"] is None
