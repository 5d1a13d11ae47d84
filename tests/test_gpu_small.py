"""The fused single-launch path for small batches (csrc/small.cuh; BASELINE.json configs[0]): == the oracle on the
shapes that take it (F <= 32 functions of at most 128 terms, little work per lane) and just outside its gate (where
the general path answers), both bases, both probe offsets, several primes, status codes."""
import numpy as np
import pytest

from paper_2505_24256_b200 import workloads as wl

pytestmark = pytest.mark.gpu

P63 = wl.P63


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


def both(zp, ref, w, vals, s0, basis):
    import torch

    want, wnodes, wst = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, vals, w.p, s0, basis)
    dn = torch.zeros(w.T_tot, dtype=torch.int64, device="cuda")
    n0 = zp.zippel_launch_count()
    got, st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(w.anchors), zp.to_dev(w.samples), zp.to_dev(vals),
                                  w.p, s0, basis, nodes_out=dn)
    torch.cuda.synchronize()
    launches = zp.zippel_launch_count() - n0
    assert (zp.to_host(dn) == wnodes).all()
    return want, wst, zp.to_host(got), zp.to_host(st), launches


@pytest.mark.parametrize("ts,B,nv", [([50], 11, 2), ([1], 1, 1), ([1, 2, 3, 128, 127, 64, 65, 33], 3, 3), ([128] * 32, 2, 5),
                                     ([17, 40], 21, 4), ([5], 20, 2), ([10, 3], 24, 2), ([100, 31], 8, 3)])
@pytest.mark.parametrize("s0", [0, 1])
@pytest.mark.parametrize("basis", [0, 1])
def test_small_batches_take_one_launch_and_match(zp, ref, ts, B, nv, s0, basis):
    w = wl.make_box_workload("small", wl.SEED_BASE + 300 + len(ts) + B, len(ts), nv, ts, 12, B)
    want, wst, got, st, launches = both(zp, ref, w, w.vals, s0, basis)
    assert not wst.any() and (st == wst).all() and (got == want).all()
    assert launches == 1, "the small batch did not take the fused launch"


def test_config1_planted_recovery_through_the_fused_launch(zp, ref):
    w = wl.config(1, dense=True)
    nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
    at = ref.poly_rows_eval(w.samples, w.planted, w.p)
    vals = ref.power_sums(nodes, w.offsets, at, w.p, 0)
    want, wst, got, st, launches = both(zp, ref, w, vals, 0, 1)
    assert launches == 1 and not st.any() and (got == want).all() and (got == w.planted).all()


@pytest.mark.parametrize("p", [101, 65537, (1 << 31) - 1, (1 << 61) - 1])
def test_small_path_other_primes(zp, ref, p):
    r = np.random.Generator(np.random.Philox(key=[31, p & 0xFFFF]))
    ts = [7, 20, 1, 33] if p > 101 else [7, 20, 1, 12]
    F, nv, B = len(ts), 2, 5
    offs = np.zeros(F + 1, dtype=np.int64)
    offs[1:] = np.cumsum(ts)
    T = int(offs[-1])
    # distinct nodes need distinct exponent rows AND no collision mod a small p: draw anchors until the oracle is happy
    for attempt in range(200):
        exps = np.concatenate([wl.box_rows(r, t, nv, 9) for t in ts])
        anchors = wl.distinct_residues(r, 2, p, nv)
        samples = wl.distinct_residues(r, 1, p, B)
        vals = r.integers(0, p, (B, T), dtype=np.uint64)
        want, _, wst = ref.zippel_lift_step(exps, offs, anchors, samples, vals, p, 0, 1)
        if not wst.any():
            break
    else:
        pytest.skip("no collision-free draw")
    got, st = zp.zippel_lift_step(zp.to_dev(exps), offs, zp.to_dev(anchors), zp.to_dev(samples), zp.to_dev(vals), p, 0, 1)
    assert not zp.to_host(st).any() and (zp.to_host(got) == want).all()


def test_small_path_status_codes(zp, ref):
    """Duplicate node (two equal exponent rows), zero node with s0 = 1 (an anchor 0), duplicate sample: the status
    words of the oracle; the functions without a failure still match."""
    w = wl.make_box_workload("smallst", wl.SEED_BASE + 310, 3, 2, [9, 14, 6], 8, 4)
    exps = w.exps.copy()
    exps[int(w.offsets[1]) + 5] = exps[int(w.offsets[1]) + 2]  # function 1: terms 2 and 5 share a node
    want, _, wst = ref.zippel_lift_step(exps, w.offsets, w.anchors, w.samples, w.vals, w.p, 0, 1)
    got, st = zp.zippel_lift_step(zp.to_dev(exps), w.offsets, zp.to_dev(w.anchors), zp.to_dev(w.samples), zp.to_dev(w.vals),
                                  w.p, 0, 1)
    st, got = zp.to_host(st), zp.to_host(got)
    assert (st == wst).all() and st[1] == ((2 << 8) | zp.ST_DUPLICATE_NODE) and st[0] == 0 and st[2] == 0
    for f in (0, 2):
        sl = slice(int(w.offsets[f]), int(w.offsets[f + 1]))
        assert (got[:, sl] == want[:, sl]).all()
    # zero node with s0 = 1: anchor 0 and a term whose exponent on it is positive
    anchors = w.anchors.copy()
    anchors[0] = 0
    want, _, wst = ref.zippel_lift_step(w.exps, w.offsets, anchors, w.samples, w.vals, w.p, 1, 0)
    got, st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(anchors), zp.to_dev(w.samples), zp.to_dev(w.vals),
                                  w.p, 1, 0)
    assert (zp.to_host(st) == wst).all() and wst.any()
    # duplicate sample
    samples = w.samples.copy()
    samples[3] = samples[1]
    want, _, wst = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, samples, w.vals, w.p, 0, 0)
    got, st = zp.zippel_lift_step(zp.to_dev(w.exps), w.offsets, zp.to_dev(w.anchors), zp.to_dev(samples), zp.to_dev(w.vals),
                                  w.p, 0, 0)
    assert (zp.to_host(st) == wst).all() and (wst == ((3 << 8) | zp.ST_DUPLICATE_SAMPLE)).all()


@pytest.mark.parametrize("ts,B", [([129], 3), ([50] * 33, 3), ([128], 40)])
def test_just_outside_the_gate_takes_the_general_path(zp, ref, ts, B):
    w = wl.make_box_workload("notsmall", wl.SEED_BASE + 320 + B, len(ts), 3, ts, 12, B)
    want, wst, got, st, launches = both(zp, ref, w, w.vals, 0, 1)
    assert launches > 1 and not st.any() and (got == want).all()


def test_host_entry_small_batch(zp, ref):
    import torch

    w = wl.config(1)
    want, _, wst = ref.zippel_lift_step(w.exps, w.offsets, w.anchors, w.samples, w.vals, w.p, 0, 1)
    pin = lambda a: torch.from_numpy(a.view(np.int64) if a.dtype == np.uint64 else a.view(np.int16)).pin_memory()
    h_out = torch.empty(w.vals.shape, dtype=torch.int64).pin_memory()
    h_st = torch.empty(w.F, dtype=torch.int32).pin_memory()
    ws = torch.empty(zp.host_workspace_bytes(w.offsets, w.nv, w.B), dtype=torch.uint8, device="cuda")
    zp.zippel_lift_step_host(pin(w.exps), w.offsets, pin(w.anchors), pin(w.samples), pin(w.vals), w.p, h_out, h_st, ws, 0, 1)
    torch.cuda.synchronize()
    assert not h_st.numpy().any() and (h_out.numpy().view(np.uint64) == want).all()
