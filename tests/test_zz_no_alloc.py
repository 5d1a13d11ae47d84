"""zippel_extend_skeleton_static (include/zippel.h): the entry point that allocates nothing -- its scratch (function offsets
and the look-back descriptors of k_ext_fused) is a file-scope `static __device__` array inside the library instead of a
caller's workspace.  Its output == the existing path's (zippel_extend_skeleton with a workspace), bit for bit, on two
calls in a row that share the array: a larger batch first, then a smaller one whose blocks meet the first call's stale
tickets and flags unless the call clears them, then the first again.  Collected last (test_zz_*): a failure here must
not hide the parity tests under `pytest -x`.  Passes alone in a fresh process and after the other tests (the array is
looked up per device on first use, and nothing else in the library touches it)."""
import numpy as np
import pytest

from paper_2505_24256_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def zp():
    from paper_2505_24256_b200 import api

    api.lib()
    return api


def _batch(seed, ts, B, nv, holes):
    w = wl.make_box_workload("noalloc", wl.SEED_BASE + seed, len(ts), nv, ts, 40, B)
    coefs = w.planted.copy()
    for rows, cols in holes:
        coefs[rows, cols] = 0
    return w, coefs


def _static(zp, w, coefs, cap, outs=None):
    """the static entry point on outputs the caller owns (allocated before the call, poisoned so that stale contents show)"""
    import torch

    F, nv = w.F, w.exps.shape[1]
    if outs is None:
        outs = (torch.empty((cap, nv + 1), dtype=torch.int16, device="cuda"), torch.empty(cap, dtype=torch.int64, device="cuda"),
                torch.empty(F + 1, dtype=torch.int64, device="cuda"), torch.empty(F, dtype=torch.int32, device="cuda"))
    for o in outs:
        o.fill_(-7)
    zp.zippel_extend_skeleton_static(zp.to_dev(w.exps), w.offsets, zp.to_dev(coefs), w.p, *outs)
    torch.cuda.synchronize()
    return outs


def _same(zp, w, coefs, got, cap):
    import torch

    ee, ec, eo, ed = zp.zippel_extend_skeleton(zp.to_dev(w.exps), w.offsets, zp.to_dev(coefs), w.p, cap)
    torch.cuda.synchronize()
    ge, gc, go, gd = got
    assert torch.equal(go, eo) and torch.equal(gd, ed)
    n = min(int(eo[-1]), cap)
    assert n > 0
    assert torch.equal(gc[:n], ec[:n]) and torch.equal(ge[:n], ee[:n])


def test_static_scratch_entry_matches_the_workspace_path_on_consecutive_calls(zp):
    # 82 blocks of 1024 terms, ragged functions, vanished terms and a function of degree < B - 1
    big = _batch(131, [30000, 1, 2049, 2048, 7, 25000, 26000], 7, 3, [(slice(None), 5), (slice(4, None), slice(30001, 32050))])
    # 3 blocks: its blocks take the tickets 0 .. 2 and look back at descriptors the first call left set
    small = _batch(132, [2000, 900, 3], 5, 3, [(slice(None), 2001)])
    cap_big, cap_small = big[1].size, small[1].size
    _same(zp, *big, _static(zp, *big, cap_big), cap_big)
    _same(zp, *small, _static(zp, *small, cap_small), cap_small)
    _same(zp, *big, _static(zp, *big, cap_big), cap_big)
    _same(zp, *big, _static(zp, *big, 1000), 1000)  # truncated output, full count


def test_static_scratch_entry_allocates_nothing(zp):
    """The device allocator is not touched by the call (torch's allocator statistics are unchanged when the inputs and
    outputs exist beforehand; a cudaMalloc inside the library would show as less free device memory)."""
    import torch

    w, coefs = _batch(133, [5000, 4000], 6, 3, [])
    cap = coefs.size
    outs = _static(zp, w, coefs, cap)  # first call: symbol look-up, kernel attributes
    exps_d, coefs_d = zp.to_dev(w.exps), zp.to_dev(coefs)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    stats0 = torch.cuda.memory_stats()["allocation.all.allocated"]
    for _ in range(3):
        zp.zippel_extend_skeleton_static(exps_d, w.offsets, coefs_d, w.p, *outs)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == stats0
    assert free1 >= free0
    _same(zp, w, coefs, outs, cap)


def test_static_scratch_limit_is_a_clear_error(zp):
    """Beyond ZP_STATIC_SCRATCH_BYTES the call enqueues nothing and says so."""
    import torch

    lim = zp.zippel_static_scratch_bytes()
    assert lim == 1 << 20
    F = lim // 8 + 1  # the offsets alone exceed the array
    offsets = np.arange(F + 1, dtype=np.int64)
    exps = torch.zeros((F, 2), dtype=torch.int16, device="cuda")
    coefs = torch.ones((1, F), dtype=torch.int64, device="cuda")
    outs = (torch.empty((F, 3), dtype=torch.int16, device="cuda"), torch.full((F,), -7, dtype=torch.int64, device="cuda"),
            torch.empty(F + 1, dtype=torch.int64, device="cuda"), torch.empty(F, dtype=torch.int32, device="cuda"))
    n0 = zp.zippel_launch_count()
    with pytest.raises(zp.ZippelError) as e:
        zp.zippel_extend_skeleton_static(exps, offsets, coefs, wl.P63, *outs)
    assert "static scratch" in str(e.value) and f"code {zp.ZP_ERR_SCRATCH_LIMIT}" in str(e.value)
    torch.cuda.synchronize()
    assert zp.zippel_launch_count() == n0 and int(outs[1][0]) == -7
    # just inside the limit the same shape goes through
    F = (lim - 256 - 8 * 2) * 1024 // (8 * 1025) - 64  # 8 (F + 1) bytes of offsets + 8 (F / 1024 + 1) of descriptors
    offsets = np.arange(F + 1, dtype=np.int64)
    ne, nc, no, degs = outs[0][:F], outs[1][:F], outs[2][:F + 1], outs[3][:F]
    zp.zippel_extend_skeleton_static(exps[:F], offsets, coefs[:, :F].contiguous(), wl.P63, ne, nc, no, degs)
    torch.cuda.synchronize()
    assert int(no[F]) == F and int(degs.max()) == 0 and int(degs.min()) == 0 and bool((nc == 1).all())
