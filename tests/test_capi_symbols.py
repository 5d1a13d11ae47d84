"""CPU-only: the C-ABI library builds (nvcc cross-compiles), loads, and exports every symbol that
include/zippel.h declares; host-side argument checks answer without a device."""
import ctypes as C
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header="zippel.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+char\s*\*|size_t|int|void|unsigned long long)\s+([a-z_0-9]+)\s*\(", src, flags=re.M)
    assert len(names) >= 6
    return names


def test_library_exports_every_declared_symbol():
    from paper_2505_24256_b200 import api

    L = api.lib()
    names = declared_symbols()
    for n in names:
        assert hasattr(L, n), n
    assert set(names) == set(api.EXPORTS)
    for must in ("zippel_eval_nodes", "vandermonde_solve_batch", "newton_interp_batch", "zippel_lift_step",
                 "balanced_zippel_lift_step"):  # BASELINE.json north_star
        assert must in names


def test_test_library_exports_every_declared_symbol():
    """include/zippel_test.h: the test build has the hooks AND the product's entry points; the product has no hook."""
    from paper_2505_24256_b200 import api, testhooks

    T = testhooks.lib()
    hooks = declared_symbols("zippel_test.h")
    assert set(hooks) == set(testhooks.EXPORTS)
    for n in hooks + declared_symbols():
        assert hasattr(T, n), n
    L = api.lib()
    for n in hooks:
        assert not hasattr(L, n), f"the product library exports the test hook {n}"


def test_long_skeleton_workspace_and_limits():
    """Host logic of the sub-quadratic route (no device): the workspace grows when a function crosses the
    threshold, shrinks back when the threshold is raised, and a function of 2^23 terms is refused."""
    from paper_2505_24256_b200 import api

    L = api.lib()
    offs = np.array([0, 1000, 21000, 22000], dtype=np.int64)  # short, long, short
    base = L.zippel_workspace_bytes(offs.ctypes.data, 3, 3, 0)
    assert L.zippel_set_tuning(api.TUNE_SUBQ_MIN_T, 1 << 22) == api.ZP_OK
    quad = L.zippel_workspace_bytes(offs.ctypes.data, 3, 3, 0)
    assert L.zippel_set_tuning(api.TUNE_SUBQ_MIN_T, 0) == api.ZP_OK  # back to the built-in rule
    assert quad < base and quad % 256 == 0
    assert L.zippel_set_tuning(api.TUNE_SUBQ_MIN_T, -1) == api.ZP_ERR_ARG
    assert L.zippel_set_tuning(99, 1) == api.ZP_ERR_ARG
    # the built-in rule (include/zippel.h): one function of 5000 terms is long for 21 right-hand sides, not for one;
    # a batch of 32 such functions is long for any B
    def grows(o, B):
        L.zippel_set_tuning(api.TUNE_SUBQ_MIN_T, 1 << 22)
        q = L.zippel_workspace_bytes(o.ctypes.data, len(o) - 1, B, 0)
        L.zippel_set_tuning(api.TUNE_SUBQ_MIN_T, 0)
        return L.zippel_workspace_bytes(o.ctypes.data, len(o) - 1, B, 0) > q
    one = np.array([0, 5000], dtype=np.int64)
    many = np.arange(33, dtype=np.int64) * 5000
    assert not grows(one, 1) and not grows(one, 5) and grows(one, 9) and grows(one, 21)
    assert grows(many, 1) and grows(many, 21)
    assert grows(np.arange(4097, dtype=np.int64) * 1000, 21)      # configs[1]: 4096 functions of t = 1000 take the route,
    assert not grows(np.arange(4097, dtype=np.int64) * 900, 21)    # functions of 900 terms do not,
    assert not grows(np.arange(61, dtype=np.int64) * 1000, 21)     # and neither do 60 functions of 1000 (too few to fill the GPU)
    big = np.array([0, 1 << 23], dtype=np.int64)
    assert L.zippel_workspace_bytes(big.ctypes.data, 1, 1, 0) == 0
    ok = np.array([0, (1 << 23) - 1], dtype=np.int64)
    assert L.zippel_workspace_bytes(ok.ctypes.data, 1, 1, 0) > 0


def test_host_side_checks_without_device():
    from paper_2505_24256_b200 import api

    L = api.lib()
    offs = np.array([0, 10, 30], dtype=np.int64)
    n = L.zippel_workspace_bytes(offs.ctypes.data, 2, 5, 0)
    nb = L.zippel_workspace_bytes(offs.ctypes.data, 2, 5, api.WS_BALANCED)
    assert n > 0 and n % 256 == 0 and nb >= n + 8 * 30 * 5
    assert L.zippel_workspace_bytes(offs.ctypes.data, 2, 65, 0) == 0  # B > ZP_MAX_B
    bad = np.array([0, 10, 10], dtype=np.int64)  # empty function
    assert L.zippel_workspace_bytes(bad.ctypes.data, 2, 5, 0) == 0
    assert L.zippel_host_workspace_bytes(offs.ctypes.data, 2, 3, 5) > n
    assert L.zippel_strerror(1) == b"bad argument"
    # argument errors come back before anything is enqueued (no device needed)
    assert L.zippel_eval_nodes(None, 10, 2, None, (1 << 63) - 25, None, None) == api.ZP_ERR_ARG
    assert L.zippel_eval_nodes(1, 10, 2, 1, 1 << 63, 1, None) == api.ZP_ERR_ARG  # p >= 2^63


def test_no_cpu_fallback():
    import pytest
    import torch

    from paper_2505_24256_b200 import api

    if torch.cuda.is_available():
        pytest.skip("device present")
    with pytest.raises(api.ZippelError):
        api.zippel_eval_nodes(torch.zeros((4, 2), dtype=torch.int16), torch.zeros(2, dtype=torch.int64), 101)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2505_24256_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle|libzippel_ref|zippel_ref\.h|oracle/", re.M)
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dp, f)).read()), f
