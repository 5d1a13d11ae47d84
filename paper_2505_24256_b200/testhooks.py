"""Bindings of libzippel_test.so (include/zippel_test.h): the product's sources compiled with -DZP_TEST_HOOKS.

Used by tests/ and by the ubench module only.  The test build holds the product's entry points too, with its own
copy of the process-wide state: `with routed():` sends the bindings of api.py through it for the duration of the
block, so that a test can set a dump hook and then call api.vandermonde_solve_batch on the same library.
"""
from __future__ import annotations

import contextlib
import ctypes as C
import os
from typing import Optional

import numpy as np
import torch

from . import api
from . import build as _build

EXPORTS = ("zippel_modarith_selftest", "zippel_ubench", "zippel_test_ntt_constants", "zippel_test_polymul",
           "zippel_test_polymul_workspace_bytes", "zippel_test_subq_dump")

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        path = _build.TEST_SO_PATH
        if not os.path.exists(path) or _build.test_is_stale():
            path = _build.build_test()
        L = api.declare(C.CDLL(path))
        vp, i32, i64, u64, sz = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_size_t
        L.zippel_modarith_selftest.argtypes = [i32, vp, vp, i64, u64, vp, vp]
        L.zippel_ubench.argtypes = [i32, i32, i32, u64, vp, C.POINTER(C.c_double), vp]
        L.zippel_test_ntt_constants.restype = None
        L.zippel_test_ntt_constants.argtypes = [vp]
        L.zippel_test_polymul_workspace_bytes.restype = sz
        L.zippel_test_polymul_workspace_bytes.argtypes = [i64, i64]
        L.zippel_test_polymul.argtypes = [vp, i64, vp, i64, u64, vp, i32, vp, sz, vp]
        L.zippel_test_subq_dump.argtypes = [i32, vp]
        _lib = L
    return _lib


@contextlib.contextmanager
def routed():
    """Route api.py's bindings through the test build inside the block (then back to the product library)."""
    prev = api.lib()
    api.use_library(lib())
    try:
        yield
    finally:
        api.use_library(prev)


def ntt_constants() -> dict:
    out = np.zeros(7, dtype=np.uint64)
    lib().zippel_test_ntt_constants(out.ctypes.data)
    return {"q": [int(x) for x in out[:3]], "w": [int(x) for x in out[3:6]], "log_order": int(out[6])}


def zippel_modarith_selftest(op: int, a: torch.Tensor, b: Optional[torch.Tensor], p: int, stream=None):
    """(a0) out[i] = op(a[i], b[i]) mod p on the device (see include/zippel_test.h)."""
    api._need_cuda()
    n = a.numel()
    out = torch.empty(1 if op == 5 else n, dtype=torch.int64, device=a.device)
    api._check(lib().zippel_modarith_selftest(op, api._ptr(a), api._ptr(b), n, p, api._ptr(out), api._stream(stream)),
               "zippel_modarith_selftest")
    return out


def zippel_ubench(kind: int, iters: int, blocks: int, p: int, out: torch.Tensor, stream=None) -> float:
    """Enqueue one micro-benchmark launch (csrc/ubench.cuh); returns the lane-statements it executes."""
    api._need_cuda()
    n = C.c_double(0.0)
    api._check(lib().zippel_ubench(kind, iters, blocks, p, api._ptr(out), C.byref(n), api._stream(stream)), "zippel_ubench")
    return n.value


def polymul(a: torch.Tensor, b: torch.Tensor, p: int, roundtrip: bool = False, stream=None) -> torch.Tensor:
    """a * b mod p through the three-prime NTT engine (or, roundtrip, inverse(forward([a | b])) / n per prime)."""
    api._need_cuda()
    na, nb = a.numel(), b.numel()
    need = lib().zippel_test_polymul_workspace_bytes(na, nb)
    ws = torch.empty(need, dtype=torch.uint8, device=a.device)
    n = 1 << max(1, (na + nb - 2).bit_length())
    out = torch.empty(6 * n if roundtrip else na + nb - 1, dtype=torch.int64, device=a.device)
    api._check(lib().zippel_test_polymul(api._ptr(a), na, api._ptr(b), nb, p, api._ptr(out), int(roundtrip), api._ptr(ws),
                                         ws.numel(), api._stream(stream)), "zippel_test_polymul")
    ws.record_stream(torch.cuda.current_stream() if stream is None else stream)
    return out


def subq_dump(stage: int, out: Optional[torch.Tensor]):
    api._check(lib().zippel_test_subq_dump(stage, api._ptr(out) if out is not None else None), "zippel_test_subq_dump")
