"""Thin Python binding of libzippel.so (include/zippel.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C-ABI; PyTorch is used for device
memory and streams.  Function names equal the C entry points.  Residues travel as 64-bit tensors
(torch.int64 holding the uint64 bit pattern; `to_dev` / `to_host` convert from / to numpy uint64).

There is NO CPU fallback: importing works anywhere (so that the symbol test can run), but every
compute call raises if the library or a CUDA device is missing.
"""
from __future__ import annotations

import contextlib
import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np
import torch

from . import build as _build

ZP_OK, ZP_ERR_ARG, ZP_ERR_WORKSPACE, ZP_ERR_CUDA, ZP_ERR_SCRATCH_LIMIT = 0, 1, 2, 3, 4
ST_DUPLICATE_NODE, ST_DUPLICATE_SAMPLE, ST_ZERO_PIVOT = 16, 17, 18
BASIS_NEWTON, BASIS_MONOMIAL = 0, 1
WS_BALANCED = 1
MAX_NV, MAX_B = 32, 64

EXPORTS = (
    "zippel_strerror", "zippel_workspace_bytes", "zippel_eval_nodes", "vandermonde_solve_batch",
    "newton_interp_batch", "zippel_lift_step", "zippel_power_sums", "balanced_zippel_lift_step",
    "zippel_lift_step_host", "zippel_host_workspace_bytes", "zippel_profile_events",
    "zippel_launch_count", "thiele_reconstruct_batch", "zippel_extend_skeleton", "crt_rational_reconstruct_batch",
    "zippel_set_tuning", "zippel_shutdown", "zippel_extend_skeleton_static", "zippel_static_scratch_bytes",
)
TUNE_SUBQ_MIN_T = 1
SUBQ_MIN_T_DEFAULT = 0  # g_subq_min_t in csrc/zippel_capi.cu: 0 = the built-in rule (sq_threshold)
K_EVAL_NODES, K_MASTER_POLY, K_NODE_SOLVE, K_NEWTON, K_POWER_SUMS, K_BALANCE, K_LEAF_SOLVE = 1, 2, 3, 5, 6, 7, 8


class ZippelError(RuntimeError):
    pass


class _Part(C.Structure):
    _fields_ = [("exps", C.c_void_p), ("h_offsets", C.c_void_p), ("skel", C.c_void_p),
                ("uvals", C.c_void_p), ("out", C.c_void_p)]


_lib = None


def declare(L: C.CDLL) -> C.CDLL:
    """Argument types of the entry points of include/zippel.h on a loaded library."""
    vp, i32, i64, u64, sz = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_size_t
    L.zippel_strerror.restype = C.c_char_p
    L.zippel_strerror.argtypes = [i32]
    L.zippel_workspace_bytes.restype = sz
    L.zippel_workspace_bytes.argtypes = [vp, i32, i32, i32]
    L.zippel_host_workspace_bytes.restype = sz
    L.zippel_host_workspace_bytes.argtypes = [vp, i32, i32, i32]
    L.zippel_eval_nodes.argtypes = [vp, i64, i32, vp, u64, vp, vp]
    L.vandermonde_solve_batch.argtypes = [vp, vp, i32, vp, i32, i32, u64, vp, vp, vp, sz, vp]
    L.newton_interp_batch.argtypes = [vp, i32, vp, i64, i64, u64, i32, vp, vp, vp, sz, vp]
    L.zippel_lift_step.argtypes = [vp, vp, i32, i32, vp, vp, i32, i32, vp, u64, i32, vp, vp, vp, vp, sz, vp]
    L.zippel_lift_step_host.argtypes = [vp, vp, i32, i32, vp, vp, i32, i32, vp, u64, i32, vp, vp, vp, sz, vp]
    L.zippel_power_sums.argtypes = [vp, vp, i32, vp, i32, i32, u64, vp, vp, sz, vp]
    L.balanced_zippel_lift_step.argtypes = [C.POINTER(_Part), C.POINTER(_Part), i32, i32, vp, vp, i32, i32,
                                            u64, i32, vp, vp, sz, vp]
    L.zippel_profile_events.argtypes = [i32, vp, vp]
    L.thiele_reconstruct_batch.argtypes = [vp, i32, vp, C.c_int64, C.c_int64, u64, vp, vp, vp, vp, vp, vp, C.c_size_t, vp]
    L.zippel_extend_skeleton.argtypes = [vp, vp, i32, i32, vp, i32, u64, vp, vp, C.c_int64, vp, vp, vp, C.c_size_t, vp]
    L.crt_rational_reconstruct_batch.argtypes = [vp, vp, C.c_int64, u64, u64, vp, vp, vp, vp]
    L.zippel_extend_skeleton_static.argtypes = [vp, vp, i32, i32, vp, i32, u64, vp, vp, C.c_int64, vp, vp, vp]
    L.zippel_static_scratch_bytes.argtypes = []
    L.zippel_static_scratch_bytes.restype = C.c_size_t
    L.zippel_launch_count.restype = C.c_ulonglong
    L.zippel_launch_count.argtypes = []
    L.zippel_set_tuning.argtypes = [i32, i64]
    L.zippel_shutdown.argtypes = []
    return L


def lib() -> C.CDLL:
    """Load libzippel.so (building it with nvcc if it is missing or stale).  Fails loudly."""
    global _lib
    if _lib is None:
        path = _build.SO_PATH
        if not os.path.exists(path) or _build.is_stale():
            path = _build.build()
        _lib = declare(C.CDLL(path))
    return _lib


def use_library(L: C.CDLL):
    """Route every binding of this module through an already loaded library (testhooks.routed(): the test build
    holds the same entry points plus the hooks, with its own process-wide state)."""
    global _lib
    _lib = L


def _need_cuda():
    if not torch.cuda.is_available():
        raise ZippelError("no CUDA device: libzippel has no CPU fallback")


def _check(rc: int, what: str):
    if rc != ZP_OK:
        raise ZippelError(f"{what}: {lib().zippel_strerror(rc).decode()} (code {rc})")


def _stream(stream) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _on(stream):
    """Context in which the bindings allocate their temporaries and outputs: the stream the kernels are enqueued
    on, so that the caching allocator orders every reuse of those blocks after the kernels (a tensor allocated
    on another stream could be handed out again while they are still in flight)."""
    return contextlib.nullcontext() if stream is None else torch.cuda.stream(stream)


_NO_CTX = contextlib.nullcontext()


def _on_if_allocating(stream, *buffers):
    """_on(stream) when the binding has to allocate one of `buffers` (passed as None); nothing to enter when the caller
    brought them all -- torch's stream context costs more host time than a small lifting step takes on the GPU."""
    return _on(stream) if any(b is None for b in buffers) else _NO_CTX


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device-resident contiguous tensor expected"
    return t.data_ptr()


def _offs(offsets) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(offsets), dtype=np.int64)


# ---- numpy <-> device helpers (uint64 / uint16 bit patterns) ------------------------------------
def to_dev(a: np.ndarray, device="cuda") -> torch.Tensor:
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint64:
        return torch.from_numpy(a.view(np.int64)).to(device)
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16)).to(device)
    return torch.from_numpy(a).to(device)


def to_host(t: torch.Tensor) -> np.ndarray:
    a = t.detach().cpu().numpy()
    if a.dtype == np.int64:
        return a.view(np.uint64)
    if a.dtype == np.int16:
        return a.view(np.uint16)
    return a


def workspace_bytes(offsets, B: int, flags: int = 0) -> int:
    o = _offs(offsets)
    n = lib().zippel_workspace_bytes(o.ctypes.data, len(o) - 1, B, flags)
    if n == 0:
        raise ZippelError("zippel_workspace_bytes: bad argument")
    return int(n)


def alloc_workspace(offsets, B: int, flags: int = 0, device="cuda") -> torch.Tensor:
    _need_cuda()
    return torch.empty(workspace_bytes(offsets, B, flags), dtype=torch.uint8, device=device)


# ---- entry points ------------------------------------------------------------------------------------
def zippel_eval_nodes(exps: torch.Tensor, anchors: torch.Tensor, p: int, out: Optional[torch.Tensor] = None,
                      stream=None) -> torch.Tensor:
    """(a1) nodes m_i = prod_j y_j^{e_ij}; exps int16-view [T_tot, nv], anchors [nv]."""
    _need_cuda()
    with _on(stream):
        T_tot, nv = exps.shape
        if out is None:
            out = torch.empty(T_tot, dtype=torch.int64, device=exps.device)
        _check(lib().zippel_eval_nodes(_ptr(exps), T_tot, nv, _ptr(anchors), p, _ptr(out), _stream(stream)),
               "zippel_eval_nodes")
        return out


def vandermonde_solve_batch(nodes: torch.Tensor, offsets, vals: torch.Tensor, p: int, s0: int = 0,
                            out: Optional[torch.Tensor] = None, status: Optional[torch.Tensor] = None,
                            workspace: Optional[torch.Tensor] = None, stream=None):
    """(a2)-(a4); vals [B, T_tot] -> (coefs [B, T_tot], status [F])."""
    _need_cuda()
    with _on(stream):
        o = _offs(offsets)
        F, B = len(o) - 1, vals.shape[0]
        if out is None:
            out = torch.empty_like(vals)
        if status is None:
            status = torch.empty(F, dtype=torch.int32, device=vals.device)
        if workspace is None:
            workspace = alloc_workspace(o, B)
        _check(lib().vandermonde_solve_batch(_ptr(nodes), o.ctypes.data, F, _ptr(vals), B, s0, p, _ptr(out),
                                             _ptr(status), _ptr(workspace), workspace.numel(), _stream(stream)),
               "vandermonde_solve_batch")
        return out, status


def newton_interp_batch(samples: torch.Tensor, vals: torch.Tensor, p: int, basis: int = 0,
                        out: Optional[torch.Tensor] = None, status: Optional[torch.Tensor] = None,
                        workspace: Optional[torch.Tensor] = None, stream=None):
    """(a5); vals [B, n] (row j = values at c_j) -> (out [B, n], status [1]).  out may alias vals."""
    _need_cuda()
    with _on(stream):
        B, n = vals.shape
        ld = vals.stride(0) if B > 1 else n
        assert vals.stride(1) == 1
        if out is None:
            out = torch.empty_like(vals)
        if status is None:
            status = torch.empty(1, dtype=torch.int32, device=vals.device)
        if workspace is None:
            workspace = alloc_workspace([0, 1], B)
        _check(lib().newton_interp_batch(samples.data_ptr(), B, vals.data_ptr(), n, ld, p, basis, out.data_ptr(),
                                         _ptr(status), _ptr(workspace), workspace.numel(), _stream(stream)),
               "newton_interp_batch")
        return out, status


def zippel_lift_step(exps: torch.Tensor, offsets, anchors: torch.Tensor, samples: torch.Tensor,
                     vals: torch.Tensor, p: int, s0: int = 0, basis: int = 0,
                     out: Optional[torch.Tensor] = None, nodes_out: Optional[torch.Tensor] = None,
                     status: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
                     stream=None):
    """(a1)-(a5): one lifting step; returns (out [B, T_tot], status [F])."""
    _need_cuda()
    with _on_if_allocating(stream, out, status, workspace):
        o = _offs(offsets)
        F, B = len(o) - 1, vals.shape[0]
        nv = exps.shape[1]
        if out is None:
            out = torch.empty_like(vals)
        if status is None:
            status = torch.empty(F, dtype=torch.int32, device=vals.device)
        if workspace is None:
            workspace = alloc_workspace(o, B)
        _check(lib().zippel_lift_step(_ptr(exps), o.ctypes.data, F, nv, _ptr(anchors), _ptr(samples), B, s0,
                                      _ptr(vals), p, basis, _ptr(out), _ptr(nodes_out), _ptr(status),
                                      _ptr(workspace), workspace.numel(), _stream(stream)),
               "zippel_lift_step")
        return out, status


def zippel_power_sums(nodes: torch.Tensor, offsets, coef: torch.Tensor, p: int, s0: int = 0,
                      out: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None, stream=None):
    """(a6) forward evaluation R_{b,s} = sum_i a_{b,i} m_i^(s+s0); coef [B, T_tot] -> out [B, T_tot]."""
    _need_cuda()
    with _on(stream):
        o = _offs(offsets)
        if coef.dim() == 1:
            coef = coef[None, :]
        B = coef.shape[0]
        if out is None:
            out = torch.empty_like(coef)
        if workspace is None:
            workspace = alloc_workspace(o, B)
        _check(lib().zippel_power_sums(_ptr(nodes), o.ctypes.data, len(o) - 1, _ptr(coef), B, s0, p, _ptr(out),
                                       _ptr(workspace), workspace.numel(), _stream(stream)), "zippel_power_sums")
        return out


def balanced_zippel_lift_step(num: dict, den: dict, anchors: torch.Tensor, samples: torch.Tensor, p: int,
                              s0: int = 0, basis: int = 0, status: Optional[torch.Tensor] = None,
                              workspace: Optional[torch.Tensor] = None, stream=None):
    """(a6) balanced step; num / den: dicts with device tensors exps, skel, uvals, host offsets and an
    optional out.  Returns (out_num, out_den, status [2F])."""
    _need_cuda()
    with _on(stream):
        keep, parts = [], []
        F = len(num["offsets"]) - 1
        nv = num["exps"].shape[1]
        B = num["uvals"].shape[0]
        for d in (num, den):
            o = _offs(d["offsets"])
            out = d.get("out")
            if out is None:
                out = torch.empty_like(d["uvals"])
            keep.append((o, out))
            parts.append(_Part(_ptr(d["exps"]), o.ctypes.data, _ptr(d["skel"]), _ptr(d["uvals"]), _ptr(out)))
        if status is None:
            status = torch.empty(2 * F, dtype=torch.int32, device=anchors.device)
        if workspace is None:
            big = max((num, den), key=lambda d: int(_offs(d["offsets"])[-1]))
            workspace = alloc_workspace(big["offsets"], B, WS_BALANCED)
        _check(lib().balanced_zippel_lift_step(C.byref(parts[0]), C.byref(parts[1]), F, nv, _ptr(anchors),
                                               _ptr(samples), B, s0, p, basis, _ptr(status), _ptr(workspace),
                                               workspace.numel(), _stream(stream)), "balanced_zippel_lift_step")
        return keep[0][1], keep[1][1], status


# ---- host-buffer entry (the e2e path: copies inside the call) -----------------------------------------
def host_workspace_bytes(offsets, nv: int, B: int) -> int:
    o = _offs(offsets)
    n = lib().zippel_host_workspace_bytes(o.ctypes.data, len(o) - 1, nv, B)
    if n == 0:
        raise ZippelError("zippel_host_workspace_bytes: bad argument")
    return int(n)


def zippel_lift_step_host(h_exps: torch.Tensor, offsets, h_anchors: torch.Tensor, h_samples: torch.Tensor,
                          h_vals: torch.Tensor, p: int, h_out: torch.Tensor, h_status: torch.Tensor,
                          workspace: torch.Tensor, s0: int = 0, basis: int = 0, stream=None):
    """zippel_lift_step on HOST (pinned) buffers: H2D of exps/anchors/samples/vals, the step, D2H of out and
    status, all enqueued on `stream` by the library; `workspace` is device scratch of
    host_workspace_bytes() bytes.  Asynchronous: synchronise the stream before reading h_out."""
    _need_cuda()
    o = _offs(offsets)
    F, B = len(o) - 1, h_vals.shape[0]
    nv = h_exps.shape[1]
    for t in (h_exps, h_anchors, h_samples, h_vals, h_out, h_status):
        assert not t.is_cuda and t.is_contiguous()
    _check(lib().zippel_lift_step_host(h_exps.data_ptr(), o.ctypes.data, F, nv, h_anchors.data_ptr(),
                                       h_samples.data_ptr(), B, s0, h_vals.data_ptr(), p, basis,
                                       h_out.data_ptr(), h_status.data_ptr(), _ptr(workspace), workspace.numel(),
                                       _stream(stream)), "zippel_lift_step_host")
    return h_out, h_status


def zippel_profile_events(kernel: int, ev_start: Optional[torch.cuda.Event] = None,
                          ev_stop: Optional[torch.cuda.Event] = None):
    """Measurement hook: later calls record ev_start / ev_stop around the launches of `kernel` (K_* above);
    kernel = 0 switches it off.  The events must be created with enable_timing=True."""
    if kernel:
        for ev in (ev_start, ev_stop):
            if not ev.cuda_event:  # torch creates the CUDA event lazily
                ev.record()
        _check(lib().zippel_profile_events(kernel, ev_start.cuda_event, ev_stop.cuda_event), "zippel_profile_events")
    else:
        _check(lib().zippel_profile_events(0, None, None), "zippel_profile_events")


def zippel_launch_count() -> int:
    """Kernels enqueued by the library in this process so far."""
    return int(lib().zippel_launch_count())


def zippel_set_tuning(key: int, value: int):
    """Process-wide tuning knob (TUNE_SUBQ_MIN_T: shortest skeleton that takes the sub-quadratic route)."""
    _check(lib().zippel_set_tuning(key, value), "zippel_set_tuning")


def zippel_shutdown():
    _check(lib().zippel_shutdown(), "zippel_shutdown")


ST_THIELE_DEGENERATE = 20


def thiele_reconstruct_batch(points: torch.Tensor, vals: torch.Tensor, p: int, want_cf: bool = True,
                             workspace: Optional[torch.Tensor] = None, stream=None):
    """(f2) eq. (2): vals [T, n] -> (num [T, n], den [T, n], degs [2, n] int32, cf [T, n] or None, status [n])."""
    _need_cuda()
    with _on(stream):
        T, n = vals.shape
        assert vals.stride(1) == 1
        ld = vals.stride(0) if T > 1 else n
        mk = lambda: torch.empty((T, ld), dtype=vals.dtype, device=vals.device)  # outputs share the input's leading dimension
        num, den = mk(), mk()
        cf = mk() if want_cf else None
        degs = torch.empty((2, ld), dtype=torch.int32, device=vals.device)
        status = torch.empty(n, dtype=torch.int32, device=vals.device)
        if workspace is None:
            workspace = alloc_workspace([0, 1], T)
        _check(lib().thiele_reconstruct_batch(points.data_ptr(), T, vals.data_ptr(), n, ld, p, num.data_ptr(), den.data_ptr(),
                                              degs.data_ptr(), _ptr(cf), status.data_ptr(), _ptr(workspace),
                                              workspace.numel(), _stream(stream)), "thiele_reconstruct_batch")
        return num[:, :n], den[:, :n], degs[:, :n], None if cf is None else cf[:, :n], status


def zippel_extend_skeleton(exps: torch.Tensor, offsets, coefs: torch.Tensor, p: int, cap: Optional[int] = None,
                           workspace: Optional[torch.Tensor] = None, stream=None):
    """(f1): coefs [B, T_tot] monomial in x_k -> (new_exps [cap, nv+1] int16, new_coefs [cap], new_offsets [F+1]
    int64 on the device, degs [F] int32).  The caller trims to new_offsets[-1] after a synchronisation."""
    _need_cuda()
    with _on(stream):
        o = _offs(offsets)
        F, (B, T_tot), nv = len(o) - 1, coefs.shape, exps.shape[1]
        cap = B * T_tot if cap is None else cap
        ne = torch.empty((max(cap, 1), nv + 1), dtype=torch.int16, device=coefs.device)
        nc = torch.empty(max(cap, 1), dtype=torch.int64, device=coefs.device)
        no = torch.empty(F + 1, dtype=torch.int64, device=coefs.device)
        degs = torch.empty(F, dtype=torch.int32, device=coefs.device)
        if workspace is None:
            workspace = alloc_workspace(o, B)
        _check(lib().zippel_extend_skeleton(_ptr(exps), o.ctypes.data, F, nv, _ptr(coefs), B, p, _ptr(ne), _ptr(nc), cap,
                                            _ptr(no), _ptr(degs), _ptr(workspace), workspace.numel(), _stream(stream)),
               "zippel_extend_skeleton")
        return ne, nc, no, degs


def zippel_static_scratch_bytes() -> int:
    return int(lib().zippel_static_scratch_bytes())


def zippel_extend_skeleton_static(exps: torch.Tensor, offsets, coefs: torch.Tensor, p: int, new_exps: torch.Tensor,
                                  new_coefs: torch.Tensor, new_offsets: torch.Tensor, degs: torch.Tensor, stream=None):
    """(f1) without a workspace and without any allocation (zippel.h: zippel_extend_skeleton_static): the caller passes
    the outputs -- new_exps [cap, nv+1] int16, new_coefs [cap] int64, new_offsets [F+1] int64, degs [F] int32, all on
    the device -- and cap = new_coefs.numel().  The scratch is ONE array per device inside the library: calls that
    overlap on the GPU race.  Raises ZippelError (code ZP_ERR_SCRATCH_LIMIT) beyond zippel_static_scratch_bytes()."""
    _need_cuda()
    with _on(stream):
        o = _offs(offsets)
        F, (B, T_tot), nv = len(o) - 1, coefs.shape, exps.shape[1]
        cap = int(new_coefs.numel())
        assert new_exps.dtype == torch.int16 and new_exps.is_contiguous() and tuple(new_exps.shape) == (cap, nv + 1)
        assert new_coefs.dtype == torch.int64 and new_offsets.dtype == torch.int64 and new_offsets.numel() == F + 1
        assert degs.dtype == torch.int32 and degs.numel() == F
        _check(lib().zippel_extend_skeleton_static(_ptr(exps), o.ctypes.data, F, nv, _ptr(coefs), B, p, _ptr(new_exps),
                                                   _ptr(new_coefs), cap, _ptr(new_offsets), _ptr(degs), _stream(stream)),
               "zippel_extend_skeleton_static")


ST_NO_RATIONAL = 21


def crt_rational_reconstruct_batch(r1: torch.Tensor, r2: torch.Tensor, p1: int, p2: int, stream=None):
    """(f4): images mod p1 and mod p2 [n] -> (num int64 [n] signed, den int64 [n] > 0, status int32 [n])."""
    _need_cuda()
    with _on(stream):
        n = r1.numel()
        num, den = torch.empty(n, dtype=torch.int64, device=r1.device), torch.empty(n, dtype=torch.int64, device=r1.device)
        status = torch.empty(n, dtype=torch.int32, device=r1.device)
        _check(lib().crt_rational_reconstruct_batch(r1.data_ptr(), r2.data_ptr(), n, p1, p2, num.data_ptr(), den.data_ptr(),
                                                    status.data_ptr(), _stream(stream)), "crt_rational_reconstruct_batch")
        return num, den, status
