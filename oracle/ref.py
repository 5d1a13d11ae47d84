"""ctypes wrapper of the CPU ORACLE (oracle/zippel_ref.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It loads oracle/libzippel_ref.so (built from zippel_ref.c with gcc, on demand) and
exposes the ref_* functions on numpy arrays.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "zippel_ref.c")
_HDR = os.path.join(_HERE, "zippel_ref.h")
_SO = os.path.join(_HERE, "libzippel_ref.so")

ST_DUPLICATE_NODE, ST_DUPLICATE_SAMPLE, ST_ZERO_PIVOT = 16, 17, 18


def build(force: bool = False) -> str:
    """gcc -O2 the oracle into oracle/libzippel_ref.so (no tuning flags: it is timed as it stands)."""
    stale = (not os.path.exists(_SO)) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in (_SRC, _HDR))
    if force or stale:
        tmp = _SO + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-Wall", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _SO)
    return _SO


_lib = None
u64p = C.POINTER(C.c_uint64)
u16p = C.POINTER(C.c_uint16)
i64p = C.POINTER(C.c_int64)
i32p = C.POINTER(C.c_int32)


class _Part(C.Structure):
    _fields_ = [("exps", u16p), ("offsets", i64p), ("skel", u64p), ("uvals", u64p), ("out", u64p)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u64 = C.c_uint64
        for name in ("ref_mulmod", "ref_addmod", "ref_submod", "ref_powmod"):
            getattr(L, name).restype = u64
            getattr(L, name).argtypes = [u64, u64, u64]
        L.ref_invmod.restype = u64
        L.ref_invmod.argtypes = [u64, u64]
        L.ref_is_prime_u64.restype = C.c_int
        L.ref_is_prime_u64.argtypes = [u64]
        L.ref_largest_prime_below.restype = u64
        L.ref_largest_prime_below.argtypes = [u64]
        L.ref_zippel_eval_nodes.argtypes = [u16p, C.c_int64, C.c_int, u64p, u64, u64p]
        L.ref_master_poly.restype = None
        L.ref_master_poly.argtypes = [u64p, C.c_int64, u64, u64p]
        L.ref_node_quotient.restype = None
        L.ref_node_quotient.argtypes = [u64p, C.c_int64, u64, u64, u64p]
        L.ref_node_solve.restype = None
        L.ref_node_solve.argtypes = [u64p, u64p, C.c_int64, u64p, C.c_int64, C.c_int, u64, u64p, u64p]
        L.ref_node_solve_at.restype = None
        L.ref_node_solve_at.argtypes = [u64p, C.c_int64, u64p, C.c_int64, u64p, C.c_int64, C.c_int, u64, u64p, u64p]
        L.ref_vandermonde_solve_batch.argtypes = [u64p, i64p, C.c_int, u64p, C.c_int, C.c_int, u64, u64p, i32p]
        L.ref_gauss_solve.argtypes = [u64p, C.c_int64, u64p, C.c_int, u64, u64p]
        L.ref_newton_interp_batch.argtypes = [u64p, C.c_int, u64p, C.c_int64, C.c_int64, u64, C.c_int, u64p, i32p]
        L.ref_zippel_lift_step.argtypes = [u16p, i64p, C.c_int, C.c_int, u64p, u64p, C.c_int, C.c_int,
                                           u64p, u64, C.c_int, u64p, u64p, i32p]
        L.ref_power_sums.argtypes = [u64p, i64p, C.c_int, u64p, C.c_int, C.c_int, u64, u64p]
        L.ref_balanced_zippel_lift_step.argtypes = [C.POINTER(_Part), C.POINTER(_Part), C.c_int, C.c_int,
                                                    u64p, u64p, C.c_int, C.c_int, u64, C.c_int, i32p]
        L.ref_poly_rows_eval.argtypes = [u64p, C.c_int, u64p, C.c_int64, C.c_int64, u64, u64p]
        L.ref_thiele_reconstruct_batch.argtypes = [u64p, C.c_int, u64p, C.c_int64, C.c_int64, u64, u64p, u64p, i32p, u64p, i32p]
        L.ref_extend_skeleton.argtypes = [u16p, i64p, C.c_int, C.c_int, u64p, C.c_int, u64, u16p, u64p, C.c_int64, i64p, i32p]
        L.ref_crt_rational_batch.argtypes = [u64p, u64p, C.c_int64, u64, u64, i64p, i64p, i32p]
        L.ref_eval_sparse.restype = u64
        L.ref_eval_sparse.argtypes = [u16p, u64p, C.c_int64, C.c_int, u64p, u64]
        _lib = L
    return _lib


def _a(x, dt):
    return np.ascontiguousarray(x, dtype=dt)


def _p(a, t):
    return a.ctypes.data_as(t)


def _ok(rc, what):
    if rc != 0:
        raise ValueError(f"{what}: oracle returned error {rc}")


# ---- scalars ----
def mulmod(a, b, p): return int(lib().ref_mulmod(a, b, p))
def addmod(a, b, p): return int(lib().ref_addmod(a, b, p))
def submod(a, b, p): return int(lib().ref_submod(a, b, p))
def powmod(a, e, p): return int(lib().ref_powmod(a, e, p))
def invmod(a, p): return int(lib().ref_invmod(a, p))
def is_prime(n): return bool(lib().ref_is_prime_u64(n))
def largest_prime_below(n): return int(lib().ref_largest_prime_below(n))


# ---- arrays ----
def eval_nodes(exps, anchors, p):
    exps = _a(exps, np.uint16)
    T, nv = exps.shape
    anchors = _a(anchors, np.uint64)
    out = np.empty(T, dtype=np.uint64)
    _ok(lib().ref_zippel_eval_nodes(_p(exps, u16p), T, nv, _p(anchors, u64p), p, _p(out, u64p)), "eval_nodes")
    return out


def master_poly(m, p):
    m = _a(m, np.uint64)
    M = np.empty(len(m) + 1, dtype=np.uint64)
    lib().ref_master_poly(_p(m, u64p), len(m), p, _p(M, u64p))
    return M


def node_quotient(M, m_i, p):
    M = _a(M, np.uint64)
    t = len(M) - 1
    q = np.empty(t, dtype=np.uint64)
    lib().ref_node_quotient(_p(M, u64p), t, int(m_i), p, _p(q, u64p))
    return q


def node_solve(m, M, vals, p):
    """vals [B, t] -> (den [t], num [B, t])."""
    m, M, vals = _a(m, np.uint64), _a(M, np.uint64), _a(vals, np.uint64)
    B, t = vals.shape
    den = np.empty(t, dtype=np.uint64)
    num = np.empty((B, t), dtype=np.uint64)
    lib().ref_node_solve(_p(m, u64p), _p(M, u64p), t, _p(vals, u64p), t, B, p, _p(den, u64p), _p(num, u64p))
    return den, num


def node_solve_at(x, M, vals, p):
    """The per-node routine at the node values x [n]: vals [B, t] -> (den [n], num [B, n])."""
    x, M, vals = _a(x, np.uint64), _a(M, np.uint64), _a(vals, np.uint64)
    B, t = vals.shape
    assert len(M) == t + 1
    n = len(x)
    den = np.empty(n, dtype=np.uint64)
    num = np.empty((B, n), dtype=np.uint64)
    lib().ref_node_solve_at(_p(x, u64p), n, _p(M, u64p), t, _p(vals, u64p), t, B, p, _p(den, u64p), _p(num, u64p))
    return den, num


def vandermonde_solve_batch(nodes, offsets, vals, p, s0=0):
    nodes, offsets, vals = _a(nodes, np.uint64), _a(offsets, np.int64), _a(vals, np.uint64)
    F = len(offsets) - 1
    B = vals.shape[0]
    assert vals.shape[1] == offsets[-1]
    coefs = np.zeros_like(vals)
    status = np.zeros(F, dtype=np.int32)
    _ok(lib().ref_vandermonde_solve_batch(_p(nodes, u64p), _p(offsets, i64p), F, _p(vals, u64p), B, s0, p,
                                          _p(coefs, u64p), _p(status, i32p)), "vandermonde_solve_batch")
    return coefs, status


def gauss_solve(m, v, p, s0=0):
    m, v = _a(m, np.uint64), _a(v, np.uint64)
    c = np.empty(len(m), dtype=np.uint64)
    rc = lib().ref_gauss_solve(_p(m, u64p), len(m), _p(v, u64p), s0, p, _p(c, u64p))
    return (c if rc == 0 else None)


def newton_interp_batch(samples, vals, p, basis=0):
    samples, vals = _a(samples, np.uint64), _a(vals, np.uint64)
    B, n = vals.shape
    out = np.zeros_like(vals)
    status = np.zeros(1, dtype=np.int32)
    _ok(lib().ref_newton_interp_batch(_p(samples, u64p), B, _p(vals, u64p), n, n, p, basis, _p(out, u64p),
                                      _p(status, i32p)), "newton_interp_batch")
    return out, int(status[0])


def zippel_lift_step(exps, offsets, anchors, samples, vals, p, s0=0, basis=0):
    exps, offsets = _a(exps, np.uint16), _a(offsets, np.int64)
    anchors, samples, vals = _a(anchors, np.uint64), _a(samples, np.uint64), _a(vals, np.uint64)
    F, nv, B = len(offsets) - 1, exps.shape[1], len(samples)
    out = np.zeros_like(vals)
    nodes = np.empty(exps.shape[0], dtype=np.uint64)
    status = np.zeros(F, dtype=np.int32)
    _ok(lib().ref_zippel_lift_step(_p(exps, u16p), _p(offsets, i64p), F, nv, _p(anchors, u64p), _p(samples, u64p),
                                   B, s0, _p(vals, u64p), p, basis, _p(out, u64p), _p(nodes, u64p),
                                   _p(status, i32p)), "zippel_lift_step")
    return out, nodes, status


def power_sums(nodes, offsets, coef, p, s0=0):
    nodes, offsets, coef = _a(nodes, np.uint64), _a(offsets, np.int64), _a(coef, np.uint64)
    if coef.ndim == 1:
        coef = coef[None, :]
    out = np.zeros_like(coef)
    _ok(lib().ref_power_sums(_p(nodes, u64p), _p(offsets, i64p), len(offsets) - 1, _p(coef, u64p), coef.shape[0],
                             s0, p, _p(out, u64p)), "power_sums")
    return out


def balanced_zippel_lift_step(num, den, anchors, samples, p, s0=0, basis=0):
    """num, den: dicts with exps [T, nv], offsets [F+1], skel [T], uvals [B, T].
    Returns (out_num, out_den, status [2F])."""
    anchors, samples = _a(anchors, np.uint64), _a(samples, np.uint64)
    keep, parts, outs = [], [], []
    F = len(num["offsets"]) - 1
    nv = np.asarray(num["exps"]).shape[1]
    for d in (num, den):
        e, o = _a(d["exps"], np.uint16), _a(d["offsets"], np.int64)
        s, u = _a(d["skel"], np.uint64), _a(d["uvals"], np.uint64)
        out = np.zeros_like(u)
        keep += [e, o, s, u]
        outs.append(out)
        parts.append(_Part(_p(e, u16p), _p(o, i64p), _p(s, u64p), _p(u, u64p), _p(out, u64p)))
    status = np.zeros(2 * F, dtype=np.int32)
    _ok(lib().ref_balanced_zippel_lift_step(C.byref(parts[0]), C.byref(parts[1]), F, nv, _p(anchors, u64p),
                                            _p(samples, u64p), len(samples), s0, p, basis, _p(status, i32p)),
        "balanced_zippel_lift_step")
    return outs[0], outs[1], status


def poly_rows_eval(samples, P, p):
    samples, P = _a(samples, np.uint64), _a(P, np.uint64)
    B, n = P.shape
    out = np.zeros_like(P)
    _ok(lib().ref_poly_rows_eval(_p(samples, u64p), B, _p(P, u64p), n, n, p, _p(out, u64p)), "poly_rows_eval")
    return out


def eval_sparse(exps, coef, point, p):
    exps, coef, point = _a(exps, np.uint16), _a(coef, np.uint64), _a(point, np.uint64)
    return int(lib().ref_eval_sparse(_p(exps, u16p), _p(coef, u64p), exps.shape[0], exps.shape[1],
                                     _p(point, u64p), p))


def thiele_reconstruct_batch(points, vals, p):
    """(f2) eq. (2): vals [T, n] -> (num [T, n], den [T, n], degs [2, n], cf [T, n], status [n])."""
    points, vals = _a(points, np.uint64), _a(vals, np.uint64)
    T, n = vals.shape
    num, den, cf = np.zeros_like(vals), np.zeros_like(vals), np.zeros_like(vals)
    degs = np.zeros((2, n), dtype=np.int32)
    status = np.zeros(n, dtype=np.int32)
    _ok(lib().ref_thiele_reconstruct_batch(_p(points, u64p), T, _p(vals, u64p), n, n, p, _p(num, u64p), _p(den, u64p),
                                           _p(degs, i32p), _p(cf, u64p), _p(status, i32p)), "thiele_reconstruct_batch")
    return num, den, degs, cf, status


def extend_skeleton(exps, offsets, coefs, p, cap=None):
    """(f1): monomial coefficients [B, T_tot] -> (new_exps [T', nv+1], new_coefs [T'], new_offsets [F+1], degs [F])."""
    exps, offsets, coefs = _a(exps, np.uint16), _a(offsets, np.int64), _a(coefs, np.uint64)
    B, T_tot = coefs.shape
    F, nv = len(offsets) - 1, exps.shape[1]
    cap = B * T_tot if cap is None else cap
    ne = np.zeros((max(cap, 1), nv + 1), dtype=np.uint16)
    nc = np.zeros(max(cap, 1), dtype=np.uint64)
    no = np.zeros(F + 1, dtype=np.int64)
    degs = np.zeros(F, dtype=np.int32)
    _ok(lib().ref_extend_skeleton(_p(exps, u16p), _p(offsets, i64p), F, nv, _p(coefs, u64p), B, p, _p(ne, u16p),
                                  _p(nc, u64p), cap, _p(no, i64p), _p(degs, i32p)), "extend_skeleton")
    n = min(int(no[-1]), cap)
    return ne[:n], nc[:n], no, degs


def crt_rational_batch(r1, r2, p1, p2):
    """(f4): residues mod p1 and mod p2 -> (num int64 [n], den int64 [n], status [n])."""
    r1, r2 = _a(r1, np.uint64), _a(r2, np.uint64)
    n = len(r1)
    num, den = np.zeros(n, dtype=np.int64), np.zeros(n, dtype=np.int64)
    status = np.zeros(n, dtype=np.int32)
    _ok(lib().ref_crt_rational_batch(_p(r1, u64p), _p(r2, u64p), n, p1, p2, _p(num, i64p), _p(den, i64p),
                                     _p(status, i32p)), "crt_rational_batch")
    return num, den, status
