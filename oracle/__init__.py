"""CPU oracle for the FlexMoE routed-expert FFN hot path -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2606_27866_b200 (and vice versa).  The arithmetic
lives in oracle.c (plain C, fp64 by default); this file only compiles it with gcc and
marshals numpy arrays.  See oracle.c's header for citations, pins and what is unpinned.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "oracle.c")
_lib = None


def build(force: bool = False) -> str:
    """gcc-compile oracle.c twice (fp64 default + fp32 variant) into one shared object."""
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    o64 = os.path.join(_HERE, "oracle_f64.o")
    o32 = os.path.join(_HERE, "oracle_f32.o")
    base = ["gcc", "-O2", "-fopenmp", "-fPIC", "-std=c11", "-Wall", "-c", _SRC]
    subprocess.check_call(base + ["-DFXO_COMMON", "-DFXO_REAL=double", "-DFXO_SUF=f64", "-o", o64])
    subprocess.check_call(base + ["-DFXO_IS_FLOAT", "-DFXO_REAL=float", "-DFXO_SUF=f32", "-o", o32])
    subprocess.check_call(["gcc", "-shared", "-fopenmp", "-o", _SO, o64, o32, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.fxo_budget_rho.restype = ctypes.c_double
        _lib.fxo_ratio_to_width.restype = ctypes.c_int32
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct)) if a is not None else None


def _c(a, dt):
    a = np.ascontiguousarray(a, dtype=dt)
    return a


def pack(W_gate, W_up, W_down, channel_rank=None):
    """Eq. 3.  Inputs [E,I,d],[E,I,d],[E,d,I] bf16 bits, channel_rank [E,I] int32 or None."""
    Wg, Wu, Wd = _c(W_gate, np.uint16), _c(W_up, np.uint16), _c(W_down, np.uint16)
    E, I, d = Wg.shape
    assert Wu.shape == (E, I, d) and Wd.shape == (E, d, I)
    rk = _c(channel_rank, np.int32) if channel_rank is not None else None
    Gt, Ut, Dt = np.empty_like(Wg), np.empty_like(Wu), np.empty_like(Wd)
    lib().fxo_pack(E, I, d, _p(Wg, ctypes.c_uint16), _p(Wu, ctypes.c_uint16), _p(Wd, ctypes.c_uint16),
                   _p(rk, ctypes.c_int32), _p(Gt, ctypes.c_uint16), _p(Ut, ctypes.c_uint16),
                   _p(Dt, ctypes.c_uint16))
    return Gt, Ut, Dt


def route(topk_ids, E):
    ids = _c(topk_ids, np.int32)
    T, k = ids.shape
    counts = np.empty(E, np.int32)
    offsets = np.empty(E + 1, np.int32)
    perm = np.empty(T * k, np.int32)
    inv = np.empty(T * k, np.int32)
    rc = lib().fxo_route(_p(ids, ctypes.c_int32), T, k, E, _p(counts, ctypes.c_int32),
                         _p(offsets, ctypes.c_int32), _p(perm, ctypes.c_int32), _p(inv, ctypes.c_int32))
    if rc != 0:
        raise ValueError("expert id out of range")
    return counts, offsets, perm, inv


def moe_ffn(x, Gt, Ut, Dt, r, topk_ids, topk_w, rows=None, precision="f64"):
    """Eq. 4 summed over each token's k experts.  Returns y [n_rows, d] (float64 or float32)."""
    x = _c(x, np.uint16)
    Gt, Ut, Dt = _c(Gt, np.uint16), _c(Ut, np.uint16), _c(Dt, np.uint16)
    ids, w, r = _c(topk_ids, np.int32), _c(topk_w, np.float32), _c(r, np.int32)
    T, d = x.shape
    E, I, _ = Gt.shape
    k = ids.shape[1]
    assert r.shape == (E,) and (r >= 0).all() and (r <= I).all()
    assert ids.min(initial=0) >= 0 and ids.max(initial=0) < E
    if rows is not None:
        rows = _c(rows, np.int32)
        n_rows = rows.shape[0]
    else:
        n_rows = T
    if precision == "f64":
        y = np.empty((n_rows, d), np.float64)
        fn, ct = lib().fxo_moe_ffn_f64, ctypes.c_double
    else:
        y = np.empty((n_rows, d), np.float32)
        fn, ct = lib().fxo_moe_ffn_f32, ctypes.c_float
    fn(_p(x, ctypes.c_uint16), _p(Gt, ctypes.c_uint16), _p(Ut, ctypes.c_uint16), _p(Dt, ctypes.c_uint16),
       _p(r, ctypes.c_int32), _p(ids, ctypes.c_int32), _p(w, ctypes.c_float), T, k, E, d, I,
       _p(rows, ctypes.c_int32), n_rows, _p(y, ct))
    return y


def budget_rho(r, I):
    r = _c(np.asarray(r).ravel(), np.int32)
    return float(lib().fxo_budget_rho(_p(r, ctypes.c_int32), r.size, int(I)))


def ratio_to_width(I, num, den):
    return int(lib().fxo_ratio_to_width(int(I), int(num), int(den)))


def threads() -> int:
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
