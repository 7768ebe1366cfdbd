"""ctypes wrapper of the CPU oracle (oracle/lr_oracle.cpp).

TEST INFRASTRUCTURE: imported only by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / `--impl reference` legs.  Never imported by paper_2204_06633_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lr_oracle.cpp")
_LIB = os.path.join(_HERE, "liblr_oracle.so")
_lib = None

LD = np.longdouble
CH_XYZ, CH_AET, CH_XYZ_AET = 0, 1, 2


def build(force=False):
    """g++ -O2 -fopenmp; no hand vectorisation, no fast-math."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC]
    subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        i64, dbl, vp, ci = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p, ctypes.c_int
        L.orc_create.argtypes = [i64, dbl, dbl, vp, vp, dbl, dbl, ci, ctypes.POINTER(vp)]
        L.orc_destroy.argtypes = [vp]
        L.orc_destroy.restype = None
        L.orc_margins.argtypes = [vp, ci, ctypes.POINTER(i64), ctypes.POINTER(i64), ctypes.POINTER(i64)]
        L.orc_spline_eval_ld.argtypes = [vp, ci, vp, i64, vp]
        L.orc_lagrange_weights_ld.argtypes = [ci, vp, vp]
        L.orc_interp_ld.argtypes = [vp, i64, vp, ci, vp]
        for name in ("orc_project_ld", "orc_project_ldin", "orc_project_d"):
            getattr(L, name).argtypes = [vp, vp, vp, i64, dbl, dbl, dbl, i64, i64, vp]
        for name in ("orc_tdi_ld", "orc_tdi_ldin", "orc_tdi_d"):
            getattr(L, name).argtypes = [vp, vp, i64, ci, ci, ci, i64, i64, vp]
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def lagrange_weights(order, eps):
    w = np.zeros(order + 1, dtype=LD)
    e = np.array([eps], dtype=LD)
    lib().orc_lagrange_weights_ld(order, _ptr(e), _ptr(w))
    return w


def interp(x, n, D, order):
    x = _c(x, LD)
    out = np.zeros(1, dtype=LD)
    d = np.array([D], dtype=LD)
    lib().orc_interp_ld(_ptr(x), n, _ptr(d), order, _ptr(out))
    return out[0]


class Oracle:
    """One orbit table + (dt, t0, order).  Methods mirror lr_project / lr_tdi for one template."""

    def __init__(self, table, dt, t0, order):
        self._h = ctypes.c_void_p()
        x, ltt = _c(table.x, np.float64), _c(table.ltt, np.float64)
        rc = lib().orc_create(table.n_knots, table.t_start, table.knot_dt, _ptr(x), _ptr(ltt), dt, t0, order,
                              ctypes.byref(self._h))
        if rc != 0:
            raise ValueError(f"orc_create failed: {rc}")
        self.dt, self.t0, self.order = dt, t0, order

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def margins(self, tdi_gen):
        a, b, c = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        lib().orc_margins(self._h, tdi_gen, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c))
        return a.value, b.value, c.value

    def spline(self, channel, t):
        t = _c(np.atleast_1d(t), LD)
        out = np.zeros_like(t)
        lib().orc_spline_eval_ld(self._h, channel, _ptr(t), t.size, _ptr(out))
        return out

    def project(self, hp, hc, beta, lam, psi, lo=0, hi=None, precision="ld"):
        """y[6, n]; samples outside [lo, hi) are left 0.  precision: "ld" (truth) | "d" (timed baseline)."""
        n = len(hp)
        hi = n if hi is None else hi
        if precision == "d":
            hp, hc = _c(hp, np.float64), _c(hc, np.float64)
            y = np.zeros((6, n), dtype=np.float64)
            fn = lib().orc_project_d
        elif np.asarray(hp).dtype == LD:
            hp, hc = _c(hp, LD), _c(hc, LD)
            y = np.zeros((6, n), dtype=LD)
            fn = lib().orc_project_ldin
        else:
            hp, hc = _c(hp, np.float64), _c(hc, np.float64)
            y = np.zeros((6, n), dtype=LD)
            fn = lib().orc_project_ld
        rc = fn(self._h, _ptr(hp), _ptr(hc), n, beta, lam, psi, lo, hi, _ptr(y))
        if rc != 0:
            raise ValueError(f"oracle project failed: {rc}")
        return y

    def tdi(self, y, gen, nested=True, channels=CH_XYZ, lo=0, hi=None, precision="ld"):
        """out[3 or 6, n] from y[6, n]."""
        n = y.shape[-1]
        hi = n if hi is None else hi
        nout = 6 if channels == CH_XYZ_AET else 3
        if precision == "d":
            y = _c(y, np.float64)
            out = np.zeros((nout, n), dtype=np.float64)
            fn = lib().orc_tdi_d
        elif np.asarray(y).dtype == LD:
            y = _c(y, LD)
            out = np.zeros((nout, n), dtype=LD)
            fn = lib().orc_tdi_ldin
        else:
            y = _c(y, np.float64)
            out = np.zeros((nout, n), dtype=LD)
            fn = lib().orc_tdi_ld
        rc = fn(self._h, _ptr(y), n, gen, 1 if nested else 0, channels, lo, hi, _ptr(out))
        if rc != 0:
            raise ValueError(f"oracle tdi failed: {rc}")
        return out
