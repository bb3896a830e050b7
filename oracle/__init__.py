"""ctypes loader for oracle/lsp_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares nothing with paper_2105_04006_b200/ (the CUDA path) and never imports it.

`build()` compiles the C file with gcc (-O2 -fopenmp, no -ffast-math: the oracle's arithmetic must be
IEEE) into oracle/liblsp_oracle.so; every call below is argument marshalling only -- the arithmetic
(Eq. 1-2) lives in the C file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lsp_oracle.c")
_SRC_GLS = os.path.join(_HERE, "gls_oracle.c")      # generalised LSP (floating mean + errors)
_LIB = os.path.join(_HERE, "liblsp_oracle.so")
_lib = None

_i64p = ctypes.POINTER(ctypes.c_int64)
_f64p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile oracle/lsp_oracle.c -> oracle/liblsp_oracle.so if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_GLS)):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, _SRC_GLS, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.lsp_oracle_grid.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int64, ctypes.c_int64, _i64p, _f64p]
        lib.lsp_oracle_grid.restype = None
        lib.lsp_oracle_periodogram.argtypes = [ctypes.c_int64, _i64p, _f64p, _f64p, ctypes.c_double, ctypes.c_double,
                                               ctypes.c_int64, ctypes.c_int64, _i64p, _f64p, ctypes.c_int, ctypes.c_int]
        lib.lsp_oracle_periodogram.restype = ctypes.c_int
        lib.lsp_oracle_best.argtypes = [ctypes.c_int64, _i64p, ctypes.c_int64, _f64p, ctypes.c_double, ctypes.c_double,
                                        _i64p, _f64p, _f64p]
        lib.lsp_oracle_best.restype = None
        lib.gls_oracle_periodogram.argtypes = [ctypes.c_int64, _i64p, _f64p, _f64p, _f64p, ctypes.c_double, ctypes.c_double,
                                               ctypes.c_int64, ctypes.c_int64, _i64p, _f64p, ctypes.c_int]
        lib.gls_oracle_periodogram.restype = ctypes.c_int
        _lib = lib
    return _lib


def _p(a, typ):
    return a.ctypes.data_as(typ) if a is not None else None


def grid(f_min: float, f_max: float, n_freq: int, k_list=None) -> np.ndarray:
    """f_k = f_min + k*(f_max - f_min)/n_freq, for all k or the listed ones."""
    lib = _load()
    kl = None if k_list is None else np.ascontiguousarray(k_list, dtype=np.int64)
    n_k = int(n_freq) if kl is None else int(kl.size)
    out = np.empty(n_k, dtype=np.float64)
    lib.lsp_oracle_grid(float(f_min), float(f_max), int(n_freq), n_k, _p(kl, _i64p), _p(out, _f64p))
    return out


def periodogram(offsets, t, y, f_min: float, f_max: float, n_freq: int, *, k_list=None,
                long_double: bool = False, n_threads: int = 0, return_threads: bool = False):
    """Eq. 2 of a CSR batch on the shared grid; power[n_obj, n_k] in FP64.

    t and y of any float dtype are widened to float64 (FP32 inputs are used as their exact values,
    DESIGN.md reading a11)."""
    lib = _load()
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    tt = np.ascontiguousarray(t, dtype=np.float64)
    yy = np.ascontiguousarray(y, dtype=np.float64)
    n_obj = int(off.size - 1)
    if n_obj < 0 or (n_obj >= 0 and off.size and (off[0] != 0 or int(off[-1]) != tt.size or tt.size != yy.size)):
        raise ValueError("bad CSR batch")
    kl = None if k_list is None else np.ascontiguousarray(k_list, dtype=np.int64)
    n_k = int(n_freq) if kl is None else int(kl.size)
    out = np.empty((n_obj, n_k), dtype=np.float64)
    used = lib.lsp_oracle_periodogram(n_obj, _p(off, _i64p), _p(tt, _f64p), _p(yy, _f64p), float(f_min), float(f_max),
                                      int(n_freq), n_k, _p(kl, _i64p), _p(out, _f64p), int(bool(long_double)),
                                      int(n_threads))
    if used < 0:
        raise ValueError("lsp_oracle_periodogram: bad argument")
    return (out, used) if return_threads else out


def best(offsets, power, f_min: float, f_max: float, n_freq: int):
    """(index, power, period) per object from a FULL periodogram: argmax, lowest index on ties, NaN never
    wins, period = 1/f_k* (readings a1, a7)."""
    lib = _load()
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    pw = np.ascontiguousarray(power, dtype=np.float64)
    n_obj = int(off.size - 1)
    if pw.shape != (n_obj, int(n_freq)):
        raise ValueError("power must be [n_obj, n_freq]")
    idx = np.empty(n_obj, dtype=np.int64)
    bp = np.empty(n_obj, dtype=np.float64)
    per = np.empty(n_obj, dtype=np.float64)
    lib.lsp_oracle_best(n_obj, _p(off, _i64p), int(n_freq), _p(pw, _f64p), float(f_min), float(f_max),
                        _p(idx, _i64p), _p(bp, _f64p), _p(per, _f64p))
    return idx, bp, per


def periodogram_generalized(offsets, t, y, sigma, f_min: float, f_max: float, n_freq: int, *, k_list=None, n_threads: int = 0):
    """Generalised LSP (floating mean, weights sigma^-2) of a CSR batch: P = (chi0^2 - chi^2(f)) / chi0^2 in [0, 1]
    (oracle/gls_oracle.c).  power[n_obj, n_k] in FP64."""
    lib = _load()
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    tt = np.ascontiguousarray(t, dtype=np.float64)
    yy = np.ascontiguousarray(y, dtype=np.float64)
    ss = np.ascontiguousarray(sigma, dtype=np.float64)
    n_obj = int(off.size - 1)
    if off[0] != 0 or int(off[-1]) != tt.size or tt.size != yy.size or tt.size != ss.size:
        raise ValueError("bad CSR batch")
    kl = None if k_list is None else np.ascontiguousarray(k_list, dtype=np.int64)
    n_k = int(n_freq) if kl is None else int(kl.size)
    out = np.empty((n_obj, n_k), dtype=np.float64)
    if lib.gls_oracle_periodogram(n_obj, _p(off, _i64p), _p(tt, _f64p), _p(yy, _f64p), _p(ss, _f64p), float(f_min), float(f_max),
                                  int(n_freq), n_k, _p(kl, _i64p), _p(out, _f64p), int(n_threads)) < 0:
        raise ValueError("gls_oracle_periodogram: bad argument")
    return out
