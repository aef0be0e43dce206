"""ctypes loader for oracle/gbk_cpu_fast.c: an OPTIMISED CPU restatement used for TIMING ONLY.

TEST / BENCH INFRASTRUCTURE, NOT PRODUCT CODE and NOT THE ORACLE: only tests/ and bench.py's
cpu_baseline leg may import this module; it never imports the product package.  Marshalling only.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gbk_cpu_fast.c")
_LIB = os.path.join(_HERE, "libgbk_cpu_fast.so")


def build(force: bool = False) -> str:
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O3", "-ffast-math", "-march=native", "-std=c11", "-fopenmp", "-fPIC",
                               "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nv", C.c_int32), ("u", C.c_int32),
                ("v_center", C.c_float), ("dv", C.c_float), ("rc_model", C.c_int32),
                ("r_p", C.c_int32), ("psf", C.POINTER(C.c_float)),
                ("r_v", C.c_int32), ("lsf", C.POINTER(C.c_float))]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        fp, u8p = C.POINTER(C.c_float), C.POINTER(C.c_uint8)
        L.gbkf_eval_rows.argtypes = [C.POINTER(_Grid), fp, fp, fp, fp, u8p, fp, C.c_int64, fp, C.c_int]
        L.gbkf_eval_rows.restype = C.c_int
        _lib = L
    return _lib


def _fp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_float))


def eval_rows(*, nx, ny, nv, u, v_center, dv, rc_model, psf_taps, lsf_taps, vobs, verr, sobs, serr, mask,
              params, nthreads: int = 0) -> np.ndarray:
    """chi2 [K] (float32).  psf_taps / lsf_taps: normalised 1-D Gaussian taps (odd lengths)."""
    c32 = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float32)
    psf, lsf = c32(psf_taps), c32(lsf_taps)
    vobs, verr, sobs, serr = c32(vobs), c32(verr), c32(sobs), c32(serr)
    mk = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    rows = np.ascontiguousarray(params, dtype=np.float32).reshape(-1, 10)
    out = np.empty(rows.shape[0], dtype=np.float32)
    g = _Grid(nx, ny, nv, u, v_center, dv, rc_model, psf.size // 2, _fp(psf), lsf.size // 2, _fp(lsf))
    rc = lib().gbkf_eval_rows(C.byref(g), _fp(vobs), _fp(verr), _fp(sobs), _fp(serr),
                              None if mk is None else mk.ctypes.data_as(C.POINTER(C.c_uint8)),
                              _fp(rows), rows.shape[0], _fp(out), int(nthreads))
    if rc != 0:
        raise MemoryError("allocation failed")
    return out
