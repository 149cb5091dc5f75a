"""ctypes loader of oracle/cpu_fast.c - the plain -O3 AVX2 CPU restatement timed as bench.py's `cpu_fast` line.

Timing context only (see the header of cpu_fast.c): not the parity oracle, pinned TO the oracle in
tests/test_oracle_cpu_fast.py.  May be imported by tests/ and bench.py only, never by the product package."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cpu_fast.c")
_LIB = os.path.join(_HERE, "libcpu_fast.so")
# x86-64-v3 (AVX2 + FMA), not -march=native: the .so travels from the build container to the GPU box
CFLAGS = ["-O3", "-mavx2", "-mfma", "-fopenmp", "-fPIC", "-shared", "-std=c11"]

_lib = None
_I64, _D, _P = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *CFLAGS, _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.cpu_fast_acc.argtypes = [_I64, _P, _P, _P, _I64, _P, _I64, _D, _D, _P]
        lib.cpu_fast_grad.argtypes = [_I64, _P, _P, _P, _P, _I64, _P, _I64, _D, _D, _P]
        _lib = lib
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _idx(a):
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data


def acc(pos, mass, G, eps, sink_idx=None, src_idx=None) -> np.ndarray:
    pos, mass = _f64(pos), _f64(mass)
    n = mass.shape[0]
    si, sp = _idx(sink_idx); sj, jp = _idx(src_idx)
    ns = n if si is None else si.shape[0]
    nj = n if sj is None else sj.shape[0]
    out = np.zeros((ns, 3))
    rc = _load().cpu_fast_acc(n, pos.ctypes.data, mass.ctypes.data, sp, ns, jp, nj, G, eps, out.ctypes.data)
    assert rc == 0
    return out


def grad(pos, mass, acc_in, G, eps, sink_idx=None, src_idx=None) -> np.ndarray:
    pos, mass, acc_in = _f64(pos), _f64(mass), _f64(acc_in)
    n = mass.shape[0]
    si, sp = _idx(sink_idx); sj, jp = _idx(src_idx)
    ns = n if si is None else si.shape[0]
    nj = n if sj is None else sj.shape[0]
    out = np.zeros((ns, 3))
    rc = _load().cpu_fast_grad(n, pos.ctypes.data, mass.ctypes.data, acc_in.ctypes.data, sp, ns, jp, nj, G, eps,
                               out.ctypes.data)
    assert rc == 0
    return out
