"""ctypes loader for the CPU parity oracle (oracle/bifrost_oracle.cpp).

TEST INFRASTRUCTURE ONLY: may be imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs, never by the product package
paper_2210_02472_b200.  It shares no code with the CUDA path and does not
import it.  See the header of bifrost_oracle.cpp for what each routine computes,
the passages of /root/reference/PAPER.md it follows and how it is pinned.

oracle/integrator.py (plain numpy over these routines) is the oracle of the FSI / HHS-FSI integrator
(NEXT-4).

All routines take host numpy arrays (float64 / int32, C-contiguous) and return
new numpy arrays; per-sink outputs are compact (row k belongs to sink_idx[k]).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bifrost_oracle.cpp")
_LIB = os.path.join(_HERE, "libbifrost_oracle.so")

CXXFLAGS = ["-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared"]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (plain IEEE arithmetic: no contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", *CXXFLAGS, _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_D = ctypes.c_double
_I64 = ctypes.c_int64
_P = ctypes.c_void_p


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        common = [_I64, _P, _P, _P, _I64, _P, _I64, _D, _D, _P]
        for name in ("oracle_acc", "oracle_acc_ld"):
            getattr(lib, name).argtypes = common
        for name in ("oracle_grad", "oracle_grad_ld"):
            getattr(lib, name).argtypes = [_I64, _P, _P, _P, _P, _I64, _P, _I64, _D, _D, _P]
        lib.oracle_dtmin.argtypes = [_I64, _P, _P, _P, _P, _I64, _P, _I64, _D, _D, _D, _P, _P, _P, _P, _P, _P]
        for name in ("oracle_pn1", "oracle_pn1_ld"):
            getattr(lib, name).argtypes = [_I64, _P, _P, _P, _P, _I64, _D, _D, _P]
        for name in ("oracle_jerk", "oracle_jerk_ld"):
            getattr(lib, name).argtypes = [_I64, _P, _P, _P, _P, _I64, _P, _I64, _D, _D, _P]
        lib.oracle_phi.argtypes = common
        lib.oracle_criteria.argtypes = [_I64, _P, _P, _P, _P, _P, _I64, _D, _D, _D, _P, _P, _P, _P]
        for name in ("oracle_potential", "oracle_potential_ld"):
            getattr(lib, name).argtypes = [_I64, _P, _P, _D, _D]
            getattr(lib, name).restype = _D
        _lib = lib
    return _lib


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _idx(a: Optional[np.ndarray]):
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data


def n_threads() -> int:
    """Number of OpenMP threads the oracle will use (OMP_NUM_THREADS or all cores)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env.split(",")[0])
    return len(os.sched_getaffinity(0))


def acc(pos, mass, G, eps, sink_idx=None, src_idx=None, long_double=False) -> np.ndarray:
    pos, mass = _f64(pos), _f64(mass)
    n = mass.shape[0]
    si, sip = _idx(sink_idx)
    sj, sjp = _idx(src_idx)
    ns = n if si is None else si.shape[0]
    nj = n if sj is None else sj.shape[0]
    out = np.zeros((ns, 3))
    fn = _load().oracle_acc_ld if long_double else _load().oracle_acc
    fn(n, pos.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, eps, out.ctypes.data)
    return out


def grad(pos, mass, acc_in, G, eps, sink_idx=None, src_idx=None, long_double=False) -> np.ndarray:
    pos, mass, acc_in = _f64(pos), _f64(mass), _f64(acc_in)
    n = mass.shape[0]
    assert acc_in.shape == (n, 3)
    si, sip = _idx(sink_idx)
    sj, sjp = _idx(src_idx)
    ns = n if si is None else si.shape[0]
    nj = n if sj is None else sj.shape[0]
    out = np.zeros((ns, 3))
    fn = _load().oracle_grad_ld if long_double else _load().oracle_grad
    fn(n, pos.ctypes.data, mass.ctypes.data, acc_in.ctypes.data, sip, ns, sjp, nj, G, eps, out.ctypes.data)
    return out


def dtmin(pos, vel, mass, G, eta_ff, eta_fb, sink_idx=None, src_idx=None):
    """Returns dict(dt_ff, dt_fb, j_ff, j_fb, margin_ff, margin_fb)."""
    pos, vel, mass = _f64(pos), _f64(vel), _f64(mass)
    n = mass.shape[0]
    si, sip = _idx(sink_idx)
    sj, sjp = _idx(src_idx)
    ns = n if si is None else si.shape[0]
    nj = n if sj is None else sj.shape[0]
    dt_ff, dt_fb = np.zeros(ns), np.zeros(ns)
    m_ff, m_fb = np.zeros(ns), np.zeros(ns)
    j_ff, j_fb = np.zeros(ns, dtype=np.int32), np.zeros(ns, dtype=np.int32)
    _load().oracle_dtmin(n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, eta_ff, eta_fb,
                         dt_ff.ctypes.data, dt_fb.ctypes.data, j_ff.ctypes.data, j_fb.ctypes.data,
                         m_ff.ctypes.data, m_fb.ctypes.data)
    return dict(dt_ff=dt_ff, dt_fb=dt_fb, j_ff=j_ff, j_fb=j_fb, margin_ff=m_ff, margin_fb=m_fb)


def pn1(pos, vel, mass, bh_idx, G, c, long_double=False) -> np.ndarray:
    pos, vel, mass = _f64(pos), _f64(vel), _f64(mass)
    n = mass.shape[0]
    bh = np.ascontiguousarray(bh_idx, dtype=np.int32)
    out = np.zeros((n, 3))
    fn = _load().oracle_pn1_ld if long_double else _load().oracle_pn1
    fn(n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, bh.ctypes.data, bh.shape[0], G, c, out.ctypes.data)
    return out


def potential(pos, mass, G, eps=0.0, long_double=False) -> float:
    pos, mass = _f64(pos), _f64(mass)
    fn = _load().oracle_potential_ld if long_double else _load().oracle_potential
    return float(fn(mass.shape[0], pos.ctypes.data, mass.ctypes.data, G, eps))


def jerk(pos, vel, mass, G, eps, sink_idx=None, src_idx=None, long_double=False) -> np.ndarray:
    """Eq. 28, softened; compact rows of the sink list."""
    pos, vel, mass = _f64(pos), _f64(vel), _f64(mass)
    n = mass.shape[0]
    si, sip = _idx(sink_idx)
    sj, sjp = _idx(src_idx)
    ns = n if si is None else si.shape[0]
    nj = n if sj is None else sj.shape[0]
    out = np.zeros((ns, 3))
    fn = _load().oracle_jerk_ld if long_double else _load().oracle_jerk
    fn(n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, eps, out.ctypes.data)
    return out


def phi(pos, mass, G, eps, sink_idx=None, src_idx=None) -> np.ndarray:
    """Per-sink potential phi_i = -G sum_j m_j / s_ij (Eq. 4 / Eq. 68); compact rows."""
    pos, mass = _f64(pos), _f64(mass)
    n = mass.shape[0]
    si, sip = _idx(sink_idx)
    sj, sjp = _idx(src_idx)
    ns = n if si is None else si.shape[0]
    nj = n if sj is None else sj.shape[0]
    out = np.zeros(ns)
    _load().oracle_phi(n, pos.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, eps, out.ctypes.data)
    return out


def criteria(vel, acc_in, grad_c, jerk_in, eta, eta_grad, eta_jerk, sink_idx=None):
    """Eq. 24, 26, 27, 29: returns dict(dt_va, dt_gradv, dt_grada, dt_jerk), compact rows."""
    vel, acc_in, grad_c, jerk_in = _f64(vel), _f64(acc_in), _f64(grad_c), _f64(jerk_in)
    n = vel.shape[0]
    si, sip = _idx(sink_idx)
    ns = n if si is None else si.shape[0]
    outs = [np.zeros(ns) for _ in range(4)]
    _load().oracle_criteria(n, vel.ctypes.data, acc_in.ctypes.data, grad_c.ctypes.data, jerk_in.ctypes.data, sip, ns,
                            eta, eta_grad, eta_jerk, *[o.ctypes.data for o in outs])
    return dict(dt_va=outs[0], dt_gradv=outs[1], dt_grada=outs[2], dt_jerk=outs[3])


# ---- NEXT-2: subsystem-aware variants -------------------------

def _sub_arr(subsys, n):
    s = np.ascontiguousarray(subsys, dtype=np.int32)
    assert s.shape == (n,)
    return s


def _lists(n, sink_idx, src_idx):
    si, sip = _idx(sink_idx)
    sj, sjp = _idx(src_idx)
    return si, sip, (n if si is None else si.shape[0]), sj, sjp, (n if sj is None else sj.shape[0])


def _sub_sigs():
    lib = _load()
    if not getattr(lib, "_sub_ready", False):
        lists = [_P, _I64, _P, _I64]
        lib.oracle_acc_sub.argtypes = [_I64, _P, _P, *lists, _D, _D, _P, _P]
        lib.oracle_phi_sub.argtypes = [_I64, _P, _P, *lists, _D, _D, _P, _P]
        lib.oracle_grad_sub.argtypes = [_I64, _P, _P, _P, *lists, _D, _D, _P, _P]
        lib.oracle_jerk_sub.argtypes = [_I64, _P, _P, _P, *lists, _D, _D, _P, _P]
        lib.oracle_dtmin_sub.argtypes = [_I64, _P, _P, _P, *lists, _D, _D, _D, _P, _P, _P, _P, _P, _P, _P]
        lib.oracle_pn1_sub.argtypes = [_I64, _P, _P, _P, _P, _I64, _D, _D, _P, _P]
        lib.oracle_subsys_min.argtypes = [_I64, _P, _P, _P]
        lib._sub_ready = True
    return lib


def acc_sub(pos, mass, G, eps, subsys, sink_idx=None, src_idx=None) -> np.ndarray:
    """O-acc with pairs inside one subsystem dropped (Alg. 1)."""
    pos, mass = _f64(pos), _f64(mass)
    n = mass.shape[0]
    sub = _sub_arr(subsys, n)
    si, sip, ns, sj, sjp, nj = _lists(n, sink_idx, src_idx)
    out = np.zeros((ns, 3))
    _sub_sigs().oracle_acc_sub(n, pos.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, eps, sub.ctypes.data,
                               out.ctypes.data)
    return out


def phi_sub(pos, mass, G, eps, subsys, sink_idx=None, src_idx=None) -> np.ndarray:
    pos, mass = _f64(pos), _f64(mass)
    n = mass.shape[0]
    sub = _sub_arr(subsys, n)
    si, sip, ns, sj, sjp, nj = _lists(n, sink_idx, src_idx)
    out = np.zeros(ns)
    _sub_sigs().oracle_phi_sub(n, pos.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, eps, sub.ctypes.data,
                               out.ctypes.data)
    return out


def grad_sub(pos, mass, acc_in, G, eps, subsys, sink_idx=None, src_idx=None) -> np.ndarray:
    pos, mass, acc_in = _f64(pos), _f64(mass), _f64(acc_in)
    n = mass.shape[0]
    sub = _sub_arr(subsys, n)
    si, sip, ns, sj, sjp, nj = _lists(n, sink_idx, src_idx)
    out = np.zeros((ns, 3))
    _sub_sigs().oracle_grad_sub(n, pos.ctypes.data, mass.ctypes.data, acc_in.ctypes.data, sip, ns, sjp, nj, G, eps,
                                sub.ctypes.data, out.ctypes.data)
    return out


def jerk_sub(pos, vel, mass, G, eps, subsys, sink_idx=None, src_idx=None) -> np.ndarray:
    pos, vel, mass = _f64(pos), _f64(vel), _f64(mass)
    n = mass.shape[0]
    sub = _sub_arr(subsys, n)
    si, sip, ns, sj, sjp, nj = _lists(n, sink_idx, src_idx)
    out = np.zeros((ns, 3))
    _sub_sigs().oracle_jerk_sub(n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, eps,
                                sub.ctypes.data, out.ctypes.data)
    return out


def dtmin_sub(pos, vel, mass, G, eta_ff, eta_fb, subsys, sink_idx=None, src_idx=None):
    """O-dt with same-subsystem sources excluded (§3.5.2); dict like dtmin()."""
    pos, vel, mass = _f64(pos), _f64(vel), _f64(mass)
    n = mass.shape[0]
    sub = _sub_arr(subsys, n)
    si, sip, ns, sj, sjp, nj = _lists(n, sink_idx, src_idx)
    dt_ff, dt_fb, m_ff, m_fb = np.zeros(ns), np.zeros(ns), np.zeros(ns), np.zeros(ns)
    j_ff, j_fb = np.zeros(ns, dtype=np.int32), np.zeros(ns, dtype=np.int32)
    _sub_sigs().oracle_dtmin_sub(n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, eta_ff,
                                 eta_fb, sub.ctypes.data, dt_ff.ctypes.data, dt_fb.ctypes.data, j_ff.ctypes.data,
                                 j_fb.ctypes.data, m_ff.ctypes.data, m_fb.ctypes.data)
    return dict(dt_ff=dt_ff, dt_fb=dt_fb, j_ff=j_ff, j_fb=j_fb, margin_ff=m_ff, margin_fb=m_fb)


def pn1_sub(pos, vel, mass, bh_idx, G, c, subsys) -> np.ndarray:
    pos, vel, mass = _f64(pos), _f64(vel), _f64(mass)
    n = mass.shape[0]
    sub = _sub_arr(subsys, n)
    bh = np.ascontiguousarray(bh_idx, dtype=np.int32)
    out = np.zeros((n, 3))
    _sub_sigs().oracle_pn1_sub(n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, bh.ctypes.data, bh.shape[0], G, c,
                               sub.ctypes.data, out.ctypes.data)
    return out


def subsys_min(subsys, dt) -> np.ndarray:
    """Eq. 20: every member of a subsystem gets the minimum time-step of its members."""
    dt = _f64(dt)
    n = dt.shape[0]
    sub = _sub_arr(subsys, n)
    out = np.zeros(n)
    _sub_sigs().oracle_subsys_min(n, sub.ctypes.data, dt.ctypes.data, out.ctypes.data)
    return out


# ---- NEXT-3: neighbour search (§3.4, Eq. 18-19) and subsystem construction ------------

def ngb(pos, vel, mass, G, r_ngb, r_ngb_max, tau, C, cap=16, sink_idx=None, src_idx=None):
    """Returns (count[n_sink], list[n_sink][cap]) - neighbour ids in source-list order, -1 padded."""
    pos, vel, mass = _f64(pos), _f64(vel), _f64(mass)
    n = mass.shape[0]
    si, sip, ns, sj, sjp, nj = _lists(n, sink_idx, src_idx)
    lib = _load()
    lib.oracle_ngb.argtypes = [_I64, _P, _P, _P, _P, _I64, _P, _I64, _D, _D, _D, _D, _D, _I64, _P, _P]
    count = np.zeros(ns, dtype=np.int32)
    lst = np.full((ns, cap), -1, dtype=np.int32)
    lib.oracle_ngb(n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, sip, ns, sjp, nj, G, r_ngb, r_ngb_max, tau, C,
                   cap, count.ctypes.data, lst.ctypes.data)
    return count, lst


def components(n, edge_i, edge_j) -> np.ndarray:
    """Subsystem id (smallest member id) of every particle, -1 for particles without an edge."""
    ei = np.ascontiguousarray(edge_i, dtype=np.int32)
    ej = np.ascontiguousarray(edge_j, dtype=np.int32)
    lib = _load()
    lib.oracle_components.argtypes = [_I64, _P, _P, _I64, _P]
    out = np.zeros(n, dtype=np.int32)
    lib.oracle_components(n, ei.ctypes.data, ej.ctypes.data, ei.shape[0], out.ctypes.data)
    return out


def edges_from_lists(sinks, count, lst):
    """(edge_i, edge_j) arrays from per-sink neighbour lists (each listed pair once per direction)."""
    sinks = np.arange(count.shape[0], dtype=np.int32) if sinks is None else np.asarray(sinks, dtype=np.int32)
    ei, ej = [], []
    for k, i in enumerate(sinks):
        for q in range(min(int(count[k]), lst.shape[1])):
            ei.append(int(i)); ej.append(int(lst[k, q]))
    return np.asarray(ei, dtype=np.int32), np.asarray(ej, dtype=np.int32)
