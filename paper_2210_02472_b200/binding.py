"""Thin Python binding of the C ABI in include/bifrost.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/bifrost.cu; this module only
checks dtypes/devices, passes `tensor.data_ptr()` and the current CUDA stream, and
allocates output tensors.  There is NO CPU fallback: if libbifrost.so is missing or
fails to load, or a call returns an error code, a BifrostError is raised.

    ctx = Context(max_n)                       # bifrost_create on the current device
    a   = ctx.acc(pos, mass, G, eps)           # torch.float64 CUDA tensors in, tensor out
    c   = ctx.grad(pos, mass, a, G, eps)
    dt  = ctx.dtmin(pos, vel, mass, G, eta_ff, eta_fb)   # (dt_ff, dt_fb, j_ff, j_fb)
    apn = ctx.pn1(pos, vel, mass, bh_idx, G, c)
Host-buffer calls (numpy in / numpy out through bifrost_*_host): ctx.acc_host(...), etc.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbifrost.so")

SYMBOLS = [
    "bifrost_create", "bifrost_destroy", "bifrost_strerror", "bifrost_last_cuda_error", "bifrost_launch_count",
    "bifrost_acc", "bifrost_grad", "bifrost_dtmin", "bifrost_pn1",
    "bifrost_jerk", "bifrost_potential", "bifrost_timestep_criteria",
    "bifrost_acc_host", "bifrost_grad_host", "bifrost_dtmin_host", "bifrost_pn1_host",
    "bifrost_fp64_probe", "bifrost_set_subsystems", "bifrost_subsys_min",
    "bifrost_neighbours", "bifrost_components", "bifrost_dtmin_neighbours",
    "bifrost_reserve", "bifrost_set_tuning", "bifrost_set_shard", "bifrost_acc_mutual", "bifrost_grad_mutual",
    "bifrost_acc_jerk", "bifrost_kick", "bifrost_drift", "bifrost_fsi_step", "bifrost_hhs_fsi", "bifrost_kinetic_energy",
    "bifrost_acc_static", "bifrost_static_error", "bifrost_set_level_criteria",
]


class BifrostError(RuntimeError):
    pass


_lib = None
_P, _I64, _D, _I = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int


def load_library() -> ctypes.CDLL:
    """dlopen libbifrost.so (built by paper_2210_02472_b200.build) and declare signatures."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise BifrostError(f"{LIB_PATH} not found: run `python -m paper_2210_02472_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    lib.bifrost_create.argtypes = [ctypes.POINTER(_P), _I, _I64]
    lib.bifrost_destroy.argtypes = [_P]
    lib.bifrost_strerror.argtypes = [_I]
    lib.bifrost_strerror.restype = ctypes.c_char_p
    lib.bifrost_last_cuda_error.argtypes = [_P]
    lib.bifrost_last_cuda_error.restype = ctypes.c_char_p
    lib.bifrost_launch_count.argtypes = [_P]
    lib.bifrost_launch_count.restype = _I64
    lists = [_P, _I64, _P, _I64]
    lib.bifrost_acc.argtypes = [_P, _I64, _P, _P, *lists, _D, _D, _P, _P]
    lib.bifrost_grad.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _P, _P]
    lib.bifrost_dtmin.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _D, _P, _P, _P, _P, _P]
    lib.bifrost_pn1.argtypes = [_P, _I64, _P, _P, _P, _P, _I64, _D, _D, _P, _P]
    lib.bifrost_jerk.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _P, _P]
    lib.bifrost_potential.argtypes = [_P, _I64, _P, _P, *lists, _D, _D, _P, _P, _P]
    lib.bifrost_timestep_criteria.argtypes = [_P, _I64, _P, _P, _P, _P, _P, _I64, _D, _D, _D, _P, _P, _P, _P, _P, _P]
    lib.bifrost_acc_host.argtypes = [_P, _I64, _P, _P, *lists, _D, _D, _P]
    lib.bifrost_grad_host.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _P]
    lib.bifrost_dtmin_host.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _D, _P, _P, _P, _P]
    lib.bifrost_pn1_host.argtypes = [_P, _I64, _P, _P, _P, _P, _I64, _D, _D, _P]
    lib.bifrost_reserve.argtypes = [_P, _I]
    lib.bifrost_set_tuning.argtypes = [_P, _I, _I64]
    lib.bifrost_set_shard.argtypes = [_P, _I, _I]
    lib.bifrost_set_level_criteria.argtypes = [_P, _D, _D, _D]
    lib.bifrost_acc_mutual.argtypes = [_P, _I64, _P, _P, *lists, _D, _D, _P, _P]
    lib.bifrost_grad_mutual.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _P, _P]
    lib.bifrost_set_subsystems.argtypes = [_P, _P, _I64]
    lib.bifrost_subsys_min.argtypes = [_P, _I64, _P, _P, _P]
    lib.bifrost_neighbours.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _D, _D, _D, _I64, _P, _P, _P]
    lib.bifrost_components.argtypes = [_P, _I64, _P, _P, _I64, _P, _P]
    lib.bifrost_dtmin_neighbours.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _D, _D, _D, _D, _D, _I64,
                                             _P, _P, _P, _P, _P, _P, _P]
    lib.bifrost_acc_jerk.argtypes = [_P, _I64, _P, _P, _P, *lists, _D, _D, _P, _P, _P]
    lib.bifrost_kick.argtypes = [_P, _I64, _P, _I64, _P, _P, _D, _D, _P, _P]
    lib.bifrost_drift.argtypes = [_P, _I64, _P, _I64, _P, _D, _P, _P]
    lib.bifrost_fsi_step.argtypes = [_P, _I64, _P, _P, _P, _P, _I64, _D, _D, _D, _P]
    lib.bifrost_hhs_fsi.argtypes = [_P, _I64, _P, _P, _P, _D, _D, _D, _D, _P, _D, _I, _P, _I64, _P, _P]
    lib.bifrost_kinetic_energy.argtypes = [_P, _I64, _P, _P, _P, _I64, _P, _P]
    lib.bifrost_fp64_probe.argtypes = [_P, _I, _I64, _I, ctypes.POINTER(_D), ctypes.POINTER(_D)]
    lib.bifrost_acc_static.argtypes = [_I, _I64, _P, _P, _D, _D, _P, _P]
    lib.bifrost_static_error.argtypes = []
    lib.bifrost_static_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


# Tensors marshalled for the call being prepared: Context._stream(), evaluated as the last argument of every C call,
# checks them together (same device as the context, equal row counts, index values in debug mode) and clears the list.
_seen = []
DEBUG_INDEX_CHECK = False      # True: every index list is range-checked against n (one device -> host sync per list)


def _dev_f64(t, shape_tail, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise BifrostError(f"{name}: expected a contiguous float64 CUDA tensor")
    if t.dim() < 1 or tuple(t.shape[1:]) != shape_tail:
        raise BifrostError(f"{name}: bad shape {tuple(t.shape)}")
    _seen.append(("rows", name, t))
    return t


def _dev_i32_rows(t, shape_tail, name):
    """An int32 per-particle array ([n] or [n, cap]): counted with the float64 arrays for the row check."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()):
        raise BifrostError(f"{name}: expected a contiguous int32 CUDA tensor")
    if t.dim() < 1 or tuple(t.shape[1:]) != shape_tail:
        raise BifrostError(f"{name}: bad shape {tuple(t.shape)}")
    _seen.append(("rows", name, t))
    return t


def _dev_idx(t, name):
    import torch
    if t is None:
        return None, 0
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.int32 and t.is_contiguous() and t.dim() == 1):
        raise BifrostError(f"{name}: expected a contiguous 1-D int32 CUDA tensor")
    _seen.append(("index", name, t))
    # an empty list is not NULL ("all particles"): hand the library a valid dummy address
    return t, (t.data_ptr() if t.numel() else _dummy_ptr(t.device))


_dummies = {}
_HOST_DUMMY = np.zeros(1, dtype=np.int32)


def _dummy_ptr(device) -> int:
    import torch
    if device not in _dummies:
        _dummies[device] = torch.zeros(1, dtype=torch.int32, device=device)
    return _dummies[device].data_ptr()


def _host_f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _host_idx(a):
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, (a.ctypes.data if a.size else _HOST_DUMMY.ctypes.data)


STATIC_MAX_N = 16384           # BIFROST_STATIC_MAX_N


def acc_static(pos, mass, G, eps, out):
    """bifrost_acc_static: Eq. 6 over all particles with NO context and no allocation anywhere - the scratch is a
    static device array inside libbifrost.so (n <= STATIC_MAX_N; calls that overlap on one GPU race on it).  `out` is
    the caller's [n, 3] tensor (this function allocates nothing either); returns it."""
    import torch
    lib = load_library()
    _seen.clear()
    pos = _dev_f64(pos, (3,), "pos"); mass = _dev_f64(mass, (), "mass"); out = _dev_f64(out, (3,), "out")
    _seen.clear()
    n = mass.shape[0]
    if pos.shape[0] != n or out.shape[0] != n:
        raise BifrostError(f"acc_static: pos has {pos.shape[0]} rows, out {out.shape[0]}, mass {n}")
    if pos.device != mass.device or out.device != mass.device:
        raise BifrostError("acc_static: pos, mass and out must be on one device")
    dev = mass.device.index
    rc = lib.bifrost_acc_static(dev, n, pos.data_ptr(), mass.data_ptr(), float(G), float(eps), out.data_ptr(),
                                torch.cuda.current_stream(dev).cuda_stream)
    if rc != 0:
        raise BifrostError(f"bifrost_acc_static: {lib.bifrost_strerror(rc).decode()} [{lib.bifrost_static_error().decode()}]")
    return out


class Context:
    """Owns one bifrost_ctx (device scratch for up to max_n particles) on `device`."""

    def __init__(self, max_n: int, device: Optional[int] = None):
        import torch
        self._lib = load_library()
        if not torch.cuda.is_available():
            raise BifrostError("no CUDA device: the BIFROST path has no CPU fallback")
        self.device = torch.cuda.current_device() if device is None else int(device)
        self.max_n = int(max_n)
        h = _P()
        rc = self._lib.bifrost_create(ctypes.byref(h), self.device, self.max_n)
        if rc != 0:
            raise BifrostError(f"bifrost_create: {self._lib.bifrost_strerror(rc).decode()}")
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._lib.bifrost_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        _seen.clear()
        if rc != 0:
            msg = self._lib.bifrost_strerror(rc).decode()
            cu = self._lib.bifrost_last_cuda_error(self._h).decode()
            raise BifrostError(f"{what}: {msg}" + (f" [{cu}]" if cu else ""))

    RESERVE_HOST, RESERVE_INTEGRATOR = 1, 2
    TUNE_FUSED_MAX_SINKS, TUNE_SMALL_M, TUNE_SYM_MIN_N, TUNE_MUTUAL_MIN_PAIRS, TUNE_FEW_MAX_SINKS, TUNE_FEW_MAX_PAIRS, TUNE_FUSED_CLUSTER = 0, 1, 2, 3, 4, 5, 6

    def reserve(self, what: int):
        self._check(self._lib.bifrost_reserve(self._h, int(what)), "bifrost_reserve")

    def set_shard(self, rank: int, world: int):
        """Shard the pair work of same-list acc / grad calls over `world` ranks: outputs become partial sums that
        the caller all-reduces (sharding.allreduce_sum)."""
        self._check(self._lib.bifrost_set_shard(self._h, int(rank), int(world)), "bifrost_set_shard")

    def set_tuning(self, knob: int, value: int):
        self._check(self._lib.bifrost_set_tuning(self._h, int(knob), int(value)), "bifrost_set_tuning")

    @property
    def launch_count(self) -> int:
        return int(self._lib.bifrost_launch_count(self._h))

    def _stream(self):
        """The context's device's current stream; also the one place where the tensors marshalled for this call are
        checked together: all on the context's device, all per-particle arrays with the same number of rows, index
        values inside [0, n) when DEBUG_INDEX_CHECK is set.  A mismatch raises BifrostError instead of becoming an
        out-of-bounds device access."""
        import torch
        seen, n_rows = list(_seen), None
        _seen.clear()
        for kind, name, t in seen:
            if t.device.index != self.device:
                raise BifrostError(f"{name}: tensor on {t.device}, context on cuda:{self.device}")
            if kind == "rows":
                if n_rows is None:
                    n_rows = (t.shape[0], name)
                elif t.shape[0] != n_rows[0]:
                    raise BifrostError(f"{name}: {t.shape[0]} rows, but {n_rows[1]} has {n_rows[0]}")
        if DEBUG_INDEX_CHECK and n_rows is not None:
            for kind, name, t in seen:
                if kind == "index" and t.numel() and (int(t.min()) < 0 or int(t.max()) >= n_rows[0]):
                    raise BifrostError(f"{name}: ids outside [0, {n_rows[0]})")
        return torch.cuda.current_stream(self.device).cuda_stream

    # ---- device-pointer entry points -------------------------------------------------
    def acc(self, pos, mass, G, eps, sink_idx=None, src_idx=None, out=None):
        import torch
        pos = _dev_f64(pos, (3,), "pos"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx"); sj, sjp = _dev_idx(src_idx, "src_idx")
        if out is None:
            out = torch.zeros((n, 3), dtype=torch.float64, device=pos.device)
        _dev_f64(out, (3,), "out")
        rc = self._lib.bifrost_acc(self._h, n, pos.data_ptr(), mass.data_ptr(), sip or None,
                                   n if si is None else si.shape[0], sjp or None, n if sj is None else sj.shape[0],
                                   float(G), float(eps), out.data_ptr(), self._stream())
        self._check(rc, "bifrost_acc")
        return out

    def grad(self, pos, mass, acc, G, eps, sink_idx=None, src_idx=None, out=None):
        import torch
        pos = _dev_f64(pos, (3,), "pos"); mass = _dev_f64(mass, (), "mass"); acc = _dev_f64(acc, (3,), "acc")
        n = mass.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx"); sj, sjp = _dev_idx(src_idx, "src_idx")
        if out is None:
            out = torch.zeros((n, 3), dtype=torch.float64, device=pos.device)
        _dev_f64(out, (3,), "out")
        rc = self._lib.bifrost_grad(self._h, n, pos.data_ptr(), mass.data_ptr(), acc.data_ptr(), sip or None,
                                    n if si is None else si.shape[0], sjp or None, n if sj is None else sj.shape[0],
                                    float(G), float(eps), out.data_ptr(), self._stream())
        self._check(rc, "bifrost_grad")
        return out

    def acc_mutual(self, pos, mass, G, eps, a_idx, b_idx, out=None):
        """Eq. 12 for both sets of a level: out[a] = acc of a over sources B, out[b] = acc of b over sources A."""
        import torch
        pos = _dev_f64(pos, (3,), "pos"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        ia, iap = _dev_idx(a_idx, "a_idx"); ib, ibp = _dev_idx(b_idx, "b_idx")
        if ia is None or ib is None:
            raise BifrostError("acc_mutual: both lists are required")
        if out is None:
            out = torch.zeros((n, 3), dtype=torch.float64, device=pos.device)
        _dev_f64(out, (3,), "out")
        rc = self._lib.bifrost_acc_mutual(self._h, n, pos.data_ptr(), mass.data_ptr(), iap, ia.shape[0], ibp, ib.shape[0],
                                          float(G), float(eps), out.data_ptr(), self._stream())
        self._check(rc, "bifrost_acc_mutual")
        return out

    def grad_mutual(self, pos, mass, acc, G, eps, a_idx, b_idx, out=None):
        """Eq. 13 for both sets of a level (see acc_mutual)."""
        import torch
        pos = _dev_f64(pos, (3,), "pos"); mass = _dev_f64(mass, (), "mass"); acc = _dev_f64(acc, (3,), "acc")
        n = mass.shape[0]
        ia, iap = _dev_idx(a_idx, "a_idx"); ib, ibp = _dev_idx(b_idx, "b_idx")
        if ia is None or ib is None:
            raise BifrostError("grad_mutual: both lists are required")
        if out is None:
            out = torch.zeros((n, 3), dtype=torch.float64, device=pos.device)
        _dev_f64(out, (3,), "out")
        rc = self._lib.bifrost_grad_mutual(self._h, n, pos.data_ptr(), mass.data_ptr(), acc.data_ptr(), iap, ia.shape[0],
                                           ibp, ib.shape[0], float(G), float(eps), out.data_ptr(), self._stream())
        self._check(rc, "bifrost_grad_mutual")
        return out

    def dtmin(self, pos, vel, mass, G, eta_ff, eta_fb, sink_idx=None, src_idx=None, out=None):
        """Returns (dt_ff, dt_fb, j_ff, j_fb), each of length n, written at sink ids
        (rows of inactive particles keep their initial value: +inf / -1)."""
        import torch
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx"); sj, sjp = _dev_idx(src_idx, "src_idx")
        if out is None:
            out = (torch.full((n,), float("inf"), dtype=torch.float64, device=pos.device),
                   torch.full((n,), float("inf"), dtype=torch.float64, device=pos.device),
                   torch.full((n,), -1, dtype=torch.int32, device=pos.device),
                   torch.full((n,), -1, dtype=torch.int32, device=pos.device))
        _dev_f64(out[0], (), "out dt_ff"); _dev_f64(out[1], (), "out dt_fb")
        _dev_i32_rows(out[2], (), "out j_ff"); _dev_i32_rows(out[3], (), "out j_fb")
        rc = self._lib.bifrost_dtmin(self._h, n, pos.data_ptr(), vel.data_ptr(), mass.data_ptr(), sip or None,
                                     n if si is None else si.shape[0], sjp or None, n if sj is None else sj.shape[0],
                                     float(G), float(eta_ff), float(eta_fb),
                                     out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), out[3].data_ptr(),
                                     self._stream())
        self._check(rc, "bifrost_dtmin")
        return out

    def pn1(self, pos, vel, mass, bh_idx, G, c, out=None):
        import torch
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        bh, bhp = _dev_idx(bh_idx, "bh_idx")
        if out is None:
            out = torch.empty((n, 3), dtype=torch.float64, device=pos.device)
        rc = self._lib.bifrost_pn1(self._h, n, pos.data_ptr(), vel.data_ptr(), mass.data_ptr(), bhp or None,
                                   0 if bh is None else bh.shape[0], float(G), float(c), out.data_ptr(), self._stream())
        self._check(rc, "bifrost_pn1")
        return out

    # ---- NEXT rows ------------------------------------------------------------------
    def jerk(self, pos, vel, mass, G, eps, sink_idx=None, src_idx=None, out=None):
        import torch
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx"); sj, sjp = _dev_idx(src_idx, "src_idx")
        if out is None:
            out = torch.zeros((n, 3), dtype=torch.float64, device=pos.device)
        _dev_f64(out, (3,), "out")
        rc = self._lib.bifrost_jerk(self._h, n, pos.data_ptr(), vel.data_ptr(), mass.data_ptr(), sip or None,
                                    n if si is None else si.shape[0], sjp or None, n if sj is None else sj.shape[0],
                                    float(G), float(eps), out.data_ptr(), self._stream())
        self._check(rc, "bifrost_jerk")
        return out

    def potential(self, pos, mass, G, eps, sink_idx=None, src_idx=None, want_phi=True, want_W=True):
        """Returns (phi [n] or None, W 0-dim device tensor or None)."""
        import torch
        pos = _dev_f64(pos, (3,), "pos"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx"); sj, sjp = _dev_idx(src_idx, "src_idx")
        phi = torch.zeros(n, dtype=torch.float64, device=pos.device) if want_phi else None
        W = torch.zeros((), dtype=torch.float64, device=pos.device) if want_W else None
        rc = self._lib.bifrost_potential(self._h, n, pos.data_ptr(), mass.data_ptr(), sip or None,
                                         n if si is None else si.shape[0], sjp or None, n if sj is None else sj.shape[0],
                                         float(G), float(eps), phi.data_ptr() if want_phi else None,
                                         W.data_ptr() if want_W else None, self._stream())
        self._check(rc, "bifrost_potential")
        return phi, W

    def timestep_criteria(self, vel, acc, grad, jerk, eta, eta_grad, eta_jerk, sink_idx=None, inout_dt=None):
        """Returns dict(dt_va, dt_gradv, dt_grada, dt_jerk) of [n] tensors (+inf at non-sinks; gradv/grada/jerk
        entries are None when grad / jerk is None).  inout_dt, if given, is min-updated in place."""
        import torch
        vel = _dev_f64(vel, (3,), "vel"); acc = _dev_f64(acc, (3,), "acc")
        if grad is not None:
            grad = _dev_f64(grad, (3,), "grad")
        if jerk is not None:
            jerk = _dev_f64(jerk, (3,), "jerk")
        n = vel.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx")

        def new():
            return torch.full((n,), float("inf"), dtype=torch.float64, device=vel.device)
        o = dict(dt_va=new(), dt_gradv=new() if grad is not None else None,
                 dt_grada=new() if grad is not None else None, dt_jerk=new() if jerk is not None else None)
        ptr = lambda t: None if t is None else t.data_ptr()
        rc = self._lib.bifrost_timestep_criteria(self._h, n, vel.data_ptr(), acc.data_ptr(), ptr(grad), ptr(jerk),
                                                 sip or None, n if si is None else si.shape[0], float(eta),
                                                 float(eta_grad), float(eta_jerk), ptr(o["dt_va"]), ptr(o["dt_gradv"]),
                                                 ptr(o["dt_grada"]), ptr(o["dt_jerk"]), ptr(inout_dt), self._stream())
        self._check(rc, "bifrost_timestep_criteria")
        return o

    # ---- host-buffer entry points (numpy in, numpy out; synchronous) -----------------
    def acc_host(self, pos, mass, G, eps, sink_idx=None, src_idx=None, out=None):
        pos, mass = _host_f64(pos), _host_f64(mass)
        n = mass.shape[0]
        si, sip = _host_idx(sink_idx); sj, sjp = _host_idx(src_idx)
        if out is None:
            out = np.zeros((n, 3))
        rc = self._lib.bifrost_acc_host(self._h, n, pos.ctypes.data, mass.ctypes.data, sip,
                                        n if si is None else si.shape[0], sjp, n if sj is None else sj.shape[0],
                                        float(G), float(eps), out.ctypes.data)
        self._check(rc, "bifrost_acc_host")
        return out

    def grad_host(self, pos, mass, acc, G, eps, sink_idx=None, src_idx=None, out=None):
        pos, mass, acc = _host_f64(pos), _host_f64(mass), _host_f64(acc)
        n = mass.shape[0]
        si, sip = _host_idx(sink_idx); sj, sjp = _host_idx(src_idx)
        if out is None:
            out = np.zeros((n, 3))
        rc = self._lib.bifrost_grad_host(self._h, n, pos.ctypes.data, mass.ctypes.data, acc.ctypes.data, sip,
                                         n if si is None else si.shape[0], sjp, n if sj is None else sj.shape[0],
                                         float(G), float(eps), out.ctypes.data)
        self._check(rc, "bifrost_grad_host")
        return out

    def dtmin_host(self, pos, vel, mass, G, eta_ff, eta_fb, sink_idx=None, src_idx=None):
        pos, vel, mass = _host_f64(pos), _host_f64(vel), _host_f64(mass)
        n = mass.shape[0]
        si, sip = _host_idx(sink_idx); sj, sjp = _host_idx(src_idx)
        dt_ff, dt_fb = np.full(n, np.inf), np.full(n, np.inf)
        j_ff, j_fb = np.full(n, -1, np.int32), np.full(n, -1, np.int32)
        rc = self._lib.bifrost_dtmin_host(self._h, n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, sip,
                                          n if si is None else si.shape[0], sjp, n if sj is None else sj.shape[0],
                                          float(G), float(eta_ff), float(eta_fb), dt_ff.ctypes.data, dt_fb.ctypes.data,
                                          j_ff.ctypes.data, j_fb.ctypes.data)
        self._check(rc, "bifrost_dtmin_host")
        return dt_ff, dt_fb, j_ff, j_fb

    def pn1_host(self, pos, vel, mass, bh_idx, G, c):
        pos, vel, mass = _host_f64(pos), _host_f64(vel), _host_f64(mass)
        n = mass.shape[0]
        bh, bhp = _host_idx(bh_idx)
        out = np.empty((n, 3))
        rc = self._lib.bifrost_pn1_host(self._h, n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, bhp,
                                        0 if bh is None else bh.shape[0], float(G), float(c), out.ctypes.data)
        self._check(rc, "bifrost_pn1_host")
        return out

    # ---- measurement aid --------------------------------------------------------------
    def fp64_probe(self, mix: int = 0, iters: int = 1 << 16, ctas_per_sm: int = 16):
        """Measured FP64-pipe rate of a register-only kernel: (ms, lane_instructions_per_s)."""
        ms, cnt = _D(0.0), _D(0.0)
        rc = self._lib.bifrost_fp64_probe(self._h, int(mix), int(iters), int(ctas_per_sm), ctypes.byref(ms),
                                          ctypes.byref(cnt))
        self._check(rc, "bifrost_fp64_probe")
        return ms.value, cnt.value / (ms.value * 1e-3)

    # ---- NEXT-2 ----------------------------------------------------------------------
    def set_subsystems(self, subsys):
        """subsys: int32 CUDA tensor [n] (-1 = single) or None.  The tensor is kept alive here."""
        if subsys is None:
            self._subsys = None
            self._check(self._lib.bifrost_set_subsystems(self._h, None, 0), "bifrost_set_subsystems")
            return
        _dev_i32_rows(subsys, (), "subsys")
        self._subsys = subsys
        self._check(self._lib.bifrost_set_subsystems(self._h, subsys.data_ptr(), subsys.shape[0]),
                    "bifrost_set_subsystems")

    def subsys_min(self, subsys, inout_dt):
        _dev_i32_rows(subsys, (), "subsys")
        _dev_f64(inout_dt, (), "inout_dt")
        rc = self._lib.bifrost_subsys_min(self._h, subsys.shape[0], subsys.data_ptr(), inout_dt.data_ptr(), self._stream())
        self._check(rc, "bifrost_subsys_min")
        return inout_dt

    # ---- NEXT-3 ----------------------------------------------------------------------
    def neighbours(self, pos, vel, mass, G, r_ngb, r_ngb_max, tau, C, cap=16, sink_idx=None, src_idx=None, out=None):
        """Returns (count [n] int32, list [n, cap] int32) written at sink rows; other rows keep
        count = 0 / list = -1 (the initial values of freshly allocated outputs)."""
        import torch
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx"); sj, sjp = _dev_idx(src_idx, "src_idx")
        if out is None:
            out = (torch.zeros((n,), dtype=torch.int32, device=pos.device),
                   torch.full((n, int(cap)), -1, dtype=torch.int32, device=pos.device))
        _dev_i32_rows(out[0], (), "out count"); _dev_i32_rows(out[1], (int(cap),), "out list")
        rc = self._lib.bifrost_neighbours(self._h, n, pos.data_ptr(), vel.data_ptr(), mass.data_ptr(), sip or None,
                                          n if si is None else si.shape[0], sjp or None, n if sj is None else sj.shape[0],
                                          float(G), float(r_ngb), float(r_ngb_max), float(tau), float(C), int(cap),
                                          out[0].data_ptr(), out[1].data_ptr(), self._stream())
        self._check(rc, "bifrost_neighbours")
        return out

    def dtmin_neighbours(self, pos, vel, mass, G, eta_ff, eta_fb, r_ngb, r_ngb_max, tau, C, cap=16, sink_idx=None,
                         src_idx=None):
        """bifrost_dtmin and bifrost_neighbours in one pass: returns ((dt_ff, dt_fb, j_ff, j_fb), (count, list))."""
        import torch
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx"); sj, sjp = _dev_idx(src_idx, "src_idx")
        d = (torch.full((n,), float("inf"), dtype=torch.float64, device=pos.device),
             torch.full((n,), float("inf"), dtype=torch.float64, device=pos.device),
             torch.full((n,), -1, dtype=torch.int32, device=pos.device),
             torch.full((n,), -1, dtype=torch.int32, device=pos.device))
        g = (torch.zeros((n,), dtype=torch.int32, device=pos.device),
             torch.full((n, int(cap)), -1, dtype=torch.int32, device=pos.device))
        rc = self._lib.bifrost_dtmin_neighbours(
            self._h, n, pos.data_ptr(), vel.data_ptr(), mass.data_ptr(), sip or None, n if si is None else si.shape[0],
            sjp or None, n if sj is None else sj.shape[0], float(G), float(eta_ff), float(eta_fb), float(r_ngb),
            float(r_ngb_max), float(tau), float(C), int(cap), d[0].data_ptr(), d[1].data_ptr(), d[2].data_ptr(),
            d[3].data_ptr(), g[0].data_ptr(), g[1].data_ptr(), self._stream())
        self._check(rc, "bifrost_dtmin_neighbours")
        return d, g

    def components(self, count, lst, out=None):
        """Subsystem id (smallest member id; -1 = single) of every particle from neighbour lists."""
        import torch
        if not (isinstance(lst, torch.Tensor) and lst.dim() == 2):
            raise BifrostError("list: expected an [n, cap] int32 CUDA tensor")
        n, cap = int(lst.shape[0]), int(lst.shape[1])
        _dev_i32_rows(count, (), "count"); _dev_i32_rows(lst, (cap,), "list")
        if out is None:
            out = torch.empty((n,), dtype=torch.int32, device=count.device)
        _dev_i32_rows(out, (), "out")
        rc = self._lib.bifrost_components(self._h, n, count.data_ptr(), lst.data_ptr(), cap, out.data_ptr(), self._stream())
        self._check(rc, "bifrost_components")
        return out

    # ---- NEXT-4 ----------------------------------------------------------------------
    def kick(self, vel, acc, h, grad=None, c=0.0, idx=None):
        vel = _dev_f64(vel, (3,), "vel"); acc = _dev_f64(acc, (3,), "acc")
        if grad is not None:
            _dev_f64(grad, (3,), "grad")
        n = vel.shape[0]
        ix, ixp = _dev_idx(idx, "idx")
        rc = self._lib.bifrost_kick(self._h, n, ixp or None, n if ix is None else ix.shape[0], acc.data_ptr(),
                                    None if grad is None else grad.data_ptr(), float(h), float(c), vel.data_ptr(),
                                    self._stream())
        self._check(rc, "bifrost_kick")
        return vel

    def drift(self, pos, vel, h, idx=None):
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel")
        n = pos.shape[0]
        ix, ixp = _dev_idx(idx, "idx")
        rc = self._lib.bifrost_drift(self._h, n, ixp or None, n if ix is None else ix.shape[0], vel.data_ptr(), float(h),
                                     pos.data_ptr(), self._stream())
        self._check(rc, "bifrost_drift")
        return pos

    def fsi_step(self, pos, vel, mass, G, eps_soft, eps, idx=None):
        """One FSI cycle (Eq. 10) in place over idx (None: all)."""
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        ix, ixp = _dev_idx(idx, "idx")
        rc = self._lib.bifrost_fsi_step(self._h, n, pos.data_ptr(), vel.data_ptr(), mass.data_ptr(), ixp or None,
                                        n if ix is None else ix.shape[0], float(G), float(eps_soft), float(eps),
                                        self._stream())
        self._check(rc, "bifrost_fsi_step")

    def set_level_criteria(self, eta, eta_grad, eta_jerk):
        """Eq. 24-29 at every level of hhs_fsi (all three > 0), or off (all three 0, the default)."""
        self._check(self._lib.bifrost_set_level_criteria(self._h, float(eta), float(eta_grad), float(eta_jerk)),
                    "bifrost_set_level_criteria")

    def hhs_fsi(self, pos, vel, mass, G, eps_soft, eta_ff, eta_fb, tau, max_depth=32, log_cap=0, dt_cap=None):
        """One HHS-FSI interval (Eq. 11) in place.  Returns (summary dict, level log as an int64 array [k, 3])."""
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        log = np.zeros((max(int(log_cap), 1), 3), dtype=np.int64)
        summ = np.zeros(3, dtype=np.int64)
        rc = self._lib.bifrost_hhs_fsi(self._h, n, pos.data_ptr(), vel.data_ptr(), mass.data_ptr(), float(G),
                                       float(eps_soft), float(eta_ff), float(eta_fb),
                                       None if dt_cap is None else _dev_f64(dt_cap, (), "dt_cap").data_ptr(), float(tau), int(max_depth),
                                       log.ctypes.data if log_cap else None, int(log_cap), summ.ctypes.data, self._stream())
        self._check(rc, "bifrost_hhs_fsi")
        k = min(int(summ[0]), int(log_cap))
        return {"levels": int(summ[0]), "deepest": int(summ[1]), "fsi_steps": int(summ[2])}, log[:k]

    def kinetic_energy(self, vel, mass, idx=None):
        import torch
        vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        ix, ixp = _dev_idx(idx, "idx")
        out = torch.zeros(1, dtype=torch.float64, device=vel.device)
        rc = self._lib.bifrost_kinetic_energy(self._h, n, vel.data_ptr(), mass.data_ptr(), ixp or None,
                                              n if ix is None else ix.shape[0], out.data_ptr(), self._stream())
        self._check(rc, "bifrost_kinetic_energy")
        return out

    def acc_jerk(self, pos, vel, mass, G, eps, sink_idx=None, src_idx=None, out=None):
        """Acceleration (Eq. 6) and jerk (Eq. 28) in one pass; returns (acc, jerk), each [n, 3]."""
        import torch
        pos = _dev_f64(pos, (3,), "pos"); vel = _dev_f64(vel, (3,), "vel"); mass = _dev_f64(mass, (), "mass")
        n = mass.shape[0]
        si, sip = _dev_idx(sink_idx, "sink_idx"); sj, sjp = _dev_idx(src_idx, "src_idx")
        if out is None:
            out = (torch.zeros((n, 3), dtype=torch.float64, device=pos.device),
                   torch.zeros((n, 3), dtype=torch.float64, device=pos.device))
        _dev_f64(out[0], (3,), "out_acc"); _dev_f64(out[1], (3,), "out_jerk")
        rc = self._lib.bifrost_acc_jerk(self._h, n, pos.data_ptr(), vel.data_ptr(), mass.data_ptr(), sip or None,
                                        n if si is None else si.shape[0], sjp or None, n if sj is None else sj.shape[0],
                                        float(G), float(eps), out[0].data_ptr(), out[1].data_ptr(), self._stream())
        self._check(rc, "bifrost_acc_jerk")
        return out
