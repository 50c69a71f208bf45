"""Thin ctypes binding of ``include/rgrmhd.h`` (argument marshalling only).

Every step of the path runs in the CUDA kernels of ``librgrmhd.so``; this module only converts
NumPy arrays / torch tensors to plain pointers.  There is no CPU fallback: ``load()`` raises when
the library is missing, and the library returns ``E_CUDA`` when no device is usable.  This module
never imports ``oracle``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# RGRMHD_LIB: load another build of the same library (kernel-variant experiments); default: the in-tree build
_LIB_PATH = os.environ.get("RGRMHD_LIB") or os.path.join(_HERE, "librgrmhd.so")
_LIB: Optional[C.CDLL] = None

NPRIM = NCONS = 14
NMETRIC = 16

SYMBOLS = ["rgrmhd_params_default", "rgrmhd_create", "rgrmhd_destroy", "rgrmhd_set_stream", "rgrmhd_set_metric",
           "rgrmhd_set_sigma", "rgrmhd_set_prims", "rgrmhd_step", "rgrmhd_max_speed", "rgrmhd_get_prims",
           "rgrmhd_get_cons", "rgrmhd_get_stats", "rgrmhd_reset_stats", "rgrmhd_set_rhs_variant", "rgrmhd_get_rhs_variant", "rgrmhd_step_begin", "rgrmhd_step_continue", "rgrmhd_halo_doubles",
           "rgrmhd_halo_pack", "rgrmhd_halo_unpack", "rgrmhd_max_speed_static",
           "rgrmhd_launch_count", "rgrmhd_flush", "rgrmhd_set_timing", "rgrmhd_get_timing", "rgrmhd_measure_fp64_peak",
           "rgrmhd_strerror", "rgrmhd_last_cuda_error"]

KERNEL_CLASSES = ("c2p", "ghost", "rhs")


class Params(C.Structure):
    _fields_ = [("n", C.c_int * 3), ("dx", C.c_double * 3), ("ng", C.c_int), ("bc", C.c_int * 3),
                ("gamma_eos", C.c_double), ("sigma_model", C.c_int), ("sigma0", C.c_double),
                ("sigma_exp", C.c_double), ("sigma_dref", C.c_double), ("kappa", C.c_double),
                ("rho_floor", C.c_double), ("k_atmo", C.c_double), ("c2p_tol", C.c_double),
                ("c2p_max_iter", C.c_int), ("charge_mode", C.c_int), ("weno_eps", C.c_double),
                ("device", C.c_int), ("wave_speed_mode", C.c_int), ("wave_rho_switch", C.c_double)]


class Stats(C.Structure):
    _fields_ = [("c2p_solves", C.c_longlong), ("c2p_evals", C.c_longlong), ("c2p_failures", C.c_longlong),
                ("floor_resets", C.c_longlong), ("c2p_max_evals", C.c_int), ("reserved", C.c_int)]


class RgrmhdError(RuntimeError):
    def __init__(self, what: str, code: int, detail: str = ""):
        super().__init__("%s failed: %d (%s)%s" % (what, code, _strerror(code), (" -- " + detail) if detail else ""))
        self.code = code


def load() -> C.CDLL:
    """Load ``librgrmhd.so`` (built in-tree by ``paper_2510_18968_b200.build``).  Fails loudly."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError("%s is missing: run `python -m paper_2510_18968_b200.build` "
                              "(there is no CPU fallback)" % _LIB_PATH)
        L = C.CDLL(_LIB_PATH)
        vp, dp = C.c_void_p, C.POINTER(C.c_double)
        L.rgrmhd_params_default.argtypes = [C.POINTER(Params)]
        L.rgrmhd_create.argtypes = [C.POINTER(vp), C.POINTER(Params)]
        L.rgrmhd_destroy.argtypes = [vp]
        L.rgrmhd_set_stream.argtypes = [vp, vp]
        L.rgrmhd_set_metric.argtypes = [vp, vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.rgrmhd_set_sigma.argtypes = [vp, vp]
        L.rgrmhd_set_prims.argtypes = [vp, C.POINTER(vp)]
        L.rgrmhd_step.argtypes = [vp, C.c_double, C.c_int]
        L.rgrmhd_max_speed.argtypes = [vp, dp]
        L.rgrmhd_get_prims.argtypes = [vp, C.POINTER(vp)]
        L.rgrmhd_get_cons.argtypes = [vp, C.POINTER(vp)]
        L.rgrmhd_get_stats.argtypes = [vp, C.POINTER(Stats)]
        L.rgrmhd_reset_stats.argtypes = [vp]
        L.rgrmhd_flush.argtypes = [vp]
        L.rgrmhd_set_rhs_variant.argtypes = [vp, C.c_int]
        L.rgrmhd_get_rhs_variant.argtypes = [vp, C.POINTER(C.c_int)]
        L.rgrmhd_step_begin.argtypes = [vp, C.c_double, C.c_int]
        L.rgrmhd_step_continue.argtypes = [vp, C.POINTER(C.c_int)]
        L.rgrmhd_halo_doubles.argtypes = [vp, C.c_int, C.POINTER(C.c_longlong)]
        L.rgrmhd_halo_pack.argtypes = [vp, C.c_int, C.c_int, vp]
        L.rgrmhd_halo_unpack.argtypes = [vp, C.c_int, C.c_int, vp]
        L.rgrmhd_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.rgrmhd_set_timing.argtypes = [vp, C.c_int]
        L.rgrmhd_get_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.rgrmhd_measure_fp64_peak.argtypes = [C.c_int, C.c_int, dp]
        L.rgrmhd_strerror.argtypes = [C.c_int]
        L.rgrmhd_strerror.restype = C.c_char_p
        L.rgrmhd_last_cuda_error.argtypes = [vp]
        L.rgrmhd_last_cuda_error.restype = C.c_char_p
        for s in SYMBOLS:
            if s not in ("rgrmhd_strerror", "rgrmhd_last_cuda_error"):
                getattr(L, s).restype = C.c_int
        _LIB = L
    return _LIB


def _strerror(code: int) -> str:
    try:
        return load().rgrmhd_strerror(code).decode()
    except Exception:  # pragma: no cover
        return "?"


def params_default() -> Params:
    p = Params()
    load().rgrmhd_params_default(C.byref(p))
    return p


def make_params(p: dict, device: int = 0) -> Params:
    """rgrmhd_params from the plain dict produced by ``workloads.Workload.params()``."""
    q = params_default()
    q.n[:] = list(p["n"]); q.dx[:] = list(p["dx"]); q.ng = int(p.get("ng", 3)); q.bc[:] = list(p["bc"])
    q.gamma_eos = p["gamma_eos"]
    for k in ("sigma_model", "c2p_max_iter", "charge_mode", "wave_speed_mode"):
        if k in p:
            setattr(q, k, int(p[k]))
    for k in ("sigma0", "sigma_exp", "sigma_dref", "kappa", "rho_floor", "k_atmo", "c2p_tol", "weno_eps", "wave_rho_switch"):
        if k in p:
            setattr(q, k, float(p[k]))
    q.device = int(device)
    return q


def _ptr(a) -> int:
    """Address of a contiguous float64 NumPy array (host) or torch tensor (host or device)."""
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"], "need contiguous float64"
        return a.ctypes.data
    # torch tensor (duck-typed so that importing this module does not import torch)
    assert str(a.dtype) == "torch.float64" and a.is_contiguous(), "need contiguous float64"
    return a.data_ptr()


def _table(arrs: Sequence) -> "C.Array":
    T = C.c_void_p * len(arrs)
    return T(*[_ptr(a) for a in arrs])


STATIC_MAX_CELLS = 16777216   # RGRMHD_STATIC_MAX_CELLS
E_TOO_LARGE = -5              # RGRMHD_E_TOO_LARGE


def max_speed_static(n, dx, metric, prims, gamma_eos: float, wave_speed_mode: int, wave_rho_switch: float, out,
                     device: int = 0, stream: int = 0) -> None:
    """rgrmhd_max_speed_static: the CFL reduction without a handle and without any allocation (scratch in a fixed
    device array of the library).  ``metric``: the first 10 padded fields of the metric stack (alpha, beta, gamma) as
    CUDA tensors; ``prims``: the 14 padded primitive fields as CUDA tensors, or None in mode LIGHT; ``out``: a CUDA
    float64 tensor of one element, written asynchronously on ``stream``.  Argument marshalling only."""
    L = load()
    ni = (C.c_int * 3)(*[int(v) for v in n])
    dxi = (C.c_double * 3)(*[float(v) for v in dx])
    for a in list(metric[:10]) + (list(prims) if prims is not None else []) + [out]:
        assert getattr(a, "is_cuda", False), "rgrmhd_max_speed_static takes device pointers only"
    rc = L.rgrmhd_max_speed_static(ni, dxi, _table([metric[i] for i in range(10)]),
                                   _table([prims[i] for i in range(NPRIM)]) if prims is not None else None,
                                   C.c_double(gamma_eos), int(wave_speed_mode), C.c_double(wave_rho_switch), int(device),
                                   C.c_void_p(stream), C.c_void_p(_ptr(out)))
    if rc != 0:
        raise RgrmhdError("rgrmhd_max_speed_static", rc)


class Rgrmhd:
    """Handle wrapper with the names of the C-ABI.  Field arguments are stacks ``(nfields, nzp, nyp,
    nxp)`` (or sequences of per-field arrays) of float64: NumPy arrays (host) or torch tensors (host or
    CUDA).  Output goes into caller-provided arrays when given, else into new NumPy arrays."""

    def __init__(self, params: dict, device: int = 0):
        self.L = load()
        self.par = make_params(params, device)
        self.h = C.c_void_p()
        rc = self.L.rgrmhd_create(C.byref(self.h), C.byref(self.par))
        if rc != 0:
            self.h = None
            raise RgrmhdError("rgrmhd_create", rc)
        n = params["n"]
        self.n = tuple(int(m) for m in n)
        self.shape = tuple(int(m + 6) if m > 1 else 1 for m in (n[2], n[1], n[0]))

    def close(self):
        if getattr(self, "h", None):
            self.L.rgrmhd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # pragma: no cover
            pass

    def _check(self, rc: int, what: str):
        if rc != 0:
            detail = self.L.rgrmhd_last_cuda_error(self.h).decode() if rc == -3 else ""
            raise RgrmhdError(what, rc, detail)

    def set_stream(self, cuda_stream: int):
        self._check(self.L.rgrmhd_set_stream(self.h, C.c_void_p(cuda_stream)), "rgrmhd_set_stream")

    def set_metric(self, metric):
        assert len(metric) == NMETRIC and tuple(metric[0].shape) == self.shape, (len(metric), metric[0].shape, self.shape)
        self._keep = metric
        self._check(self.L.rgrmhd_set_metric(self.h, C.c_void_p(_ptr(metric[0])), _table([metric[1 + i] for i in range(3)]),
                                             _table([metric[4 + i] for i in range(6)]),
                                             _table([metric[10 + i] for i in range(6)])), "rgrmhd_set_metric")

    def set_sigma(self, sigma):
        assert tuple(sigma.shape) == self.shape
        self._check(self.L.rgrmhd_set_sigma(self.h, C.c_void_p(_ptr(sigma))), "rgrmhd_set_sigma")

    def set_prims(self, prims):
        assert len(prims) == NPRIM and tuple(prims[0].shape) == self.shape
        self._check(self.L.rgrmhd_set_prims(self.h, _table([prims[i] for i in range(NPRIM)])), "rgrmhd_set_prims")

    def step(self, dt: float, scheme: int):
        self._check(self.L.rgrmhd_step(self.h, C.c_double(dt), int(scheme)), "rgrmhd_step")

    def max_speed(self) -> float:
        out = C.c_double()
        self._check(self.L.rgrmhd_max_speed(self.h, C.byref(out)), "rgrmhd_max_speed")
        return out.value

    def get_prims(self, out=None):
        if out is None:
            out = np.empty((NPRIM,) + self.shape)
        self._check(self.L.rgrmhd_get_prims(self.h, _table([out[i] for i in range(NPRIM)])), "rgrmhd_get_prims")
        return out

    def get_cons(self, out=None):
        if out is None:
            out = np.empty((NCONS,) + self.shape)
        self._check(self.L.rgrmhd_get_cons(self.h, _table([out[i] for i in range(NCONS)])), "rgrmhd_get_cons")
        return out

    def stats(self) -> dict:
        s = Stats()
        self._check(self.L.rgrmhd_get_stats(self.h, C.byref(s)), "rgrmhd_get_stats")
        return {k: getattr(s, k) for k, _ in Stats._fields_ if k != "reserved"}

    def reset_stats(self):
        self._check(self.L.rgrmhd_reset_stats(self.h), "rgrmhd_reset_stats")

    def flush(self):
        """Enqueue the deferred final recovery of the last step (no host synchronisation)."""
        self._check(self.L.rgrmhd_flush(self.h), "rgrmhd_flush")

    def set_rhs_variant(self, variant: int):
        self._check(self.L.rgrmhd_set_rhs_variant(self.h, int(variant)), "rgrmhd_set_rhs_variant")

    def step_begin(self, dt: float, scheme: int):
        self._check(self.L.rgrmhd_step_begin(self.h, C.c_double(dt), int(scheme)), "rgrmhd_step_begin")

    def step_continue(self) -> bool:
        """Runs the next part; True if one more exchange + continue are due."""
        more = C.c_int()
        self._check(self.L.rgrmhd_step_continue(self.h, C.byref(more)), "rgrmhd_step_continue")
        return bool(more.value)

    def halo_doubles(self, direction: int) -> int:
        out = C.c_longlong()
        self._check(self.L.rgrmhd_halo_doubles(self.h, int(direction), C.byref(out)), "rgrmhd_halo_doubles")
        return out.value

    def halo_pack(self, direction: int, side: int, buf):
        self._check(self.L.rgrmhd_halo_pack(self.h, int(direction), int(side), C.c_void_p(_ptr(buf))), "rgrmhd_halo_pack")

    def halo_unpack(self, direction: int, side: int, buf):
        self._check(self.L.rgrmhd_halo_unpack(self.h, int(direction), int(side), C.c_void_p(_ptr(buf))), "rgrmhd_halo_unpack")

    def get_rhs_variant(self) -> int:
        out = C.c_int()
        self._check(self.L.rgrmhd_get_rhs_variant(self.h, C.byref(out)), "rgrmhd_get_rhs_variant")
        return out.value

    def set_timing(self, enable: bool):
        self._check(self.L.rgrmhd_set_timing(self.h, int(bool(enable))), "rgrmhd_set_timing")

    def get_timing(self) -> dict:
        """{class: (milliseconds, launches)} accumulated since the last call."""
        ms = (C.c_double * 3)(); ln = (C.c_longlong * 3)()
        self._check(self.L.rgrmhd_get_timing(self.h, ms, ln), "rgrmhd_get_timing")
        return {k: (ms[i], ln[i]) for i, k in enumerate(KERNEL_CLASSES)}

    def launch_count(self) -> int:
        out = C.c_longlong()
        self._check(self.L.rgrmhd_launch_count(self.h, C.byref(out)), "rgrmhd_launch_count")
        return out.value


def measure_fp64_peak(device: int = 0, repeats: int = 5) -> float:
    out = C.c_double()
    rc = load().rgrmhd_measure_fp64_peak(int(device), int(repeats), C.byref(out))
    if rc != 0:
        raise RgrmhdError("rgrmhd_measure_fp64_peak", rc)
    return out.value


def from_workload(w, fields: Optional[dict] = None, n=None, bc=None, device: int = 0, **over) -> Rgrmhd:
    """Create a handle for workload ``w`` (or a sub-block of it) and load its fields."""
    par = w.params(n=n, bc=bc)
    par.update(over)
    g = Rgrmhd(par, device=device)
    f = fields if fields is not None else w.fields()
    g.set_metric(f["metric"])
    if f["sigma"] is not None and par["sigma_model"] == 1:
        g.set_sigma(f["sigma"])
    g.set_prims(f["prims"])
    return g
