"""CPU ORACLE loader (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Builds ``oracle/rgrmhd_oracle.cpp`` with ``g++ -O2 -ffp-contract=off`` and exposes it through
ctypes.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; ``paper_2510_18968_b200`` never does, and
this package never imports the CUDA binding.

Two builds of the same source: ``liboracle.so`` (single thread: the oracle by definition, and
what ``cpu_baseline`` times) and ``liboracle_omp.so`` (``-fopenmp`` over independent cells, used
only to make the large parity samples finish; results are thread-count independent).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rgrmhd_oracle.cpp")
_LIBS: Dict[object, C.CDLL] = {}

NPRIM = NCONS = 14


def build(force: bool = False) -> None:
    """Compile both oracle variants in-tree (idempotent)."""
    for omp in (False, True):
        out = os.path.join(_HERE, "liboracle_omp.so" if omp else "liboracle.so")
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-Wno-unknown-pragmas"]
        if omp:
            cmd.append("-fopenmp")
        cmd += ["-o", out + ".tmp%d" % os.getpid(), _SRC]
        subprocess.check_call(cmd)
        os.replace(out + ".tmp%d" % os.getpid(), out)


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


def build_count() -> str:
    """The instrumented variant (-DORACLE_COUNT_FLOPS: a counting scalar replaces double; oracle/flopcount.h).  Used by
    oracle/count_flops.py only."""
    out = os.path.join(_HERE, "liboracle_count.so")
    hdr = os.path.join(_HERE, "flopcount.h")
    if not (os.path.exists(out) and os.path.getmtime(out) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr))):
        tmp = out + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-Wno-unknown-pragmas",
                               "-DORACLE_COUNT_FLOPS", "-I", _HERE, "-o", tmp, _SRC])
        os.replace(tmp, out)
    return out


def lib(omp=False) -> C.CDLL:
    """omp: False (single thread: the oracle by definition), True (OpenMP build), or "count" (instrumented build)."""
    if omp not in _LIBS:
        if omp == "count":
            path = build_count()
        else:
            build()
            path = os.path.join(_HERE, "liboracle_omp.so" if omp else "liboracle.so")
        if omp is True:   # libgomp reads these when it is first loaded; an unset thread count makes it 10x slower on small grids here
            ncpu = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
            os.environ.setdefault("OMP_NUM_THREADS", str(ncpu))
        L = C.CDLL(path)
        L.oracle_max_speed.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.oracle_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.oracle_sigma_point.restype = C.c_double
        L.oracle_sigma_point.argtypes = [C.c_int] + [C.c_double] * 5
        for name in ("oracle_prim2cons_point", "oracle_c2p_point", "oracle_c2p_literal_point", "oracle_c2p_plain_point",
                     "oracle_implicit_E_point", "oracle_state_flux_point", "oracle_recon_1d"):
            getattr(L, name).restype = C.c_int
        if omp is True:   # the cores this process may run on (a container's cpu set can be smaller than the host's count)
            L.oracle_set_threads(len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
        _LIBS[omp] = L
    return _LIBS[omp]


def omp_threads() -> int:
    """Threads the OpenMP build runs on."""
    return lib(True).oracle_set_threads(0)


def _dp(a: Optional[np.ndarray]):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ptr_table(arrs: Sequence[np.ndarray]):
    T = C.POINTER(C.c_double) * len(arrs)
    return T(*[_dp(a) for a in arrs])


def make_params(p: dict) -> Params:
    q = Params()
    q.n[:] = list(p["n"]); q.dx[:] = list(p["dx"]); q.ng = int(p.get("ng", 3)); q.bc[:] = list(p["bc"])
    q.gamma_eos = p["gamma_eos"]; q.sigma_model = int(p.get("sigma_model", 0)); q.sigma0 = p.get("sigma0", 0.0)
    q.sigma_exp = p.get("sigma_exp", 0.0); q.sigma_dref = p.get("sigma_dref", 1.0); q.kappa = p.get("kappa", 1.0)
    q.rho_floor = p.get("rho_floor", 0.0); q.k_atmo = p.get("k_atmo", 0.0); q.c2p_tol = p.get("c2p_tol", 0.0)
    q.c2p_max_iter = int(p.get("c2p_max_iter", 0)); q.charge_mode = int(p.get("charge_mode", 1))
    q.weno_eps = p.get("weno_eps", 0.0); q.device = 0
    q.wave_speed_mode = int(p.get("wave_speed_mode", 0)); q.wave_rho_switch = p.get("wave_rho_switch", 0.0)
    return q


class Oracle:
    """Handle-level wrapper mirroring include/rgrmhd.h (host NumPy arrays)."""

    def __init__(self, params: dict, omp=False):
        self.L = lib(omp)
        self.par = make_params(params)
        self.h = C.c_void_p()
        rc = self.L.oracle_create(C.byref(self.h), C.byref(self.par))
        if rc != 0:
            raise ValueError("oracle_create failed: %d" % rc)
        n = params["n"]
        self.shape = tuple(int(m + 6) if m > 1 else 1 for m in (n[2], n[1], n[0]))

    def __del__(self):
        if getattr(self, "h", None):
            self.L.oracle_destroy(self.h)
            self.h = None

    def _check(self, rc, what):
        if rc != 0:
            raise RuntimeError("%s failed: %d" % (what, rc))

    def set_metric(self, metric: np.ndarray):
        m = np.ascontiguousarray(metric, dtype=np.float64)
        assert m.shape == (16,) + self.shape, (m.shape, self.shape)
        self._check(self.L.oracle_set_metric(self.h, _dp(m[0]), _ptr_table([m[1], m[2], m[3]]),
                                             _ptr_table([m[4 + i] for i in range(6)]),
                                             _ptr_table([m[10 + i] for i in range(6)])), "set_metric")

    def set_sigma(self, sigma: np.ndarray):
        s = np.ascontiguousarray(sigma, dtype=np.float64)
        assert s.shape == self.shape
        self._check(self.L.oracle_set_sigma(self.h, _dp(s)), "set_sigma")

    def set_prims(self, prims: np.ndarray):
        p = np.ascontiguousarray(prims, dtype=np.float64)
        assert p.shape == (14,) + self.shape
        self._check(self.L.oracle_set_prims(self.h, _ptr_table([p[i] for i in range(14)])), "set_prims")

    def set_solver(self, which: str):
        """'plain' (default: bisection inside an un-accelerated fixed point) or 'robust' (secant + Anderson)."""
        self._check(self.L.oracle_set_solver(self.h, {"plain": 0, "robust": 1}[which]), "set_solver")

    def step(self, dt: float, scheme: int):
        self._check(self.L.oracle_step(self.h, C.c_double(dt), int(scheme)), "step")

    def max_speed(self) -> float:
        out = C.c_double()
        self._check(self.L.oracle_max_speed(self.h, C.byref(out)), "max_speed")
        return out.value

    def get_prims(self) -> np.ndarray:
        p = np.empty((14,) + self.shape)
        self._check(self.L.oracle_get_prims(self.h, _ptr_table([p[i] for i in range(14)])), "get_prims")
        return p

    def get_cons(self) -> np.ndarray:
        u = np.empty((14,) + self.shape)
        self._check(self.L.oracle_get_cons(self.h, _ptr_table([u[i] for i in range(14)])), "get_cons")
        return u

    def rhs(self, scheme: int) -> np.ndarray:
        f = np.empty((14,) + self.shape)
        self._check(self.L.oracle_rhs(self.h, int(scheme), _ptr_table([f[i] for i in range(14)])), "rhs")
        return f

    def sources(self) -> np.ndarray:
        """Explicit sources S of the current primitives (interior cells; ghosts of the result are zero)."""
        f = np.zeros((14,) + self.shape)
        self._check(self.L.oracle_sources(self.h, _ptr_table([f[i] for i in range(14)])), "sources")
        return f

    def face_states(self, scheme: int, d: int, i: int, j: int = 0, k: int = 0):
        """(PL, PR, fixups) at the lower face in direction d of interior cell (i, j, k); fills the ghosts first."""
        self.get_prims()
        PL, PR = np.empty(14), np.empty(14)
        r = self.L.oracle_face_states(self.h, int(scheme), int(d), int(i), int(j), int(k), _dp(PL), _dp(PR))
        if r < 0:
            raise RuntimeError("face_states failed")
        return PL, PR, r

    def ghost_fill(self, field: np.ndarray) -> np.ndarray:
        f = np.ascontiguousarray(field, dtype=np.float64).copy()
        self._check(self.L.oracle_ghost_fill(self.h, _dp(f)), "ghost_fill")
        return f

    def stats(self) -> dict:
        s = Stats()
        self._check(self.L.oracle_get_stats(self.h, C.byref(s)), "get_stats")
        d = {k: getattr(s, k) for k, _ in Stats._fields_ if k != "reserved"}
        d["face_fixups"] = s.reserved      # reading R4 fix-ups (rho/p fallbacks + |v| limiter hits) of the RHS evaluations
        return d

    def reset_stats(self):
        self.L.oracle_reset_stats(self.h)


def from_workload(w, fields: Optional[dict] = None, omp=False, n=None, bc=None, solver: str = "plain",
                  **over) -> Oracle:
    """Create an oracle handle for workload `w` (or a sub-block of it) and load its fields."""
    par = w.params(n=n, bc=bc)
    par.update(over)
    o = Oracle(par, omp=omp)
    o.set_solver(solver)
    f = fields if fields is not None else w.fields()
    o.set_metric(f["metric"])
    if f["sigma"] is not None and par["sigma_model"] == 1:
        o.set_sigma(f["sigma"])
    o.set_prims(f["prims"])
    return o


# ---- point-wise wrappers (used by the pins) -------------------------------------------------------
_G_FLAT = np.array([1.0, 0, 0, 1.0, 0, 1.0])


def _a(x, n=None):
    a = np.ascontiguousarray(x, dtype=np.float64)
    if n is not None:
        assert a.shape == (n,)
    return a


def prim2cons_point(P, gamma_eos, alpha=1.0, beta=None, g6=None):
    U = np.empty(14)
    lib().oracle_prim2cons_point(C.c_double(gamma_eos), C.c_double(alpha), _dp(_a(beta, 3)) if beta is not None else None,
                                 _dp(_a(_G_FLAT if g6 is None else g6, 6)), _dp(_a(P, 14)), _dp(U))
    return U


def wave_speeds_point(P, k, gamma_eos, alpha=1.0, beta=None, g6=None):
    """(lambda-, lambda+) of the ideal-GRMHD bound (A9) for one state in direction k."""
    lm, lp = C.c_double(), C.c_double()
    lib().oracle_wave_speeds_point(C.c_double(gamma_eos), C.c_double(alpha), _dp(_a(beta, 3)) if beta is not None else None,
                                   _dp(_a(_G_FLAT if g6 is None else g6, 6)), C.c_int(k), _dp(_a(P, 14)),
                                   C.byref(lm), C.byref(lp))
    return lm.value, lp.value


def tableau(time_scheme: int):
    """(s, At, wt, A, w) of the oracle's double Butcher tableau for a time scheme (0..4), cut to s stages."""
    At, A = np.zeros((4, 4)), np.zeros((4, 4))
    wt, w = np.zeros(4), np.zeros(4)
    s = lib().oracle_tableau(int(time_scheme), _dp(At), _dp(wt), _dp(A), _dp(w))
    if s < 0:
        raise ValueError("unknown time scheme")
    return s, At[:s, :s], wt[:s], A[:s, :s], w[:s]


def sigma_point(model, sigma0, sigma_exp, sigma_dref, Dhat, sigma_cell=0.0):
    return lib().oracle_sigma_point(int(model), float(sigma0), float(sigma_exp), float(sigma_dref), float(Dhat),
                                    float(sigma_cell))


def c2p_point(U, guess, gamma_eos, adt=0.0, sigma=0.0, alpha=1.0, g6=None, tol=0.0, maxit=0, literal=False,
              plain=False):
    """Returns (prims, evals, failed).  Default: the robust solver; plain=True: c2p_plain (maxit = cap on
    outer passes); literal=True: the paper's loop."""
    P = _a(guess, 14).copy()
    fn = (lib().oracle_c2p_literal_point if literal else lib().oracle_c2p_plain_point if plain
          else lib().oracle_c2p_point)
    if literal and tol <= 0:
        tol = 1e-13
    if literal and maxit <= 0:
        maxit = 100
    r = fn(C.c_double(gamma_eos), C.c_double(alpha), _dp(_a(_G_FLAT if g6 is None else g6, 6)), _dp(_a(U, 14)),
           C.c_double(adt), C.c_double(sigma), C.c_double(tol), C.c_int(maxit), _dp(P))
    return P, (r if r >= 0 else -r - 1), r < 0


def implicit_E_point(v, s, Estar, B, alpha=1.0, g6=None, newton=False, E0=None, iters=1):
    E = np.empty(3)
    E0 = _a(np.zeros(3) if E0 is None else E0, 3)
    lib().oracle_implicit_E_point(C.c_double(alpha), _dp(_a(_G_FLAT if g6 is None else g6, 6)), _dp(_a(v, 3)),
                                  C.c_double(s), _dp(_a(Estar, 3)), _dp(_a(B, 3)), C.c_int(1 if newton else 0),
                                  _dp(E0), C.c_int(iters), _dp(E))
    return E


def state_flux_point(P, k, gamma_eos, alpha=1.0, beta=None, g6=None, charge_mode=1, sigma=0.0, jck=0.0):
    U = np.empty(14); F = np.empty(14)
    lib().oracle_state_flux_point(C.c_double(gamma_eos), C.c_double(alpha), _dp(_a(beta, 3)) if beta is not None else None,
                                  _dp(_a(_G_FLAT if g6 is None else g6, 6)), C.c_int(k), _dp(_a(P, 14)),
                                  C.c_int(charge_mode), C.c_double(sigma), C.c_double(jck), _dp(U), _dp(F))
    return U, F


def recon_1d(u, scheme, eps_w=0.0):
    u = _a(u)
    lo = np.full_like(u, np.nan); hi = np.full_like(u, np.nan)
    lib().oracle_recon_1d(C.c_int(scheme), C.c_double(eps_w), C.c_int(u.size), _dp(u), _dp(lo), _dp(hi))
    return lo, hi
