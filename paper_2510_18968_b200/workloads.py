"""Seeded synthetic workloads (input generators only -- no method arithmetic).

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle's
tests.  It produces initial primitive fields, the fixed 3+1 metric and (where needed) a
per-cell conductivity array as NumPy float64 arrays, so that no transcendental function is
ever evaluated separately on the two sides.  It imports neither ``oracle/`` nor the CUDA
binding and contains none of the scheme's arithmetic (no prim->cons, no fluxes, no solver).

Workloads are synthetic stand-ins shaped like the paper's tests (Sec. IV) with the
sizes/values of BASELINE.json ``configs`` (gaps filled as stated in SURVEY.md Sec. 8(d) and
DESIGN.md "Input recipe"):

  cfg1  1D resistive shocktube            (Eq. 51; BASELINE config 1)
  cfg2  1D self-similar current sheet     (Eq. 54-55)
  cfg3  3D rotated CP Alfven wave         (Eq. 56-59)
  cfg4  3D blast in a static curved metric(PAPER.md:303-321 relative, curved metric)
  cfg5  3D TOV-like magnetised star       (Eq. 60)
and the paper's own tests that BASELINE.json does not list:
  e2    1D shocktube, sigma = sigma0 D^gamma (Eq. 51-52)
  e3    2D cylindrical explosion 200^2      (Eq. 53)

Layout: every field is a padded array of shape (nzp, nyp, nxp) (x fastest), where
n?p = n? + 2*ng for an active direction (n? > 1) and 1 for an inactive one.

A workload can generate any sub-block of its global grid (``fields(lo, shape)``) because all
fields are pointwise functions of the global cell index; the oracle uses this to check
sampled sub-blocks of the 256^3 / 512^3 runs.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional, Sequence, Tuple

import numpy as np
from scipy.special import erf as _erf  # input generation only (cfg2 profile)

NG = 3

PRIM_NAMES = ["rho", "p", "vx", "vy", "vz", "Ex", "Ey", "Ez", "Bx", "By", "Bz", "psi", "phi", "q"]
CONS_NAMES = ["D", "Sx", "Sy", "Sz", "tau", "calEx", "calEy", "calEz",
              "calBx", "calBy", "calBz", "Psi", "Phi", "calQ"]
METRIC_NAMES = ["alpha", "betax", "betay", "betaz",
                "gxx", "gxy", "gxz", "gyy", "gyz", "gzz",
                "Kxx", "Kxy", "Kxz", "Kyy", "Kyz", "Kzz"]
NPRIM, NCONS, NMETRIC = 14, 14, 16
(RHO, PRS, VX, VY, VZ, EX, EY, EZ, BX, BY, BZ, PSI, PHI, QCH) = range(14)

# enums mirrored from include/rgrmhd.h (plain integers, no arithmetic)
BC_PERIODIC, BC_OUTFLOW, BC_EXTERNAL = 0, 1, 2
SIGMA_UNIFORM, SIGMA_ARRAY, SIGMA_POWER_D, SIGMA_ATMO = 0, 1, 2, 3
RECON_MINMOD, RECON_MC, RECON_WENO5 = 0, 1, 2
CHARGE_FACE_OHM, CHARGE_CELL_CURRENT, CHARGE_DIV_E = 0, 1, 2
WAVE_LIGHT, WAVE_MHD_INSIDE = 0, 1
# time schemes: `scheme` argument of step = recon | (time << 8)
TIME_SSP2_222, TIME_SSP2_332, TIME_SSP3_332, TIME_SSP3_433, TIME_SSP2_222_GENERAL = 0, 1 << 8, 2 << 8, 3 << 8, 4 << 8


def splitmix64_uniform(seed: int, idx: np.ndarray) -> np.ndarray:
    """Counter-based uniform numbers in [0,1): splitmix64 of (seed, idx), top 53 bits."""
    idx = np.asarray(idx).astype(np.uint64)
    with np.errstate(over="ignore"):
        z = (np.uint64(seed) + (idx + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15))
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def padded_shape(n: Sequence[int], ng: int = NG) -> Tuple[int, int, int]:
    """(nzp, nyp, nxp) of a padded field for interior sizes n = (nx, ny, nz)."""
    return tuple(int(m + 2 * ng) if m > 1 else 1 for m in (n[2], n[1], n[0]))  # type: ignore


@dataclasses.dataclass
class Workload:
    name: str
    n: Tuple[int, int, int]                 # global interior cells (nx, ny, nz)
    dx: Tuple[float, float, float]
    x0: Tuple[float, float, float]          # lower corner of global cell (0,0,0)
    bc: Tuple[int, int, int]
    gamma_eos: float
    recon: int
    cfl: float
    nsteps: int
    sigma_model: int = SIGMA_UNIFORM
    sigma0: float = 0.0
    sigma_exp: float = 0.0
    sigma_dref: float = 1.0
    kappa: float = 1.0
    rho_floor: float = 0.0
    k_atmo: float = 0.0
    charge_mode: int = CHARGE_CELL_CURRENT
    seed: int = 0
    flat: bool = True
    extra: dict = dataclasses.field(default_factory=dict)

    # ---- grid helpers -------------------------------------------------------------------
    @property
    def ncells(self) -> int:
        return int(self.n[0]) * int(self.n[1]) * int(self.n[2])

    @property
    def dt(self) -> float:
        """CFL * min active dx / (coordinate light speed bound).  For these workloads the
        lapse <= 1, shift = 0 and gamma^kk <= 1, so alpha*sqrt(gamma^kk) <= 1: the value
        used is CFL * dx_min (exact for the flat configs); tests obtain the library's own
        max-speed reduction separately."""
        act = [self.dx[d] for d in range(3) if self.n[d] > 1]
        return self.cfl * min(act)

    def params(self, n: Optional[Sequence[int]] = None, bc: Optional[Sequence[int]] = None) -> dict:
        """Plain-dict version of rgrmhd_params (see include/rgrmhd.h)."""
        n = tuple(self.n if n is None else n)
        bc = tuple(self.bc if bc is None else bc)
        return dict(n=n, dx=tuple(self.dx), ng=NG, bc=bc, gamma_eos=self.gamma_eos,
                    sigma_model=self.sigma_model, sigma0=self.sigma0, sigma_exp=self.sigma_exp,
                    sigma_dref=self.sigma_dref, kappa=self.kappa, rho_floor=self.rho_floor,
                    k_atmo=self.k_atmo, charge_mode=self.charge_mode)

    def coords(self, lo=(0, 0, 0), shape=None):
        """Cell-centre coordinates (X, Y, Z) of the padded sub-block, broadcastable 3D arrays,
        and the matching global integer indices (I, J, K)."""
        shape = tuple(self.n if shape is None else shape)
        out_x, out_i = [], []
        for d in range(3):
            if self.n[d] > 1:
                g = NG if shape[d] > 1 else 0
                ii = np.arange(lo[d] - g, lo[d] + shape[d] + g, dtype=np.int64)
                xx = self.x0[d] + (ii.astype(np.float64) + 0.5) * self.dx[d]
            else:
                ii = np.zeros(1, dtype=np.int64)
                xx = np.array([self.x0[d] + 0.5 * self.dx[d]])
            out_x.append(xx)
            out_i.append(ii)
        X = out_x[0][None, None, :]
        Y = out_x[1][None, :, None]
        Z = out_x[2][:, None, None]
        I = out_i[0][None, None, :]
        J = out_i[1][None, :, None]
        K = out_i[2][:, None, None]
        return (X, Y, Z), (I, J, K)

    def linear_interior_index(self, I, J, K) -> np.ndarray:
        """Global linear interior index with ghost indices mapped into the interior by the
        workload's own boundary rule (wrap for periodic, clamp for outflow)."""
        idx = []
        for d, a in enumerate((I, J, K)):
            m = self.n[d]
            if self.bc[d] == BC_PERIODIC:
                idx.append(np.mod(a, m))
            else:
                idx.append(np.clip(a, 0, m - 1))
        return (idx[0] + self.n[0] * (idx[1] + self.n[1] * idx[2])).astype(np.int64)

    # ---- field generation ---------------------------------------------------------------
    def fields(self, lo=(0, 0, 0), shape=None) -> Dict[str, np.ndarray]:
        """Return {'prims': (14,nzp,nyp,nxp), 'metric': (16,...), 'sigma': (...) or None}
        for the padded sub-block of interior cells [lo, lo+shape)."""
        shape = tuple(self.n if shape is None else shape)
        (X, Y, Z), (I, J, K) = self.coords(lo, shape)
        full = np.broadcast_shapes(X.shape, Y.shape, Z.shape)
        gen = _GENERATORS[self.extra["kind"]]
        prims, metric, sigma = gen(self, X, Y, Z, I, J, K, full)
        prims = np.ascontiguousarray(np.stack([np.broadcast_to(a, full) for a in prims]).astype(np.float64))
        metric = np.ascontiguousarray(np.stack([np.broadcast_to(a, full) for a in metric]).astype(np.float64))
        if sigma is not None:
            sigma = np.ascontiguousarray(np.broadcast_to(sigma, full).astype(np.float64))
        return {"prims": prims, "metric": metric, "sigma": sigma}


# ------------------------------------------------------------------------------------------
# metric helpers (inputs only: analytic grid functions)
# ------------------------------------------------------------------------------------------
def _flat_metric(full):
    one = np.ones(full)
    zero = np.zeros(full)
    return [one, zero, zero, zero, one, zero, zero, one, zero, one,
            zero, zero, zero, zero, zero, zero]


def _conformally_flat_metric(X, Y, Z, M, a_soft, full):
    """alpha = 1 - M/(2 r_s), gamma_ij = psi^4 delta_ij, psi = 1 + M/(2 r_s),
    r_s = sqrt(r^2 + a_soft^2); zero shift, K_ij = 0  (BASELINE.json configs 4, 5)."""
    rs = np.sqrt(X * X + Y * Y + Z * Z + a_soft * a_soft)
    alpha = 1.0 - M / (2.0 * rs)
    psi = 1.0 + M / (2.0 * rs)
    p4 = (psi * psi) * (psi * psi)
    zero = np.zeros(full)
    return [alpha, zero, zero, zero, p4, zero, zero, p4, zero, p4,
            zero, zero, zero, zero, zero, zero], alpha, psi


# ------------------------------------------------------------------------------------------
# generators
# ------------------------------------------------------------------------------------------
def _gen_shocktube(w: Workload, X, Y, Z, I, J, K, full):
    e = w.extra
    left = X < e.get("x_split", 0.0)
    z = np.zeros(full)
    P = [z.copy() for _ in range(NPRIM)]
    for name, idx in (("rho", RHO), ("p", PRS), ("vx", VX), ("vy", VY), ("vz", VZ),
                      ("Bx", BX), ("By", BY), ("Bz", BZ)):
        l, r = e["left"].get(name, 0.0), e["right"].get(name, 0.0)
        P[idx] = np.where(left, l, r) + z
    # E = -v x B (flat space); zero for v = 0
    vx, vy, vz, bx, by, bz = P[VX], P[VY], P[VZ], P[BX], P[BY], P[BZ]
    P[EX] = -(vy * bz - vz * by)
    P[EY] = -(vz * bx - vx * bz)
    P[EZ] = -(vx * by - vy * bx)
    return P, _flat_metric(full), None


def _gen_current_sheet(w: Workload, X, Y, Z, I, J, K, full):
    e = w.extra
    z = np.zeros(full)
    P = [z.copy() for _ in range(NPRIM)]
    P[RHO] = z + e["rho"]
    P[PRS] = z + e["p"]
    eta = 1.0 / w.sigma0
    P[BY] = z + e["B0"] * _erf(X / (2.0 * math.sqrt(eta * e["t0"])))
    return P, _flat_metric(full), None


def alfven_speed(rho, p, gamma_eos, B0, etaA):
    """Eq. 58 -- an input parameter of the exact solution, h = enthalpy density."""
    h = rho + gamma_eos / (gamma_eos - 1.0) * p
    den = h + B0 * B0 * (1.0 + etaA * etaA)
    return math.sqrt(2.0 * B0 * B0 / den / (1.0 + math.sqrt(1.0 - (2.0 * etaA * B0 * B0 / den) ** 2)))


def alfven_exact(w: Workload, X, Y, Z, t: float):
    """Exact CP Alfven wave fields (B, v, E) at time t (Eq. 56-59 rotated onto nhat)."""
    e = w.extra
    nh = np.array(e["nhat"], dtype=np.float64)
    e1 = np.array(e["e1"], dtype=np.float64)
    e2 = np.array(e["e2"], dtype=np.float64)
    B0, etaA, vA = e["B0"], e["etaA"], e["vA"]
    kwave = e["k"]           # phase = k * (nhat.x - vA t)
    s = nh[0] * X + nh[1] * Y + nh[2] * Z
    ph = kwave * (s - vA * t)
    c, sn = np.cos(ph), np.sin(ph)
    Bp = [etaA * B0 * (c * e1[i] + sn * e2[i]) for i in range(3)]     # transverse part
    B = [B0 * nh[i] + Bp[i] for i in range(3)]
    v = [-(vA / B0) * Bp[i] for i in range(3)]
    E = [-(v[1] * B[2] - v[2] * B[1]), -(v[2] * B[0] - v[0] * B[2]), -(v[0] * B[1] - v[1] * B[0])]
    return B, v, E


def _gen_alfven(w: Workload, X, Y, Z, I, J, K, full):
    e = w.extra
    z = np.zeros(full)
    P = [z.copy() for _ in range(NPRIM)]
    P[RHO] = z + e["rho"]
    P[PRS] = z + e["p"]
    B, v, E = alfven_exact(w, X, Y, Z, 0.0)
    for i in range(3):
        P[VX + i] = v[i] + z
        P[EX + i] = E[i] + z
        P[BX + i] = B[i] + z
    return P, _flat_metric(full), None


def _gen_blast(w: Workload, X, Y, Z, I, J, K, full):
    e = w.extra
    z = np.zeros(full)
    metric, alpha, psi = _conformally_flat_metric(X, Y, Z, e["M"], e["a_soft"], full)
    P = [z.copy() for _ in range(NPRIM)]
    inside = (X * X + Y * Y) < e["r_in"] ** 2
    P[RHO] = np.where(inside, e["rho_in"], e["rho_out"]) + z
    P[PRS] = np.where(inside, e["p_in"], e["p_out"]) + z
    P[BX] = z + e["Bx"]
    u = splitmix64_uniform(w.seed, w.linear_interior_index(I, J, K))
    sigma = 10.0 ** (e["sigma_log10_max"] * u)
    return P, metric, sigma


def _tov_profile(w: Workload, X, Y, Z):
    e = w.extra
    M, a, Kp, rho_c, rho_atmo = e["M"], e["a_soft"], e["K"], e["rho_c"], e["rho_atmo"]
    rs = np.sqrt(X * X + Y * Y + Z * Z + a * a)
    alpha = 1.0 - M / (2.0 * rs)
    alpha_c = 1.0 - M / (2.0 * a)
    h_c = 1.0 + 2.0 * Kp * rho_c
    rho = np.maximum((h_c * alpha_c / alpha - 1.0) / (2.0 * Kp), rho_atmo)
    return rho, Kp * rho * rho


def _tov_A(w: Workload, X, Y, Z, Ab):
    """Vector potential of Eq. 60: A_phi = varpi^2 max(Ab (P - Pcut), 0)^2,
    A_x = -y A_phi / varpi^2, A_y = x A_phi / varpi^2."""
    e = w.extra
    _, P = _tov_profile(w, X, Y, Z)
    Pcut = e["pcut_frac"] * e["K"] * e["rho_c"] ** 2
    f = np.maximum(Ab * (P - Pcut), 0.0) ** 2
    return -Y * f, X * f


def _tov_B(w: Workload, X, Y, Z, Ab):
    """B^i = [ijk] d_j A_k / sqrt(gamma), centred differences of the analytic A (spacing dx)."""
    e = w.extra
    dx, dy, dz = w.dx
    rs = np.sqrt(X * X + Y * Y + Z * Z + e["a_soft"] ** 2)
    psi = 1.0 + e["M"] / (2.0 * rs)
    sqrtg = psi ** 6
    Ax_zp, Ay_zp = _tov_A(w, X, Y, Z + dz, Ab)
    Ax_zm, Ay_zm = _tov_A(w, X, Y, Z - dz, Ab)
    _, Ay_xp = _tov_A(w, X + dx, Y, Z, Ab)
    _, Ay_xm = _tov_A(w, X - dx, Y, Z, Ab)
    Ax_yp, _ = _tov_A(w, X, Y + dy, Z, Ab)
    Ax_ym, _ = _tov_A(w, X, Y - dy, Z, Ab)
    Bx = -(Ay_zp - Ay_zm) / (2.0 * dz) / sqrtg
    By = (Ax_zp - Ax_zm) / (2.0 * dz) / sqrtg
    Bz = ((Ay_xp - Ay_xm) / (2.0 * dx) - (Ax_yp - Ax_ym) / (2.0 * dy)) / sqrtg
    return Bx, By, Bz, psi


def _tov_Ab(w: Workload) -> float:
    """Scale A_b so that max |B| (gamma-norm) on the y=0 meridional slice of the GLOBAL grid
    equals extra['Bmax'].  B is quadratic in A_b.  Cached per workload."""
    if "_Ab" in w.extra:
        return w.extra["_Ab"]
    (X, _, Z), _ = w.coords((0, 0, 0), w.n)
    Y0 = np.array(w.x0[1] + (w.n[1] // 2 + 0.5) * w.dx[1]).reshape(1, 1, 1)
    Bx, By, Bz, psi = _tov_B(w, X, Y0, Z, 1.0)
    bmax = float(np.max(psi ** 2 * np.sqrt(Bx * Bx + By * By + Bz * Bz)))
    Ab = math.sqrt(w.extra["Bmax"] / bmax) if bmax > 0 else 0.0
    w.extra["_Ab"] = Ab
    return Ab


def _gen_tov(w: Workload, X, Y, Z, I, J, K, full):
    e = w.extra
    z = np.zeros(full)
    metric, alpha, psi = _conformally_flat_metric(X, Y, Z, e["M"], e["a_soft"], full)
    rho, prs = _tov_profile(w, X, Y, Z)
    u = splitmix64_uniform(w.seed, w.linear_interior_index(I, J, K))
    inside = rho > e["rho_atmo"]
    rho = np.where(inside, rho * (1.0 + e["pert"] * (2.0 * u - 1.0)), rho)
    Bx, By, Bz, _ = _tov_B(w, X, Y, Z, _tov_Ab(w))
    P = [z.copy() for _ in range(NPRIM)]
    P[RHO] = rho + z
    P[PRS] = prs + z
    P[BX], P[BY], P[BZ] = Bx + z, By + z, Bz + z
    return P, metric, None


def _gen_explosion2d(w: Workload, X, Y, Z, I, J, K, full):
    """Eq. 53: rho_in inside r_in, rho_out outside r_out, log-linear ramp between (the pressure
    likewise); uniform B^x; everything else zero."""
    e = w.extra
    z = np.zeros(full)
    r = np.sqrt(X * X + Y * Y) + z
    t = np.clip((r - e["r_in"]) / (e["r_out"] - e["r_in"]), 0.0, 1.0)
    P = [z.copy() for _ in range(NPRIM)]
    P[RHO] = np.exp((1.0 - t) * math.log(e["rho_in"]) + t * math.log(e["rho_out"]))
    P[PRS] = np.exp((1.0 - t) * math.log(e["p_in"]) + t * math.log(e["p_out"]))
    P[BX] = z + e["Bx"]
    return P, _flat_metric(full), None


_GENERATORS = {"shocktube": _gen_shocktube, "current_sheet": _gen_current_sheet,
               "alfven": _gen_alfven, "blast": _gen_blast, "tov": _gen_tov, "explosion2d": _gen_explosion2d}


# ------------------------------------------------------------------------------------------
# workload factories (BASELINE.json configs; sizes overridable for tests)
# ------------------------------------------------------------------------------------------
def shocktube(n=400, sigma0=1e6, recon=RECON_WENO5, cfl=0.4, axis=0, t_end=0.4,
              left=None, right=None, gamma_eos=2.0) -> Workload:
    """cfg1 (BASELINE config 1): x in [-0.5, 0.5], outflow, states of BASELINE.json."""
    left = left or dict(rho=1.0, p=1.0, Bx=0.5, By=1.0, Bz=0.0)
    right = right or dict(rho=0.125, p=0.1, Bx=0.5, By=-1.0, Bz=0.0)
    nn = [1, 1, 1]
    nn[axis] = n
    dx = 1.0 / n
    assert axis == 0, "generator splits along x"
    w = Workload("cfg1_shocktube", tuple(nn), (dx, dx, dx), (-0.5, 0.0, 0.0),
                 (BC_OUTFLOW,) * 3, gamma_eos, recon, cfl, 0,
                 sigma_model=SIGMA_UNIFORM, sigma0=sigma0,
                 extra=dict(kind="shocktube", left=left, right=right))
    w.nsteps = int(round(t_end / w.dt))
    return w


def shocktube_paper(n=400, sigma0=1e6, gamma_exp=0, recon=RECON_MINMOD, cfl=0.25, t_end=0.4) -> Workload:
    """The paper's own shocktube (Eq. 51): B = (0, +-0.5, 0), Gamma = 2, minmod, CFL 0.25, x in
    [-0.5, 0.5]; conductivity sigma0 D^gamma_exp (Eq. 52; gamma_exp = 0 is the uniform case, the paper runs 0, 6, 9, 12
    at sigma0 = 1e6 and dx = 0.0025)."""
    w = shocktube(n=n, sigma0=sigma0, recon=recon, cfl=cfl, t_end=t_end,
                  left=dict(rho=1.0, p=1.0, By=0.5), right=dict(rho=0.125, p=0.1, By=-0.5))
    w.name = "e2_shocktube_sigmaD%d" % gamma_exp
    if gamma_exp:
        w.sigma_model, w.sigma_exp, w.sigma_dref = SIGMA_POWER_D, float(gamma_exp), 1.0
    return w


def explosion2d(n=200, sigma0=1e6, recon=RECON_MINMOD, cfl=0.25, t_end=4.0) -> Workload:
    """The paper's 2D cylindrical explosion (Eq. 53): n x n cells on [-6, 6]^2, Gamma = 4/3,
    outflow, uniform sigma; rho_in = 0.01, p_in = 1 inside r = 0.8, rho_out = p_out = 1e-3 outside r = 1, B^x = 0.05."""
    dx = 12.0 / n
    w = Workload("e3_explosion2d", (n, n, 1), (dx, dx, dx), (-6.0, -6.0, 0.0), (BC_OUTFLOW,) * 3, 4.0 / 3.0,
                 recon, cfl, 0, sigma_model=SIGMA_UNIFORM, sigma0=sigma0,
                 extra=dict(kind="explosion2d", r_in=0.8, r_out=1.0, rho_in=0.01, p_in=1.0, rho_out=1e-3, p_out=1e-3,
                            Bx=0.05))
    w.nsteps = int(round(t_end / w.dt))
    return w


def current_sheet(n=800, sigma0=100.0, B0=1.0, p=50.0, recon=RECON_MC, cfl=0.25,
                  t0=1.0, t_end=10.0, half_width=1.5) -> Workload:
    """cfg2 (BASELINE config 2): self-similar current sheet, erf profile at t0."""
    dx = 2.0 * half_width / n
    w = Workload("cfg2_current_sheet", (n, 1, 1), (dx, dx, dx), (-half_width, 0.0, 0.0),
                 (BC_OUTFLOW,) * 3, 4.0 / 3.0, recon, cfl, 0,
                 sigma_model=SIGMA_UNIFORM, sigma0=sigma0,
                 extra=dict(kind="current_sheet", rho=1.0, p=p, B0=B0, t0=t0))
    w.nsteps = int(round((t_end - t0) / w.dt))
    return w


def alfven3d(n=128, sigma0=1e8, recon=RECON_WENO5, cfl=0.25, nsteps=20) -> Workload:
    """cfg3 (BASELINE config 3): CP Alfven wave along (1,1,1)/sqrt(3) on the periodic unit cube."""
    s3, s2, s6 = math.sqrt(3.0), math.sqrt(2.0), math.sqrt(6.0)
    rho, p, B0, etaA, g = 1.0, 1.0, 1.0, 1.0, 4.0 / 3.0
    vA = alfven_speed(rho, p, g, B0, etaA)
    dx = 1.0 / n
    return Workload("cfg3_alfven3d", (n, n, n), (dx, dx, dx), (0.0, 0.0, 0.0),
                    (BC_PERIODIC,) * 3, g, recon, cfl, nsteps,
                    sigma_model=SIGMA_UNIFORM, sigma0=sigma0,
                    extra=dict(kind="alfven", rho=rho, p=p, B0=B0, etaA=etaA, vA=vA,
                               nhat=(1 / s3, 1 / s3, 1 / s3), e1=(1 / s2, -1 / s2, 0.0),
                               e2=(1 / s6, 1 / s6, -2 / s6), k=2.0 * math.pi * s3))


def alfven1d(n=100, sigma0=1e6, recon=RECON_MC, cfl=0.25, B0=2.0 / math.sqrt(3.0),
             gamma_eos=2.0, periods=1.0) -> Workload:
    """The paper's own 1D CP Alfven wave: rho = p = etaA = 1, B0 = 1.1547,
    Gamma = 2 -> v_A = 0.5; x in [-0.5, 0.5], periodic, one period t = 2."""
    rho, p, etaA = 1.0, 1.0, 1.0
    vA = alfven_speed(rho, p, gamma_eos, B0, etaA)
    dx = 1.0 / n
    w = Workload("alfven1d", (n, 1, 1), (dx, dx, dx), (-0.5, 0.0, 0.0), (BC_PERIODIC,) * 3,
                 gamma_eos, recon, cfl, 0, sigma_model=SIGMA_UNIFORM, sigma0=sigma0,
                 extra=dict(kind="alfven", rho=rho, p=p, B0=B0, etaA=etaA, vA=vA,
                            nhat=(1.0, 0.0, 0.0), e1=(0.0, 1.0, 0.0), e2=(0.0, 0.0, 1.0),
                            k=2.0 * math.pi))
    w.nsteps = int(round(periods * (1.0 / vA) / w.dt))
    return w


def blast_curved(n=256, recon=RECON_WENO5, cfl=0.25, nsteps=20, seed=4) -> Workload:
    """cfg4 (BASELINE config 4): cylindrical blast, conformally flat static metric, random sigma."""
    dx = 1.0 / n
    return Workload("cfg4_blast_curved", (n, n, n), (dx, dx, dx), (-0.5, -0.5, -0.5),
                    (BC_OUTFLOW,) * 3, 4.0 / 3.0, recon, cfl, nsteps,
                    sigma_model=SIGMA_ARRAY, sigma0=0.0, seed=seed, flat=False,
                    extra=dict(kind="blast", M=0.1, a_soft=0.5, r_in=0.1, rho_in=1e-2, p_in=1.0,
                               rho_out=1e-4, p_out=3e-5, Bx=0.1, sigma_log10_max=6.0))


def tov_like(n=512, recon=RECON_WENO5, cfl=0.125, nsteps=10, seed=5) -> Workload:
    """cfg5 (BASELINE config 5): hydrostatic Gamma=2 polytrope in an analytic conformally flat
    metric, poloidal B from Eq. 60, sigma = sigma0 (D/rho_c)^2, atmosphere floor."""
    L = 12.0
    dx = 2.0 * L / n
    rho_c = 1.28e-3
    return Workload("cfg5_tov_like", (n, n, n), (dx, dx, dx), (-L, -L, -L),
                    (BC_OUTFLOW,) * 3, 2.0, recon, cfl, nsteps,
                    sigma_model=SIGMA_POWER_D, sigma0=1e8, sigma_exp=2.0, sigma_dref=rho_c,
                    rho_floor=1e-10, k_atmo=100.0, seed=seed, flat=False,
                    extra=dict(kind="tov", M=1.4, a_soft=2.60078, K=100.0, rho_c=rho_c,
                               rho_atmo=1e-10, pcut_frac=0.04, pert=1e-3,
                               Bmax=1e-4 * math.sqrt(rho_c)))


CONFIGS = {"cfg1": shocktube, "cfg2": current_sheet, "cfg3": alfven3d,
           "cfg4": blast_curved, "cfg5": tov_like, "e2": shocktube_paper, "e3": explosion2d}


def get(name: str, **kw) -> Workload:
    return CONFIGS[name](**kw)
