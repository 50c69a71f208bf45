"""Shared test helpers: group-normalised parity norm (SURVEY.md Sec. 8(c) 'Parity norm') and small
NumPy utilities.  No method arithmetic beyond norms."""
import numpy as np

from paper_2510_18968_b200 import workloads as wl


def interior(a, n):
    """Strip ghost zones from a padded (..., nzp, nyp, nxp) array."""
    sl = [slice(None)] * (a.ndim - 3)
    for m in (n[2], n[1], n[0]):
        sl.append(slice(3, 3 + m) if m > 1 else slice(0, 1))
    return a[tuple(sl)]


def prim_group_scales(P, dx_min):
    """Normalisers per primitive field: rho by max rho; p by max p; v by max(max|v|,1e-3);
    E,B by max(|E|,|B|); psi by max(|psi|,|E|); phi by max(|phi|,|B|); q by max(|q|,|E|/dx_min)."""
    mx = lambda a: float(np.max(np.abs(a)))
    vmax = max(mx(P[wl.VX:wl.VZ + 1]), 1e-3)
    Emax, Bmax = mx(P[wl.EX:wl.EZ + 1]), mx(P[wl.BX:wl.BZ + 1])
    em = max(Emax, Bmax, 1e-300)
    s = np.empty(14)
    s[wl.RHO] = mx(P[wl.RHO]); s[wl.PRS] = mx(P[wl.PRS])
    s[wl.VX:wl.VZ + 1] = vmax
    s[wl.EX:wl.BZ + 1] = em
    s[wl.PSI] = max(mx(P[wl.PSI]), Emax, 1e-300 if Emax > 0 else em)
    s[wl.PHI] = max(mx(P[wl.PHI]), Bmax, 1e-300 if Bmax > 0 else em)
    s[wl.QCH] = max(mx(P[wl.QCH]), max(Emax, 1e-300 if Emax > 0 else em) / dx_min)
    return s


def cons_group_scales(U, dx_min):
    """Same grouping for the conserved vector D,S(3),tau,calE(3),calB(3),Psi,Phi,calQ."""
    mx = lambda a: float(np.max(np.abs(a)))
    s = np.empty(14)
    s[0] = mx(U[0])
    s[1:4] = max(mx(U[1:4]), 1e-3 * (mx(U[4]) + mx(U[0])))
    s[4] = mx(U[4])
    Emax, Bmax = mx(U[5:8]), mx(U[8:11])
    em = max(Emax, Bmax, 1e-300)
    s[5:11] = em
    s[11] = max(mx(U[11]), Emax if Emax > 0 else em)
    s[12] = max(mx(U[12]), Bmax if Bmax > 0 else em)
    s[13] = max(mx(U[13]), (Emax if Emax > 0 else em) / dx_min)
    return s


def rel_linf(A, B, scales):
    """Per-field relative L-infinity difference with the given per-field normalisers."""
    return np.array([np.max(np.abs(A[i] - B[i])) / scales[i] for i in range(A.shape[0])])


def g6_from_matrix(g):
    return np.array([g[0, 0], g[0, 1], g[0, 2], g[1, 1], g[1, 2], g[2, 2]])


def random_spd(rng, amp=0.2):
    A = np.eye(3) + amp * rng.standard_normal((3, 3))
    return A @ A.T


LEVI = np.zeros((3, 3, 3))
LEVI[0, 1, 2] = LEVI[1, 2, 0] = LEVI[2, 0, 1] = 1.0
LEVI[0, 2, 1] = LEVI[2, 1, 0] = LEVI[1, 0, 2] = -1.0
