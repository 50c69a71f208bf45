"""Pins of the oracle's point-wise pieces (prim->cons, fluxes, implicit E, recovery, reconstruction)
against things fixed by the paper and the mathematics -- not against the oracle itself:
hand-computed textbook values, tensor covariance under a linear change of coordinates, closed
forms/limits, manufactured solutions, polynomial exactness.  CPU only."""
import math

import numpy as np
import pytest

import oracle
from helpers import LEVI, g6_from_matrix, random_spd
from paper_2510_18968_b200 import workloads as wl

FLAT = np.array([1.0, 0, 0, 1.0, 0, 1.0])


# ----------------------------------------------------------------------------------------------
# prim -> cons (Eq. 22-24, 28)
# ----------------------------------------------------------------------------------------------
def test_prim2cons_textbook_values_flat():
    # rho=1, p=1, Gamma=2, v=(0.5,0,0): W=2/sqrt(3), h=rho+2p=3, hW^2=4
    P = np.zeros(14); P[wl.RHO] = 1; P[wl.PRS] = 1; P[wl.VX] = 0.5
    U = oracle.prim2cons_point(P, 2.0)
    W = 2 / math.sqrt(3)
    assert U[0] == pytest.approx(W, rel=1e-15)
    assert U[1] == pytest.approx(4 * 0.5, rel=1e-15)              # S_x = h W^2 v_x
    assert U[4] == pytest.approx(4 - 1 - W, rel=1e-14)            # tau = hW^2 - p - D
    # add E=(0,1,0), B=(0,0,2): Poynting E x B = (2,0,0), energy (1+4)/2
    P[wl.EY] = 1; P[wl.BZ] = 2; P[wl.PSI] = 0.3; P[wl.PHI] = -0.2; P[wl.QCH] = 0.7
    U = oracle.prim2cons_point(P, 2.0)
    assert U[1] == pytest.approx(2 + 2, rel=1e-15)
    assert U[2] == pytest.approx(0, abs=1e-15) and U[3] == pytest.approx(0, abs=1e-15)
    assert U[4] == pytest.approx(4 - 1 + 2.5 - W, rel=1e-14)
    assert np.allclose(U[5:14], [0, 1, 0, 0, 0, 2, 0.3, -0.2, 0.7], rtol=0, atol=0)


def _random_state(rng, g, vmax=0.7, magmax=1.0):
    Gam = rng.choice([4 / 3, 5 / 3, 2.0])
    rho = 10 ** rng.uniform(-3, 1); p = rho * 10 ** rng.uniform(-2, 1)
    h = rho + Gam / (Gam - 1) * p
    unit = lambda d: d / math.sqrt(d @ g @ d)
    v = unit(rng.standard_normal(3)) * rng.uniform(0, vmax)
    mag = 10 ** rng.uniform(-2, magmax)
    B = unit(rng.standard_normal(3)) * math.sqrt(mag * h)
    E = unit(rng.standard_normal(3)) * math.sqrt(mag * h) * rng.uniform(0, 0.5)
    P = np.concatenate([[rho, p], v, E, B, rng.standard_normal(3)])
    return P, Gam


def _transform_cons(U, A):
    """Conserved densities under x' = A x (constant A): scalars and vector densities pick up
    1/det A; contravariant components transform with A, covariant with A^-T."""
    Ainv = np.linalg.inv(A); d = np.linalg.det(A)
    Up = U.copy() / d
    Up[1:4] = Ainv.T @ U[1:4] / d
    Up[5:8] = A @ U[5:8] / d
    Up[8:11] = A @ U[8:11] / d
    return Up


def test_prim2cons_and_flux_covariance_under_linear_map():
    """The same physical state described in coordinates x' = A x has gamma' = A^-T A^-1,
    v' = A v, ... ; densities and fluxes must transform as tensor densities.  This pins every
    index placement and every sqrt(gamma) factor of Eq. 22-28 (reading R1)."""
    rng = np.random.default_rng(7)
    for _ in range(20):
        A = np.eye(3) + 0.3 * rng.standard_normal((3, 3))
        if np.linalg.det(A) < 0.2:
            continue
        Ainv = np.linalg.inv(A); d = np.linalg.det(A)
        gp = Ainv.T @ Ainv
        P, Gam = _random_state(rng, np.eye(3))
        Pp = P.copy()
        for s in (wl.VX, wl.EX, wl.BX):
            Pp[s:s + 3] = A @ P[s:s + 3]
        alpha = rng.uniform(0.5, 1.0)
        beta = 0.2 * rng.standard_normal(3)
        jc = rng.standard_normal(3); sigma = 10 ** rng.uniform(0, 3)
        for mode in (0, 1):
            Fl = np.zeros((3, 14)); Fp = np.zeros((3, 14))
            for k in range(3):
                U, Fl[k] = oracle.state_flux_point(P, k, Gam, alpha, beta, FLAT, mode, sigma, jc[k])
                Up, Fp[k] = oracle.state_flux_point(Pp, k, Gam, alpha, A @ beta, g6_from_matrix(gp), mode, sigma, (A @ jc)[k])
            assert np.allclose(Up, _transform_cons(U, A), rtol=1e-12, atol=1e-13)
            # flux: F'^k(X') = A^k_m * (component transform of F^m(X))
            for k in range(3):
                expect = sum(A[k, m] * _transform_cons(Fl[m], A) for m in range(3))
                assert np.allclose(Fp[k], expect, rtol=1e-11, atol=1e-12), (mode, k)


def test_flux_flat_maxwell_and_hydro_rows():
    """Flat space, alpha=1, beta=0: Faraday d_t B = -curl E, Ampere d_t E = curl B - J, and the
    classic SRHD fluxes (textbook forms), plus the cleaning rows."""
    rng = np.random.default_rng(3)
    P, Gam = _random_state(rng, np.eye(3))
    rho, p = P[0], P[1]; v = P[2:5]; E = P[5:8]; B = P[8:11]; psi, phi, q = P[11:14]
    W = 1 / math.sqrt(1 - v @ v); h = rho + Gam / (Gam - 1) * p
    for k in range(3):
        U, F = oracle.state_flux_point(P, k, Gam, charge_mode=1, jck=0.37)
        for i in range(3):
            # d_t B^i + d_k( [ikj] E_j + delta^ik phi ) = 0 ;  d_t E^i + d_k( -[ikj] B_j + delta^ik psi ) = -J^i
            assert F[8 + i] == pytest.approx(sum(LEVI[i, k, j] * E[j] for j in range(3)) + (phi if i == k else 0), abs=1e-14)
            assert F[5 + i] == pytest.approx(-sum(LEVI[i, k, j] * B[j] for j in range(3)) + (psi if i == k else 0), abs=1e-14)
        assert F[12] == pytest.approx(B[k], abs=1e-15) and F[11] == pytest.approx(E[k], abs=1e-15)
        assert F[0] == pytest.approx(rho * W * v[k], rel=1e-14)
        assert F[13] == pytest.approx(q * v[k] + 0.37, rel=1e-14)
        # energy flux = S^k - D v^k with S = hW^2 v + E x B
        S = h * W * W * v + np.cross(E, B)
        assert F[4] == pytest.approx(S[k] - rho * W * v[k], rel=1e-13)
        # momentum flux = Maxwell + fluid stress
        for j in range(3):
            T = h * W * W * v[k] * v[j] - E[k] * E[j] - B[k] * B[j] + (k == j) * (p + 0.5 * (E @ E + B @ B))
            assert F[1 + j] == pytest.approx(T, rel=1e-13, abs=1e-14)
    # Ohm's law at a face (charge_mode FACE_OHM), Eq. 29 in flat space
    sigma = 12.5
    for k in range(3):
        U, F = oracle.state_flux_point(P, k, Gam, charge_mode=0, sigma=sigma)
        J = q * v + W * sigma * (E + np.cross(v, B) - (v @ E) * v)
        assert F[13] == pytest.approx(J[k], rel=1e-13)


def test_flux_lapse_shift_structure():
    """F(alpha,beta) = alpha F(1,0) - beta^k U for every component (Eq. 27 rows)."""
    rng = np.random.default_rng(4)
    g = random_spd(rng); g6 = g6_from_matrix(g)
    P, Gam = _random_state(rng, g)
    beta = 0.3 * rng.standard_normal(3); alpha = 0.77
    for k in range(3):
        U, F0 = oracle.state_flux_point(P, k, Gam, 1.0, np.zeros(3), g6, 1, 0.0, 0.2)
        U1, F1 = oracle.state_flux_point(P, k, Gam, alpha, beta, g6, 1, 0.0, 0.2)
        assert np.array_equal(U, U1)
        assert np.allclose(F1, alpha * F0 - beta[k] * U, rtol=1e-13, atol=1e-14)


# ----------------------------------------------------------------------------------------------
# implicit E (Eq. 42-43)
# ----------------------------------------------------------------------------------------------
def test_implicit_E_closed_form_equals_newton_and_limits():
    rng = np.random.default_rng(5)
    for t in range(50):
        g = random_spd(rng) if t % 2 else np.eye(3); g6 = g6_from_matrix(g)
        sg = math.sqrt(np.linalg.det(g))
        unit = lambda d: d / math.sqrt(d @ g @ d)
        v = unit(rng.standard_normal(3)) * rng.uniform(0, 0.9)
        B = rng.standard_normal(3); Es = rng.standard_normal(3)
        s = 10 ** rng.uniform(-3, 4)
        Ec = oracle.implicit_E_point(v, s, Es, B, 1.0, g6)
        En = oracle.implicit_E_point(v, s, Es, B, 1.0, g6, newton=True, E0=rng.standard_normal(3), iters=1)
        En2 = oracle.implicit_E_point(v, s, Es, B, 1.0, g6, newton=True, E0=rng.standard_normal(3), iters=3)
        scale = np.max(np.abs(Es)) + np.max(np.abs(B))
        assert np.max(np.abs(Ec - En)) < 1e-11 * scale / min(1.0, 1 - v @ g @ v)     # linear => one Newton step
        assert np.max(np.abs(Ec - En2)) < 1e-13 * scale / min(1.0, 1 - v @ g @ v)
        # the defining equation, evaluated independently
        vD = g @ v; BD = g @ B
        vxB = np.einsum("ijk,j,k->i", LEVI, vD, BD) / sg
        res = (1 + s) * Ec - s * (vD @ Ec) * v + s * vxB - Es
        assert np.max(np.abs(res)) < 1e-13 * (1 + s) * scale
        # limits: sigma -> 0 gives E*, sigma -> infinity gives -v x B
        assert np.allclose(oracle.implicit_E_point(v, 0.0, Es, B, 1.0, g6), Es, rtol=0, atol=0)
        Einf = oracle.implicit_E_point(v, 1e14, Es, B, 1.0, g6)
        assert np.max(np.abs(Einf + vxB)) < 1e-12 * scale / (1 - v @ g @ v)


# ----------------------------------------------------------------------------------------------
# recovery (Eq. 44-50) and the fused implicit solve
# ----------------------------------------------------------------------------------------------
def test_roundtrip_prim_cons_prim_flat_and_curved():
    """north_star pin: prim -> cons -> prim to 1e-12 relative on random physical states."""
    rng = np.random.default_rng(11)
    worst = 0.0
    for t in range(2000):
        g = random_spd(rng) if t % 2 else np.eye(3); g6 = g6_from_matrix(g)
        P, Gam = _random_state(rng, g, vmax=0.7, magmax=1.0)
        alpha = rng.uniform(0.5, 1.0)
        U = oracle.prim2cons_point(P, Gam, alpha, None, g6)
        guess = P.copy(); guess[0] *= 1.3; guess[1] *= 0.7; guess[2:5] *= 0.5
        P2, ev, failed = oracle.c2p_point(U, guess, Gam, 0.0, 0.0, alpha, g6)
        assert not failed and ev <= 20
        vs = max(math.sqrt(P[2:5] @ g @ P[2:5]), 1e-3)
        Bs = math.sqrt(P[8:11] @ g @ P[8:11])
        scale = np.array([P[0], P[1], vs, vs, vs] + [Bs] * 6 + [1, 1, 1])
        worst = max(worst, np.max(np.abs(P2 - P) / scale))
    assert worst < 1e-12, worst


def _manufactured_implicit(rng, g, vmax, magmax):
    """Pick primitives, then build the stage vector whose root they are (Eq. 42 solved for E*)."""
    sg = math.sqrt(np.linalg.det(g))
    P, Gam = _random_state(rng, g, vmax, magmax)
    v, B = P[2:5], P[8:11]
    sigma = 10 ** rng.uniform(0, 8); adt = 0.29 * 10 ** rng.uniform(-4, -2); alpha = rng.uniform(0.5, 1)
    vD = g @ v; BD = g @ B
    vxB = np.einsum("ijk,j,k->i", LEVI, vD, BD) / sg
    unit = lambda d: d / math.sqrt(d @ g @ d)
    E = -vxB + unit(rng.standard_normal(3)) * math.sqrt(B @ g @ B) * rng.uniform(0, 0.3) * min(1.0, 100 / sigma)
    P[5:8] = E
    W = 1 / math.sqrt(1 - v @ vD); s = adt * alpha * sigma * W
    Estar = (1 + s) * E - s * (vD @ E) * v + s * vxB
    U = oracle.prim2cons_point(P, Gam, alpha, None, g6_from_matrix(g))
    U[5:8] = sg * Estar
    return P, U, Gam, adt, sigma, alpha


def test_implicit_recovery_manufactured_solution():
    rng = np.random.default_rng(12)
    evs = []
    for t in range(1500):
        g = random_spd(rng) if t % 2 else np.eye(3); g6 = g6_from_matrix(g)
        P, U, Gam, adt, sigma, alpha = _manufactured_implicit(rng, g, 0.6, 1.0)
        guess = P.copy(); guess[0] *= 1.05; guess[1] *= 0.95; guess[2:5] *= 0.9
        P2, ev, failed = oracle.c2p_point(U, guess, Gam, adt, sigma, alpha, g6)
        assert not failed
        evs.append(ev)
        vs = max(math.sqrt(P[2:5] @ g @ P[2:5]), 1e-3)
        Bs = math.sqrt(P[8:11] @ g @ P[8:11])
        scale = np.array([P[0], P[1], vs, vs, vs] + [Bs] * 6 + [1, 1, 1])
        assert np.max(np.abs(P2 - P) / scale) < 2e-12
        # residual of the defining system, evaluated independently of the oracle (SURVEY pin <= 1e-13)
        sg = math.sqrt(np.linalg.det(g))
        v, E, B = P2[2:5], P2[5:8], P2[8:11]
        vD = g @ v; W = 1 / math.sqrt(1 - v @ vD); s = adt * alpha * sigma * W
        vxB = np.einsum("ijk,j,k->i", LEVI, vD, g @ B) / sg
        ohm = (1 + s) * E - s * (vD @ E) * v + s * vxB - U[5:8] / sg
        assert np.max(np.abs(ohm)) < 1e-13 * (1 + s) * Bs
        U2 = oracle.prim2cons_point(P2, Gam, alpha, None, g6)
        for i in (0, 1, 2, 3, 4):
            ref = max(abs(U[4]) + abs(U[0]), 1e-300)
            assert abs(U2[i] - U[i]) < 1e-13 * ref
    assert np.median(evs) <= 14 and max(evs) <= 60


def test_literal_and_robust_solvers_agree_and_literal_counts():
    """Paper's literal iteration (steps i-v) vs the bracketed solver: same root where both converge.
    Literal-iteration counts are indicative ('<10' intermediate sigma, '<~70' high)."""
    rng = np.random.default_rng(13)
    both = 0
    for t in range(400):
        g = random_spd(rng) if t % 2 else np.eye(3); g6 = g6_from_matrix(g)
        P, U, Gam, adt, sigma, alpha = _manufactured_implicit(rng, g, 0.4, -0.5)   # moderate magnetisation
        guess = P.copy(); guess[1] *= 0.98; guess[2:5] *= 0.97
        Pr, evr, fr = oracle.c2p_point(U, guess, Gam, adt, sigma, alpha, g6)
        Pl, evl, fl = oracle.c2p_point(U, guess, Gam, adt, sigma, alpha, g6, tol=1e-13, maxit=200, literal=True)
        assert not fr
        if fl:
            continue
        both += 1
        vs = max(math.sqrt(P[2:5] @ g @ P[2:5]), 1e-3); Bs = math.sqrt(P[8:11] @ g @ P[8:11])
        scale = np.array([P[0], P[1], vs, vs, vs] + [Bs] * 6 + [1, 1, 1])
        assert np.max(np.abs(Pr - Pl) / scale) < 1e-11
    assert both > 300
    # the paper's shocktube right state (Eq. 51) with a small flow, dt = 1e-3: counts grow with sigma
    P = np.zeros(14); P[0] = 0.125; P[1] = 0.1; P[wl.BY] = -0.5; P[wl.VX] = 0.1
    P[5:8] = -np.cross(P[2:5], P[8:11])
    counts = {}
    for sigma in (1e2, 1e4, 1e6):
        U = oracle.prim2cons_point(P, 2.0)
        guess = P.copy(); guess[1] *= 1.1; guess[2] = 0.08
        Pl, evl, fl = oracle.c2p_point(U, guess, 2.0, 0.29e-3, sigma, tol=1e-13, maxit=300, literal=True)
        assert not fl
        counts[sigma] = evl
    assert counts[1e2] < 12 and counts[1e2] <= counts[1e4] <= counts[1e6] < 150, counts


def test_pressure_newton_derivative_identity_G3():
    """f(p) = p_EOS(rho(p), eps(p)) - p at fixed E,B has, AT THE ROOT, f' = v^2 cs^2 - 1 exactly when
    cs^2 = Gamma (Gamma-1) eps / (1 + Gamma eps) (reading G3 of the garbled Eq. 50; off the root the
    exact derivative is (Gamma-1) v^2 (1 - D W / Z) - 1, which coincides there because Z = h W^2):
    checked by a finite difference of Eq. 44-47 typed out here, and by the quadratic convergence of
    the oracle's literal loop at sigma = 0 (where it is exactly that Newton iteration)."""
    rng = np.random.default_rng(14)
    for _ in range(20):
        P, Gam = _random_state(rng, np.eye(3), 0.6, 0.0)
        U = oracle.prim2cons_point(P, Gam)
        D, S, tau, E, B = U[0], U[1:4], U[4], U[5:8], U[8:11]

        def f_and_fp(p):
            Z = tau + D + p - 0.5 * (E @ E + B @ B)
            v = (S - np.cross(E, B)) / Z
            W = 1 / math.sqrt(1 - v @ v); rho = D / W
            eps = (tau - D * (W - 1) - p * (W * W - 1) - 0.5 * (E @ E + B @ B)) / (D * W)
            cs2 = Gam * (Gam - 1) * eps / (1 + Gam * eps)
            return (Gam - 1) * rho * eps - p, (v @ v) * cs2 - 1

        p0 = P[1]
        hstep = 1e-6 * p0
        fd = (f_and_fp(p0 + hstep)[0] - f_and_fp(p0 - hstep)[0]) / (2 * hstep)
        assert fd == pytest.approx(f_and_fp(p0)[1], rel=1e-6)
        guess = P.copy(); guess[1] *= 1.3
        Pl, evl, fl = oracle.c2p_point(U, guess, Gam, 0.0, 0.0, tol=1e-13, maxit=50, literal=True)
        assert not fl and evl <= 7                      # quadratic: 0.3 -> 1e-13 in <= 6 steps
        assert abs(Pl[1] - P[1]) < 1e-11 * P[1]


# ----------------------------------------------------------------------------------------------
# reconstruction (reading R4)
# ----------------------------------------------------------------------------------------------
def _cell_averages(coef, x_edges):
    """Exact cell averages of the polynomial sum coef[m] x^m."""
    out = np.zeros(len(x_edges) - 1)
    for m, c in enumerate(coef):
        out += c * (x_edges[1:] ** (m + 1) - x_edges[:-1] ** (m + 1)) / (m + 1)
    return out / np.diff(x_edges)


def test_weno5_linear_weights_exact_for_quartics():
    rng = np.random.default_rng(21)
    coef = rng.standard_normal(5)
    edges = np.linspace(-1.0, 1.3, 24)
    ubar = _cell_averages(coef, edges)
    lo, hi = oracle.recon_1d(ubar, wl.RECON_WENO5, eps_w=1e40)        # eps >> beta: linear weights
    poly = lambda x: sum(c * x ** m for m, c in enumerate(coef))
    i = np.arange(2, len(ubar) - 2)
    assert np.max(np.abs(hi[i] - poly(edges[i + 1]))) < 1e-13
    assert np.max(np.abs(lo[i] - poly(edges[i]))) < 1e-13


def test_weno5_fifth_order_and_constant_data():
    errs = []
    for n in (20, 40, 80):
        edges = np.linspace(0, 1, n + 1)
        ubar = -(np.cos(2 * np.pi * edges[1:] + 0.3) - np.cos(2 * np.pi * edges[:-1] + 0.3)) / (2 * np.pi) / np.diff(edges)
        lo, hi = oracle.recon_1d(ubar, wl.RECON_WENO5)
        i = np.arange(2, n - 2)
        errs.append(max(np.max(np.abs(hi[i] - np.sin(2 * np.pi * edges[i + 1] + 0.3))),
                        np.max(np.abs(lo[i] - np.sin(2 * np.pi * edges[i] + 0.3)))))
    assert errs[0] / errs[1] > 20 and errs[1] / errs[2] > 20, errs
    lo, hi = oracle.recon_1d(np.full(12, 3.25), wl.RECON_WENO5)
    assert np.all(lo[2:-2] == 3.25) and np.all(hi[2:-2] == 3.25)
    # mirror symmetry: reversing the data swaps the two faces
    u = np.random.default_rng(1).standard_normal(16)
    lo, hi = oracle.recon_1d(u, wl.RECON_WENO5)
    lor, hir = oracle.recon_1d(u[::-1].copy(), wl.RECON_WENO5)
    assert np.array_equal(lo[2:-2], hir[::-1][2:-2]) and np.array_equal(hi[2:-2], lor[::-1][2:-2])


@pytest.mark.parametrize("scheme", [wl.RECON_MINMOD, wl.RECON_MC])
def test_tvd_linear_exact_monotone_and_clipping(scheme):
    x = np.arange(12.0)
    u = 0.5 * x - 2.0
    lo, hi = oracle.recon_1d(u, scheme)
    assert np.allclose(hi[2:-2], u[2:-2] + 0.25, rtol=0, atol=1e-15)
    assert np.allclose(lo[2:-2], u[2:-2] - 0.25, rtol=0, atol=1e-15)
    # monotone data: face values stay between the neighbouring cell values
    rng = np.random.default_rng(2)
    u = np.cumsum(rng.uniform(0, 1, 40) ** 3)
    lo, hi = oracle.recon_1d(u, scheme)
    i = np.arange(2, 37)
    assert np.all(u[i] <= hi[i]) and np.all(hi[i] <= u[i + 1] + 1e-15)
    assert np.all(u[i] <= lo[i + 1] + 1e-15) and np.all(lo[i + 1] <= u[i + 1])
    # local extremum: zero slope
    u = np.array([0, 1, 2, 5, 2, 1, 0.0])
    lo, hi = oracle.recon_1d(u, scheme)
    assert lo[3] == 5 and hi[3] == 5
    # the two limiters differ on a convex profile: minmod takes the smaller one-sided slope,
    # MC min(2a, 2b, (a+b)/2)
    u = np.array([0, 0, 1, 4, 9, 9, 9.0])      # at i=3: a=3, b=5
    lo, hi = oracle.recon_1d(u, scheme)
    assert hi[3] == pytest.approx(4 + 0.5 * (3.0 if scheme == wl.RECON_MINMOD else 4.0))
