"""Pins of oracle parts that round 1 left to conventions or to a second typing of the same formulas: the
K_ij / shift / G^i source terms, max speed with a shift, the atmosphere rule (reading R9) and the face
fix-ups (reading R4) -- each against a closed form or a hand-computed value.  CPU only.

Arrays are (field, z, y, x); metric fields alpha, beta^x..z, gamma xx xy xz yy yz zz, K xx..zz."""
import math

import numpy as np
import pytest

import oracle
from helpers import interior
from paper_2510_18968_b200 import workloads as wl

GAMMA = 1 - 1 / math.sqrt(2)          # IMEX-SSP2(2,2,2), Eq. 35-37


def _grid(n, dx):
    """Cell-centre coordinates of the padded grid, origin at the first interior cell centre."""
    ax = [(np.arange(-3, m + 3) if m > 1 else np.zeros(1)) * d for m, d in zip(n, dx)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return X, Y, Z


def _flat_metric(shape):
    m = np.zeros((16,) + shape)
    m[0] = 1.0; m[4] = m[7] = m[9] = 1.0
    return m


def _uniform_prims(shape, rho, p, v, E, B, psi, phi, q):
    P = np.zeros((14,) + shape)
    P[0], P[1] = rho, p
    for i in range(3):
        P[2 + i], P[5 + i], P[8 + i] = v[i], E[i], B[i]
    P[11], P[12], P[13] = psi, phi, q
    return P


# ----------------------------------------------------------------------------------------------
# explicit sources (Eq. 27 S; Eq. 39-40; reading R1 / SURVEY O6)
# ----------------------------------------------------------------------------------------------
def test_sources_extrinsic_curvature_closed_form():
    """Uniform state at rest on gamma_ij = a^2 delta_ij, K_ij = -H a^2 delta_ij, alpha = 1, beta = 0 (a flat FRW
    slice): K = gamma^ij K_ij = -3H and T^ij K_ij = -H [3p + (E^2+B^2)/2], so
      S(tau) = alpha sqrt(gamma) T^ij K_ij = -H a^3 [3p + (E^2+B^2)/2],
      S(Phi) = -alpha Phi (K + kappa),  S(Psi) = -alpha Psi (K + kappa) + alpha calQ,  S(calE^i) = -alpha calQ v^i = 0,
    and every other source vanishes (no metric gradient)."""
    n, dx = (6, 5, 4), (0.1, 0.1, 0.1)
    a, H, kappa, Gam = 1.3, 0.37, 0.8, 5 / 3
    o = oracle.Oracle(dict(n=n, dx=dx, bc=(0, 0, 0), gamma_eos=Gam, sigma0=0.0, kappa=kappa))
    m = np.zeros((16,) + o.shape)
    m[0] = 1.0
    m[4] = m[7] = m[9] = a * a
    m[10] = m[13] = m[15] = -H * a * a
    rho, p, psi, phi, q = 0.9, 0.4, 0.21, -0.33, 0.17
    E, B = np.array([0.2, -0.1, 0.3]), np.array([0.5, 0.25, -0.4])       # coordinate components
    o.set_metric(m); o.set_prims(_uniform_prims(o.shape, rho, p, (0, 0, 0), E, B, psi, phi, q))
    S = interior(o.sources(), n)
    E2, B2 = a * a * (E @ E), a * a * (B @ B)
    sg = a ** 3
    exp = np.zeros(14)
    exp[4] = -H * sg * (3 * p + 0.5 * (E2 + B2))
    exp[12] = -(sg * phi) * (-3 * H + kappa)
    exp[11] = -(sg * psi) * (-3 * H + kappa) + sg * q
    for v in range(14):
        assert np.allclose(S[v], exp[v], rtol=1e-13, atol=1e-15), (v, S[v].ravel()[0], exp[v])


def test_sources_and_rhs_linear_shift_closed_form():
    """Uniform state, flat gamma, alpha = 1, LINEAR shift beta^i = A^i_j x^j (non-symmetric A: index placement
    matters).  4th-order differences and face averages are exact on linear functions, and for a uniform state HLLE
    returns F = alpha G - beta^k U exactly, so to round-off
      S(S_i) = S_j d_i beta^j = S_j A^j_i,   S(calB^i) = -calB^k A^i_k,   S(calE^i) = -calE^k A^i_k - calQ v^i,
      S(Phi) = -kappa Phi,  S(Psi) = calQ - kappa Psi,  S(D) = S(tau) = S(calQ) = 0,
      RHS = -div F + S = tr(A) U + S        (the transport of a density by the shift)."""
    n, dx = (7, 6, 5), (0.1, 0.07, 0.13)
    Gam, kappa = 4 / 3, 1.0
    A = np.array([[0.11, -0.07, 0.05], [0.02, -0.13, 0.09], [-0.06, 0.04, 0.08]])      # A[i][j] = d_j beta^i
    o = oracle.Oracle(dict(n=n, dx=dx, bc=(1, 1, 1), gamma_eos=Gam, sigma0=0.0, kappa=kappa))
    X, Y, Z = _grid(n, dx)
    m = _flat_metric(o.shape)
    for i in range(3):
        m[1 + i] = A[i, 0] * X + A[i, 1] * Y + A[i, 2] * Z + 0.01 * (i + 1)
    v, E, B = np.array([0.2, -0.3, 0.1]), np.array([0.15, 0.05, -0.2]), np.array([0.4, -0.25, 0.3])
    P = _uniform_prims(o.shape, 1.1, 0.6, v, E, B, 0.07, -0.12, 0.09)
    o.set_metric(m); o.set_prims(P)
    U = interior(o.get_cons(), n)[:, 0, 0, 0]
    S = interior(o.sources(), n)
    exp = np.zeros(14)
    exp[1:4] = U[1:4] @ A                      # S_j A^j_i
    exp[8:11] = -A @ U[8:11]                   # -A^i_k calB^k
    exp[5:8] = -A @ U[5:8] - U[13] * v
    exp[12] = -kappa * U[12]
    exp[11] = U[13] - kappa * U[11]
    scale = np.max(np.abs(U))
    for f in range(14):
        assert np.allclose(S[f], exp[f], rtol=0, atol=1e-14 * scale), (f, S[f].ravel()[0], exp[f])
    # whole right-hand side away from the boundary (outflow ghosts of P are uniform; the shift is given in ghosts)
    for scheme in (wl.RECON_WENO5, wl.RECON_MC):
        F = interior(o.rhs(scheme), n)
        for f in range(14):
            assert np.allclose(F[f], np.trace(A) * U[f] + exp[f], rtol=0, atol=2e-13 * scale), (scheme, f)


def test_sources_conformally_flat_linear_lapse_and_metric_closed_form():
    """gamma_ij = f delta_ij with LINEAR f and alpha (4th-order differences exact), K_ij = 0, beta = 0, uniform
    primitives.  Then gamma^jk Gamma^i_jk = -d_i f / (2 f^2), so
      G^i = d_i alpha / f + alpha d_i f / (2 f^2),
      S(calB^i) = Phi G^i,  S(calE^i) = Psi G^i - alpha calQ v^i,
      S(Phi) = calB^k d_k alpha - alpha kappa Phi,  S(Psi) = calE^k d_k alpha + alpha calQ - alpha kappa Psi,
      S(S_i) = 1/2 alpha sqrt(gamma) [h W^2 sum(v^j)^2 + 3p/f - sum(E^j)^2 - sum(B^j)^2 + 3 (E^2+B^2)/(2f)] d_i f
               - (tau + D) d_i alpha,
      S(tau) = -S^j d_j alpha."""
    n, dx = (6, 5, 7), (0.05, 0.04, 0.03)
    Gam, kappa = 2.0, 0.7
    ca, cf = np.array([0.3, -0.2, 0.15]), np.array([0.4, 0.25, -0.35])
    o = oracle.Oracle(dict(n=n, dx=dx, bc=(1, 1, 1), gamma_eos=Gam, sigma0=0.0, kappa=kappa))
    X, Y, Z = _grid(n, dx)
    al = 0.8 + ca[0] * X + ca[1] * Y + ca[2] * Z
    f = 1.2 + cf[0] * X + cf[1] * Y + cf[2] * Z
    m = np.zeros((16,) + o.shape)
    m[0] = al; m[4] = m[7] = m[9] = f
    rho, p, psi, phi, q = 0.7, 0.9, 0.31, -0.27, 0.13
    v, E, B = np.array([0.25, -0.15, 0.2]), np.array([0.1, 0.3, -0.2]), np.array([-0.35, 0.2, 0.45])
    o.set_metric(m); o.set_prims(_uniform_prims(o.shape, rho, p, v, E, B, psi, phi, q))
    S = interior(o.sources(), n)
    U = interior(o.get_cons(), n)
    al_i, f_i = interior(al[None], n)[0], interior(f[None], n)[0]
    sg = f_i ** 1.5
    W2 = 1 / (1 - f_i * (v @ v)); h = rho + Gam / (Gam - 1) * p
    E2, B2 = f_i * (E @ E), f_i * (B @ B)
    brack = h * W2 * (v @ v) + 3 * p / f_i - E @ E - B @ B + 1.5 * (E2 + B2) / f_i
    for i in range(3):
        Gi = ca[i] / f_i + al_i * cf[i] / (2 * f_i ** 2)
        assert np.allclose(S[8 + i], U[12] * Gi, rtol=1e-12, atol=1e-15)
        assert np.allclose(S[5 + i], U[11] * Gi - al_i * U[13] * v[i], rtol=1e-12, atol=1e-15)
        assert np.allclose(S[1 + i], 0.5 * al_i * sg * brack * cf[i] - (U[4] + U[0]) * ca[i], rtol=1e-12, atol=1e-15)
    SU = U[1:4] / f_i                                               # S^j = gamma^jk S_k
    assert np.allclose(S[4], -(SU[0] * ca[0] + SU[1] * ca[1] + SU[2] * ca[2]), rtol=1e-12, atol=1e-15)
    assert np.allclose(S[12], U[8] * ca[0] + U[9] * ca[1] + U[10] * ca[2] - al_i * kappa * U[12], rtol=1e-12, atol=1e-15)
    assert np.allclose(S[11], U[5] * ca[0] + U[6] * ca[1] + U[7] * ca[2] + al_i * U[13] - al_i * kappa * U[11],
                       rtol=1e-12, atol=1e-15)
    assert not S[0].any() and not S[13].any()


# ----------------------------------------------------------------------------------------------
# a7: max speed with a shift (Eq. 30, reading R14)
# ----------------------------------------------------------------------------------------------
def shifted_diagonal_metric(shape, n, dx):
    """Diagonal gamma_ij = diag(gx, gy, gz)(x), lapse and a shift of either sign: the closed form of Eq. 30 is
    max_k (alpha / sqrt(gamma_kk) + |beta^k|) / dx^k.  Shared with the GPU parity test."""
    X, Y, Z = _grid(n, dx)
    m = np.zeros((16,) + shape)
    m[0] = 0.9 + 0.05 * np.sin(3 * X + Y)
    m[1] = 0.3 * np.cos(2 * X + Z); m[2] = -0.25 + 0.1 * np.sin(Y); m[3] = 0.2 * np.sin(X + 2 * Z)
    m[4] = 1.2 + 0.2 * np.sin(X); m[7] = 0.9 + 0.1 * np.cos(Y + Z); m[9] = 1.5 + 0.3 * np.sin(2 * Z)
    return m


def test_max_speed_with_shift_closed_form():
    n, dx = (9, 7, 6), (0.1, 0.2, 0.15)
    o = oracle.Oracle(dict(n=n, dx=dx, bc=(1, 1, 1), gamma_eos=2.0))
    m = shifted_diagonal_metric(o.shape, n, dx)
    o.set_metric(m)
    mi = interior(m, n)
    exp = max(np.max((mi[0] / np.sqrt(mi[g]) + np.abs(mi[1 + k])) / dx[k]) for k, g in enumerate((4, 7, 9)))
    assert o.max_speed() == pytest.approx(exp, rel=1e-14)
    # the shift term matters here, with either sign, and an inactive direction drops out
    m0 = m.copy(); m0[1:4] = 0
    o.set_metric(m0)
    assert o.max_speed() < exp * 0.95
    o1 = oracle.Oracle(dict(n=(9, 1, 1), dx=dx, bc=(1, 1, 1), gamma_eos=2.0))
    m1 = np.ascontiguousarray(m[:, 3:4, 3:4, :])
    o1.set_metric(m1)
    assert o1.max_speed() == pytest.approx(np.max((m1[0, 0, 0, 3:-3] / np.sqrt(m1[4, 0, 0, 3:-3]) +
                                                   np.abs(m1[1, 0, 0, 3:-3])) / dx[0]), rel=1e-14)


# ----------------------------------------------------------------------------------------------
# atmosphere rule (reading R9)
# ----------------------------------------------------------------------------------------------
def floor_hand_case():
    """Two uniform half-blocks moving with the same velocity in flat space, E = -v x B (no current): the left one
    at rho = rho_floor (1 + 5e-4) (below the threshold rho_floor (1 + 1e-3)), the right one at rho_floor (1 + 2e-3)
    (above).  Cells further than 6 cells from the jump and from the block ends see uniform stencils in both
    right-hand sides, so there the step is known by hand.  Returns (params, metric, prims, dt, expectation(nsteps))."""
    n, dx = (32, 1, 1), (0.1, 0.1, 0.1)
    Gam, rho_fl, K, sigma = 2.0, 1e-3, 50.0, 40.0
    par = dict(n=n, dx=dx, bc=(1, 1, 1), gamma_eos=Gam, sigma_model=0, sigma0=sigma, rho_floor=rho_fl, k_atmo=K)
    shape = (1, 1, 38)
    m = _flat_metric(shape)
    v, B = np.array([0.1, 0.2, -0.15]), np.array([0.02, -0.03, 0.05])
    E = -np.cross(v, B)
    p0 = K * rho_fl ** Gam * 3.0
    P = _uniform_prims(shape, rho_fl * (1 + 2e-3), p0, v, E, B, 0.0, 0.0, 0.0)
    P[0, 0, 0, :19] = rho_fl * (1 + 5e-4)
    dt = 0.02

    def expect(nsteps):
        """Floored cell after nsteps: each stage resets rho, v, p and sets E = E*^/(1 + a alpha sigma) with
        a = gamma dt (the closed form of Eq. 42 at v = 0); D, S_i, tau, B of the stage vector are untouched by the
        uniform right-hand side; the final recovery (a = 0) keeps calE^{n+1} and writes D, S_i, tau back."""
        X = E.copy()
        s = GAMMA * dt * sigma
        for _ in range(nsteps):
            E1 = X / (1 + s)
            Xs2 = X + dt * (1 - 2 * GAMMA) * (E1 - X) / (GAMMA * dt)              # Eq. 36, R11
            E2 = Xs2 / (1 + s)
            X = X + 0.5 * dt * ((E1 - X) + (E2 - Xs2)) / (GAMMA * dt)             # Eq. 37
        p_at = K * rho_fl ** Gam
        prim = np.concatenate([[rho_fl, p_at], np.zeros(3), X, B, np.zeros(3)])
        cons = np.concatenate([[rho_fl], np.cross(X, B), [p_at / (Gam - 1) + 0.5 * (X @ X + B @ B)], X, B, np.zeros(3)])
        return prim, cons

    return par, m, P, dt, expect, (slice(0, 12), slice(26, 32))


@pytest.mark.parametrize("nsteps", [1, 2])
def test_floor_rule_hand_case(nsteps):
    par, m, P, dt, expect, (lo, hi) = floor_hand_case()
    o = oracle.Oracle(par)
    o.set_metric(m); o.set_prims(P)
    for _ in range(nsteps):
        o.step(dt, wl.RECON_WENO5)
    Po, Uo = interior(o.get_prims(), par["n"])[:, 0, 0, :], interior(o.get_cons(), par["n"])[:, 0, 0, :]
    prim, cons = expect(nsteps)
    for f in range(14):
        assert np.allclose(Po[f, lo], prim[f], rtol=1e-13, atol=1e-18), (f, Po[f, lo], prim[f])
        assert np.allclose(Uo[f, lo], cons[f], rtol=1e-13, atol=1e-18), (f, Uo[f, lo], cons[f])
    # above the threshold: not reset; the uniform, current-free flow is steady
    Pi = interior(P, par["n"])[:, 0, 0, :]
    assert np.allclose(Po[:, hi], Pi[:, hi], rtol=1e-12, atol=1e-16)
    st = o.stats()
    assert st["c2p_failures"] == 0 and st["floor_resets"] >= 3 * nsteps * 12
    # with the floor disabled nothing is reset
    o2 = oracle.Oracle(dict(par, rho_floor=0.0))
    o2.set_metric(m); o2.set_prims(P)
    o2.step(dt, wl.RECON_WENO5)
    assert o2.stats()["floor_resets"] == 0
    assert np.allclose(interior(o2.get_prims(), par["n"])[:, 0, 0, lo], Pi[:, lo], rtol=1e-12, atol=1e-16)


# ----------------------------------------------------------------------------------------------
# face fix-ups (reading R4)
# ----------------------------------------------------------------------------------------------
def fixup_stencil_prims(n=24):
    """1D block on which the WENO5 face values of p and rho undershoot below zero: a deep one-cell minimum between
    high neighbours next to a drop of six decades (found by a random search over positive 5-cell stencils; TVD
    limiters never undershoot).  Shared with the GPU parity test."""
    shape = (1, 1, n + 6)
    P = _uniform_prims(shape, 1.0, 1.0, (0.05, 0.0, 0.0), (0, 0, 0), (0.0, 0.1, 0.0), 0, 0, 0)
    prof = np.ones(n + 6)
    prof[11:16] = [0.95, 0.5, 1e-4, 0.97, 1.3e-6]
    prof[16:] = 1.3e-6
    P[0, 0, 0] = prof
    P[1, 0, 0] = 2.0 * prof
    return P


def test_face_fixups_pressure_density_fallback_and_velocity_limiter():
    n = (24, 1, 1)
    par = dict(n=n, dx=(0.1, 0.1, 0.1), bc=(1, 1, 1), gamma_eos=5 / 3, sigma0=10.0)
    o = oracle.Oracle(par)
    P = fixup_stencil_prims()
    o.set_metric(_flat_metric(o.shape)); o.set_prims(P)
    row = P[1, 0, 0]
    lo_w, hi_w = oracle.recon_1d(row, wl.RECON_WENO5)          # the unlimited reconstruction (pinned elsewhere)
    neg = [c for c in range(3, 27) if lo_w[c] <= 0 or hi_w[c] <= 0]
    assert neg, "the stencil must drive WENO5 below zero somewhere"
    total = 0
    for i in range(0, 25):                                     # faces 0..24 (lower face of cell i)
        PL, PR, nf = o.face_states(wl.RECON_WENO5, 0, i)
        total += nf
        cL, cR = i + 2, i + 3                                  # padded indices of the left / right cell
        expL = hi_w[cL] if hi_w[cL] > 0 else row[cL]
        expR = lo_w[cR] if lo_w[cR] > 0 else row[cR]
        if 2 <= cL < 28:
            assert PL[1] == expL and PL[1] > 0
        if 2 <= cR < 28:
            assert PR[1] == expR and PR[1] > 0
        assert PL[0] > 0 and PR[0] > 0
    assert total >= len(neg)
    # the same count comes out of a right-hand side evaluation
    o.reset_stats()
    o.rhs(wl.RECON_WENO5)
    assert o.stats()["face_fixups"] == total
    # |v| limiter: a uniform flow with v^2 = 1 - 2e-12 > 1 - 1e-10 is rescaled to v^2 = 1 - 1e-10 at every face,
    # with the FACE metric (gamma_xx = 4 here: v^x = sqrt(1 - 1e-10)/2)
    o2 = oracle.Oracle(par)
    m = _flat_metric(o2.shape); m[4] = 4.0
    vx = (1 - 1e-12) / 2
    o2.set_metric(m); o2.set_prims(_uniform_prims(o2.shape, 1.0, 1.0, (vx, 0, 0), (0, 0, 0), (0, 0, 0), 0, 0, 0))
    PL, PR, nf = o2.face_states(wl.RECON_MC, 0, 5)
    assert nf == 2
    assert PL[2] == pytest.approx(math.sqrt(1 - 1e-10) / 2, rel=1e-15) and PR[2] == PL[2]
    assert 4 * PL[2] ** 2 <= 1 - 1e-10 + 1e-16
    # below the bound nothing is touched
    o2.set_prims(_uniform_prims(o2.shape, 1.0, 1.0, (0.4999, 0, 0), (0, 0, 0), (0, 0, 0), 0, 0, 0))
    PL, PR, nf = o2.face_states(wl.RECON_MC, 0, 5)
    assert nf == 0 and PL[2] == 0.4999


# ----------------------------------------------------------------------------------------------
# HLLE with a shift (Eq. 30, reading R6): clipping makes it pure upwinding once |beta| exceeds the light speed
# ----------------------------------------------------------------------------------------------
def superluminal_shift_problem(sign):
    """1D block, flat gamma, alpha = 1, uniform shift beta^x = sign * 1.5 (coordinates sweeping past the fluid faster
    than light): lambda+ = max(0, 1 - beta) and lambda- = min(0, -1 - beta), so one of them is clipped to zero and the
    HLLE flux is exactly the flux of the upwind state.  Piecewise-constant data, minmod (face states = cell values)."""
    n = (16, 1, 1)
    shape = (1, 1, 22)
    m = _flat_metric(shape)
    m[1] = sign * 1.5
    rng = np.random.default_rng(12)
    P = np.zeros((14,) + shape)
    for c0, c1 in ((0, 9), (9, 15), (15, 22)):                   # three constant states
        P[0, 0, 0, c0:c1] = rng.uniform(0.5, 1.5); P[1, 0, 0, c0:c1] = rng.uniform(0.5, 1.5)
        for f in range(2, 14):
            P[f, 0, 0, c0:c1] = rng.uniform(-0.3, 0.3)
    return n, m, P


@pytest.mark.parametrize("sign", [+1, -1])
def test_hlle_is_pure_upwinding_beyond_the_light_cone(sign):
    n, m, P = superluminal_shift_problem(sign)
    Gam, dx = 5 / 3, 0.1
    o = oracle.Oracle(dict(n=n, dx=(dx, dx, dx), bc=(1, 1, 1), gamma_eos=Gam, sigma0=0.0, kappa=0.0))
    o.set_metric(m); o.set_prims(P)
    F = interior(o.rhs(wl.RECON_MINMOD), n)[:, 0, 0, :]
    S = interior(o.sources(), n)[:, 0, 0, :]
    beta = np.array([sign * 1.5, 0, 0])
    flux = lambda c: oracle.state_flux_point(P[:, 0, 0, c], 0, Gam, 1.0, beta, None, 1, 0.0, 0.0)[1]
    for i in range(16):
        c = i + 3
        # beta > c: both face fluxes come from the cell on the right of each face; beta < -c: from the left
        exp = -(flux(c + 1) - flux(c)) / dx if sign > 0 else -(flux(c) - flux(c - 1)) / dx
        assert np.allclose(F[:, i] - S[:, i], exp, rtol=1e-13, atol=1e-13), (sign, i)
