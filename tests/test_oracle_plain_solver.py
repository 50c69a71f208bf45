"""Pins of the oracle's PLAIN root solver (c2p_plain: bisection on Z inside an un-accelerated fixed point on
(W, kE)) -- the solver every parity run uses -- against what the mathematics fixes, and of the conventions
around the root (no-bracket fallback, conductivity models).  CPU only.

* manufactured solutions: primitives are chosen first, the stage vector whose root they are is built in
  NumPy (Eq. 42 solved for E*, Eq. 22-24 for D, S_i, tau), so the expected root owes nothing to the oracle;
* c2p_plain vs c2p_robust (bracketed secant + Anderson; a different iteration on the same system);
* the representative states of BASELINE configs 4 (ambient, B^2/Z ~ 45) and 5 (atmosphere, interior)."""
import math

import numpy as np
import pytest

import oracle
from helpers import LEVI, g6_from_matrix, random_spd
from paper_2510_18968_b200 import workloads as wl
from test_oracle_pointwise import _manufactured_implicit

FLAT = np.array([1.0, 0, 0, 1.0, 0, 1.0])


def _scales(P, g):
    vs = max(math.sqrt(P[2:5] @ g @ P[2:5]), 1e-3)
    Bs = math.sqrt(P[8:11] @ g @ P[8:11])
    return np.array([P[0], P[1], vs, vs, vs] + [max(Bs, 1e-300)] * 6 + [1, 1, 1]), Bs


def test_plain_vs_robust_vs_manufactured_root_12000_states():
    """>= 1e4 states, |v| <= 0.6, magnetisation B^2/h from 0.01 to 100 (config 4's ambient medium sits at 45),
    sigma in {0} U [1, 1e8], flat and random SPD metrics.  The pressure is the ill-conditioned unknown
    (p = a difference of terms of size tau + B^2): the achievable accuracy is eps * magnetisation * h/p, hence
    the looser bound in the last decade of magnetisation (measured: 1.3e-12 there, 1.6e-13 below)."""
    rng = np.random.default_rng(2025)
    worst_lo = worst_hi = worst_pr = 0.0
    evs = []
    for t in range(12000):
        g = random_spd(rng) if t % 2 else np.eye(3)
        g6 = g6_from_matrix(g)
        P, U, Gam, adt, sigma, alpha = _manufactured_implicit(rng, g, 0.6, 2.0)
        if t % 6 == 0:                                   # sigma = 0: E = E*, one outer pass
            sigma = 0.0
            U = oracle.prim2cons_point(P, Gam, alpha, None, g6)
        guess = P.copy(); guess[0] *= 1.05; guess[1] *= 0.95; guess[2:5] *= 0.9
        Pp, evp, fp = oracle.c2p_point(U, guess, Gam, adt, sigma, alpha, g6, plain=True)
        Pr, evr, fr = oracle.c2p_point(U, guess, Gam, adt, sigma, alpha, g6)
        assert not fp and not fr, (t, fp, fr)
        scale, Bs = _scales(P, g)
        mag = Bs ** 2 / (P[0] + Gam / (Gam - 1) * P[1])
        e = np.max(np.abs(Pp - P) / scale)
        if mag < 10:
            worst_lo = max(worst_lo, e)
        else:
            worst_hi = max(worst_hi, e)
        worst_pr = max(worst_pr, np.max(np.abs(Pp - Pr) / scale))
        evs.append(evp)
        if t % 50 == 0:
            # the defining system evaluated here, independently of the oracle (SURVEY pin <= 1e-13)
            sg = math.sqrt(np.linalg.det(g))
            v, E, B = Pp[2:5], Pp[5:8], Pp[8:11]
            vD = g @ v; W = 1 / math.sqrt(1 - v @ vD); s = adt * alpha * sigma * W
            vxB = np.einsum("ijk,j,k->i", LEVI, vD, g @ B) / sg
            ohm = (1 + s) * E - s * (vD @ E) * v + s * vxB - U[5:8] / sg
            assert np.max(np.abs(ohm)) < 1e-13 * (1 + s) * Bs
            U2 = oracle.prim2cons_point(Pp, Gam, alpha, None, g6)
            ref = abs(U[4]) + abs(U[0])
            assert np.max(np.abs(U2[:5] - U[:5])) < 1e-13 * ref
    assert worst_lo < 1e-12 and worst_hi < 5e-12 and worst_pr < 1e-12, (worst_lo, worst_hi, worst_pr)
    # bisection from the full bracket: ~55 evaluations per outer pass, a handful of passes
    assert 50 <= np.median(evs) <= 400 and max(evs) < 20000, (np.median(evs), max(evs))


def test_plain_roundtrip_fixed_E():
    """a = 0 (final recovery of a step): prim -> cons -> prim to 1e-12 with the plain solver."""
    rng = np.random.default_rng(77)
    worst = 0.0
    for t in range(1500):
        g = random_spd(rng) if t % 2 else np.eye(3)
        g6 = g6_from_matrix(g)
        P, U, Gam, adt, sigma, alpha = _manufactured_implicit(rng, g, 0.7, 1.0)
        U = oracle.prim2cons_point(P, Gam, alpha, None, g6)
        guess = P.copy(); guess[0] *= 1.3; guess[1] *= 0.7; guess[2:5] *= 0.5
        P2, ev, failed = oracle.c2p_point(U, guess, Gam, 0.0, 0.0, alpha, g6, plain=True)
        assert not failed and ev <= 70                   # one bisection
        scale, _ = _scales(P, g)
        worst = max(worst, np.max(np.abs(P2 - P) / scale))
    assert worst < 1e-12, worst


def _state(rho, p, v, B, Gam):
    P = np.zeros(14)
    P[0], P[1] = rho, p
    P[2:5] = v; P[8:11] = B
    P[5:8] = -np.cross(P[2:5], P[8:11])
    return P


@pytest.mark.parametrize("name,rho,p,B,Gam,adt", [
    ("cfg4 ambient", 1e-4, 3e-5, (0.1, 0.0, 0.0), 4 / 3, 0.29 * 0.25 / 256),        # B^2/h = 45
    ("cfg4 cylinder", 1e-2, 1.0, (0.1, 0.0, 0.0), 4 / 3, 0.29 * 0.25 / 256),
    ("cfg5 atmosphere", 1e-10, 100 * 1e-20, (1e-9, 0.0, 2e-9), 2.0, 0.29 * 0.125 * 24 / 512),
    ("cfg5 centre", 1.28e-3, 100 * 1.28e-3 ** 2, (0.0, 1e-6, 3.58e-6), 2.0, 0.29 * 0.125 * 24 / 512),
    ("cfg1 right state", 0.125, 0.1, (0.5, -1.0, 0.0), 2.0, 0.29e-3),               # B^2/h = 3.8
])
def test_plain_on_config_states(name, rho, p, B, Gam, adt):
    """Representative states of the BASELINE configs, moving, over the conductivity range of the configs; the stage
    vector is manufactured in NumPy (flat metric: cross products are np.cross)."""
    rng = np.random.default_rng(3)
    for sigma in (0.0, 1.0, 1e3, 1e6, 1e8):
        for _ in range(20):
            v = rng.standard_normal(3); v *= rng.uniform(0.0, 0.3) / np.linalg.norm(v)
            P = _state(rho, p, v, np.array(B), Gam)
            P[5:8] += 1e-2 * np.linalg.norm(B) * rng.standard_normal(3) * min(1.0, 100 / max(sigma, 1e-300))
            W = 1 / math.sqrt(1 - v @ v); s = adt * sigma * W
            E = P[5:8]
            Estar = (1 + s) * E - s * (v @ E) * v + s * np.cross(v, P[8:11])
            U = oracle.prim2cons_point(P, Gam)
            U[5:8] = Estar
            guess = P.copy(); guess[0] *= 1.2; guess[1] *= 0.8; guess[2:5] *= 0.7
            Pp, ev, fp = oracle.c2p_point(U, guess, Gam, adt, sigma, plain=True)
            Pr, er, fr = oracle.c2p_point(U, guess, Gam, adt, sigma)
            assert not fp and not fr, (name, sigma)
            scale, Bs = _scales(P, np.eye(3))
            # p = (Gamma-1)/Gamma (Z/W^2 - rho) is a difference of quantities of size h: absolute accuracy eps * h
            # (config 5's cold atmosphere has p/rho = 1e-8)
            scale[1] = max(p, 1e-3 * (rho + Gam / (Gam - 1) * p))
            mag = Bs ** 2 / (rho + Gam / (Gam - 1) * p)
            tol = 1e-12 * max(1.0, mag / 10)
            assert np.max(np.abs(Pp - P) / scale) < tol, (name, sigma, np.abs(Pp - P) / scale)
            assert np.max(np.abs(Pp - Pr) / scale) < tol, (name, sigma)


@pytest.mark.parametrize("plain", [True, False])
def test_no_bracket_fallback(plain):
    """D^ <= 0 or an empty bracket (tau^ + D^ <= B^2/2 + D^/Gamma) is a FAILURE; rho, p, v keep the
    guess and E is the closed form of Eq. 42 at the guess velocity -- typed out here in NumPy."""
    P = _state(1.0, 0.5, (0.2, -0.1, 0.05), np.array((0.3, 0.4, -0.2)), 5 / 3)
    U = oracle.prim2cons_point(P, 5 / 3)
    adt, sigma = 1e-3, 500.0
    guess = P.copy(); guess[0] = 0.9; guess[1] = 0.45; guess[2:5] = (0.15, -0.12, 0.02)
    for bad in ("D", "bracket"):
        Ub = U.copy()
        if bad == "D":
            Ub[0] = -1e-3
        else:
            Ub[4] = 0.5 * (P[8:11] @ P[8:11]) - 0.9 * Ub[0]        # Gamma (tau + D - B^2/2) < D
        Pf, ev, failed = oracle.c2p_point(Ub, guess, 5 / 3, adt, sigma, plain=plain)
        assert failed
        assert np.array_equal(Pf[0:5], guess[0:5])
        v = guess[2:5]; W = 1 / math.sqrt(1 - v @ v); s = adt * sigma * W
        Es, B = Ub[5:8], Ub[8:11]
        kE = (v @ Es) / (1 + s / W ** 2)
        E = (Es - s * np.cross(v, B) + s * kE * v) / (1 + s)
        assert np.allclose(Pf[5:8], E, rtol=1e-14, atol=1e-16)
        assert np.array_equal(Pf[8:14], Ub[8:14])                  # B, psi, phi, q = cons / sqrt(gamma)


def test_sigma_models_hand_values():
    """A18: Eq. 52 sigma = sigma0 D^gamma [reading R13: (D^/D_ref)^e, integer e] and Eq. 61
     sigma = sigma0 max(1 - D_atmo/D, 0)^2, hand-typed values."""
    U, A, PD, AT = wl.SIGMA_UNIFORM, wl.SIGMA_ARRAY, wl.SIGMA_POWER_D, wl.SIGMA_ATMO
    assert oracle.sigma_point(U, 7.5, 3, 2.0, 0.3, 99.0) == 7.5
    assert oracle.sigma_point(A, 7.5, 3, 2.0, 0.3, 99.0) == 99.0
    # Eq. 52: exponents 0, 2, 6 at D = 0.5, 2, 3 (D_ref = 1 in the paper) and with a reference density
    assert oracle.sigma_point(PD, 1e6, 0, 1.0, 0.5) == 1e6
    assert oracle.sigma_point(PD, 1e6, 2, 1.0, 0.5) == 2.5e5
    assert oracle.sigma_point(PD, 1e6, 6, 1.0, 0.5) == 1e6 / 64
    assert oracle.sigma_point(PD, 10.0, 6, 1.0, 2.0) == 640.0
    assert oracle.sigma_point(PD, 10.0, 2, 1.0, 3.0) == 90.0
    assert oracle.sigma_point(PD, 1e8, 2, 1.28e-3, 6.4e-4) == pytest.approx(2.5e7, rel=1e-15)     # config 5: (D/rho_c)^2
    assert oracle.sigma_point(PD, 10.0, 9, 1.0, 2.0) == 5120.0 and oracle.sigma_point(PD, 10.0, 12, 1.0, 2.0) == 40960.0
    # Eq. 61 at D = D_atmo/2, D_atmo, 2 D_atmo, 10 D_atmo: 0, 0, sigma0/4, 0.81 sigma0
    Da = 1e-10
    assert oracle.sigma_point(AT, 1e6, 0, Da, 0.5 * Da) == 0.0
    assert oracle.sigma_point(AT, 1e6, 0, Da, Da) == 0.0
    assert oracle.sigma_point(AT, 1e6, 0, Da, 2 * Da) == 2.5e5
    assert oracle.sigma_point(AT, 1e6, 0, Da, 10 * Da) == pytest.approx(8.1e5, rel=1e-15)
    assert oracle.sigma_point(AT, 1e6, 0, Da, 1.0) == pytest.approx(1e6, rel=1e-9)               # deep interior
