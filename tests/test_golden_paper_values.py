"""Pins against the numbers the paper prints (tests/golden/paper_values.txt, each with its citation)."""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2510_18968_b200 import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, value, tol = [c.strip() for c in line.split("|")[:3]]
        out[name] = (float(value), float(tol))
    return out


def test_alfven_speed_worked_value():
    v, tol = _golden()["alfven_speed"]
    assert wl.alfven_speed(1.0, 1.0, 2.0, 1.1547, 1.0) == pytest.approx(v, rel=tol)


def test_tov_pressures_of_the_config5_recipe():
    """The analytic stand-in for the paper's TOV star uses its K, Gamma, rho_c: the central pressure and the
    4 % cut-off of the vector potential (Eq. 60) come out as the paper prints them."""
    g = _golden()
    w = wl.tov_like(n=16)
    e = w.extra
    p_c = e["K"] * e["rho_c"] ** 2
    assert p_c == pytest.approx(g["tov_p_max"][0], rel=g["tov_p_max"][1])
    assert 0.04 * p_c == pytest.approx(g["tov_p_cut"][0], rel=g["tov_p_cut"][1])


def test_imex_gamma_from_one_oracle_step():
    """Eq. 35: with zero explicit flux (uniform state, flat metric) the stage-1 electric field obeys
    (1 + gamma dt sigma) E1 = E^n for a fluid at rest without B, and the full step gives
    E^{n+1} = E^n + dt/2 (R1 + R2); solving that for gamma from the oracle's output returns 1 - 1/sqrt(2)."""
    v, tol = _golden()["imex_gamma"]
    n = (4, 4, 4)
    sigma, dt, E0 = 3.0, 0.05, 1e-3
    metric = np.zeros((16, 10, 10, 10)); metric[0] = 1.0; metric[[4, 7, 9]] = 1.0
    P = np.zeros((14, 10, 10, 10)); P[wl.RHO] = 1.0; P[wl.PRS] = 1.0; P[wl.EX] = E0
    o = oracle.Oracle(dict(n=n, dx=(0.25,) * 3, bc=(0, 0, 0), gamma_eos=2.0, sigma_model=0, sigma0=sigma, kappa=0.0))
    o.set_metric(metric); o.set_prims(P)
    o.step(dt, wl.RECON_MINMOD)
    E1 = float(o.get_prims()[wl.EX, 5, 5, 5])
    # fluid at rest (E^2 back-reaction on v is O(E0^2) with B = 0: none), so per stage E_i = E*_i / (1 + g dt sigma):
    #   E1 = E0/(1+a), X*2 = E0 + (1-2g)/g (E1 - E0), E2 = X*2/(1+a), E^{n+1} = E0 + (E1 - E0 + E2 - X*2)/(2g), a = g dt sigma
    def final(g):
        a = g * dt * sigma
        e1 = E0 / (1 + a); xs2 = E0 + (1 - 2 * g) / g * (e1 - E0); e2 = xs2 / (1 + a)
        return E0 + (e1 - E0 + e2 - xs2) / (2 * g)
    lo, hi = 0.2, 0.45                                  # final(g) is monotone there; bisection for the oracle's gamma
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if (final(mid) - E1) * (final(lo) - E1) <= 0:
            hi = mid
        else:
            lo = mid
    assert abs(final(v) - E1) <= 1e-15 * E0
    assert 0.5 * (lo + hi) == pytest.approx(v, rel=1e-6)
