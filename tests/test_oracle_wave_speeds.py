"""Pins of the state-dependent HLLE wave speeds ("the characteristic speed
... used in ideal GRMHD inside the star, while outside it is fixed to the speed of light"; reading R16)
against textbook closed forms.  CPU only."""
import math

import numpy as np
import pytest

import oracle
from helpers import g6_from_matrix, interior, random_spd
from paper_2510_18968_b200 import workloads as wl


def _P(rho, p, v=(0, 0, 0), B=(0, 0, 0)):
    P = np.zeros(14)
    P[0], P[1] = rho, p
    P[2:5] = v; P[8:11] = B
    return P


def test_sound_speed_and_fast_speed_at_rest():
    """Flat space, fluid at rest.  B = 0: lambda = +-cs with cs^2 = Gamma p/h (Eq. 50, reading G3).  B perpendicular to
    the direction: the exact fast speed sqrt(cs^2 + vA^2 - cs^2 vA^2), vA^2 = B^2/(h + B^2).  B along the direction: the
    bound is an UPPER bound of the exact fast speed max(cs, vA)."""
    Gam, rho, p = 5 / 3, 1.3, 0.7
    h = rho + Gam / (Gam - 1) * p
    cs = math.sqrt(Gam * p / h)
    for k in range(3):
        lm, lp = oracle.wave_speeds_point(_P(rho, p), k, Gam)
        assert lp == pytest.approx(cs, rel=1e-15) and lm == pytest.approx(-cs, rel=1e-15)
    B = 1.1
    vA2 = B * B / (h + B * B)
    fast = math.sqrt(cs * cs + vA2 - cs * cs * vA2)
    lm, lp = oracle.wave_speeds_point(_P(rho, p, B=(0, B, 0)), 0, Gam)
    assert lp == pytest.approx(fast, rel=1e-14) and lm == pytest.approx(-fast, rel=1e-14)
    lm, lp = oracle.wave_speeds_point(_P(rho, p, B=(B, 0, 0)), 0, Gam)
    assert lp >= max(cs, math.sqrt(vA2)) and lp < 1.0


def test_relativistic_velocity_addition_and_metric_factors():
    """Unmagnetised flow along the direction: lambda = (V +- cs)/(1 +- V cs) (velocity addition), where V is the
    PHYSICAL speed.  On a diagonal metric gamma_xx = a^2 with lapse and shift the coordinate speed is
    alpha lambda / a - beta^x."""
    Gam, rho, p = 4 / 3, 0.9, 1.5
    cs = math.sqrt(Gam * p / (rho + Gam / (Gam - 1) * p))
    for V in (-0.6, 0.0, 0.3, 0.9):
        lm, lp = oracle.wave_speeds_point(_P(rho, p, v=(V, 0, 0)), 0, Gam)
        assert lp == pytest.approx((V + cs) / (1 + V * cs), rel=1e-13, abs=1e-15)
        assert lm == pytest.approx((V - cs) / (1 - V * cs), rel=1e-13, abs=1e-15)
        a, alpha, beta = 1.7, 0.8, 0.15
        g6 = np.array([a * a, 0, 0, 1.0, 0, 1.0])
        lm, lp = oracle.wave_speeds_point(_P(rho, p, v=(V / a, 0, 0)), 0, Gam, alpha, np.array([beta, 0, 0]), g6)
        assert lp == pytest.approx(alpha * (V + cs) / (1 + V * cs) / a - beta, rel=1e-13, abs=1e-15)
        assert lm == pytest.approx(alpha * (V - cs) / (1 - V * cs) / a - beta, rel=1e-13, abs=1e-15)
    # transverse flow slows the wave down: Lorentz contraction of the sound cone, lambda = +-cs sqrt((1-V^2)/(1-V^2 cs^2))
    V = 0.5
    lm, lp = oracle.wave_speeds_point(_P(rho, p, v=(0, V, 0)), 0, Gam)
    assert lp == pytest.approx(cs * math.sqrt((1 - V * V) / (1 - V * V * cs * cs)), rel=1e-13) and lm == -lp


def test_speeds_stay_inside_the_light_cone_on_random_states():
    rng = np.random.default_rng(9)
    for t in range(2000):
        g = random_spd(rng) if t % 2 else np.eye(3)
        gi = np.linalg.inv(g)
        unit = lambda d: d / math.sqrt(d @ g @ d)
        Gam = rng.choice([4 / 3, 5 / 3, 2.0])
        rho = 10 ** rng.uniform(-4, 1); p = rho * 10 ** rng.uniform(-3, 2)
        v = unit(rng.standard_normal(3)) * rng.uniform(0, 0.99)
        B = unit(rng.standard_normal(3)) * math.sqrt(10 ** rng.uniform(-3, 3) * rho)
        alpha, beta = rng.uniform(0.3, 1.0), 0.3 * rng.standard_normal(3)
        for k in range(3):
            lm, lp = oracle.wave_speeds_point(_P(rho, p, v, B), k, Gam, alpha, beta, g6_from_matrix(g))
            c = alpha * math.sqrt(gi[k, k])
            assert -c - beta[k] - 1e-12 <= lm <= lp <= c - beta[k] + 1e-12
            # the flow itself lies between the two characteristics
            assert lm - 1e-12 <= alpha * v[k] - beta[k] <= lp + 1e-12


def test_mode_switch_reduces_to_eq30_and_is_live_inside():
    """wave_speed_mode MHD_INSIDE with a switch density no state exceeds is bit-identical to Eq. 30; with every state
    inside, HLLE is less diffusive (a smooth sound wave is damped less) and the CFL speed drops below light."""
    w = wl.alfven1d(n=64, sigma0=1e4, recon=wl.RECON_MINMOD)
    f = w.fields()
    outs = {}
    for name, over in (("light", dict()), ("off", dict(wave_speed_mode=1, wave_rho_switch=1e30)),
                       ("inside", dict(wave_speed_mode=1, wave_rho_switch=0.0))):
        o = oracle.from_workload(w, fields=f, **over)
        ms = o.max_speed()
        for _ in range(40):
            o.step(w.dt, w.recon)
        outs[name] = (o.get_prims(), ms, o.max_speed(), o.stats()["c2p_failures"])
    assert np.array_equal(outs["light"][0], outs["off"][0]) and outs["light"][1] == outs["off"][1]
    assert outs["inside"][3] == 0 and np.isfinite(outs["inside"][0]).all()
    assert outs["inside"][1] < 0.95 * outs["light"][1]                 # per-cell MHD speeds < c
    assert outs["light"][1] == pytest.approx(1.0 / w.dx[0], rel=1e-15)
    # less numerical diffusion: the wave keeps more of its amplitude
    amp = lambda P: float(np.abs(P[wl.BY]).max())
    assert amp(outs["inside"][0]) > amp(outs["light"][0])
    # conservation is untouched by the choice of speeds (periodic, flat)
    U0 = interior(oracle.from_workload(w, fields=f).get_cons(), w.n).sum(axis=(1, 2, 3))
    o = oracle.from_workload(w, fields=f, wave_speed_mode=1, wave_rho_switch=0.0)
    for _ in range(10):
        o.step(w.dt, w.recon)
    U1 = interior(o.get_cons(), w.n).sum(axis=(1, 2, 3))
    for i in (0, 1, 2, 3, 4, 8, 9, 10):
        assert abs(U1[i] - U0[i]) <= 1e-12 * max(abs(U0[0]), abs(U0[4]))


def test_config5_speeds_inside_the_star_are_subluminal():
    """cfg5 sub-block at the centre of the star with the switch at 10 rho_atmo: every cell is inside, the CFL speed is
    the local fast speed (<< c at rho_c = 1.28e-3); a block in the atmosphere keeps the light speed."""
    w = wl.tov_like()
    n, bc = (12, 12, 12), (wl.BC_OUTFLOW,) * 3
    over = dict(wave_speed_mode=1, wave_rho_switch=1e-9)
    oc = oracle.from_workload(w, fields=w.fields((250, 250, 250), n), n=n, bc=bc, **over)
    oa = oracle.from_workload(w, fields=w.fields((2, 2, 2), n), n=n, bc=bc, **over)
    ol = oracle.from_workload(w, fields=w.fields((250, 250, 250), n), n=n, bc=bc)
    assert oc.max_speed() < 0.6 * ol.max_speed()
    assert oa.max_speed() * w.dx[0] == pytest.approx(1.0, rel=0.1)     # alpha / psi^2 ~ 0.94 / 1.12 out there
    oc.step(w.dt, w.recon)
    assert oc.stats()["c2p_failures"] == 0 and np.isfinite(oc.get_prims()).all()
