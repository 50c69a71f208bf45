"""GPU parity tests (-m gpu) for the code paths round 1 left unreached: the conductivity models ATMO (Eq. 61) and
POWER_D with exponents other than 2 (Eq. 52; the paper's own shocktube E2), the 2D explosion E3, the atmosphere rule
(reading R9) against hand-typed values through both recovery routes, max speed with a shift, and the face fix-ups
(reading R4).  Everything goes through the C-ABI binding; expected values come from the oracle or from closed forms."""
import math

import numpy as np
import pytest

import oracle
from helpers import cons_group_scales, interior, prim_group_scales, rel_linf
from paper_2510_18968_b200 import workloads as wl
from test_oracle_closed_forms import fixup_stencil_prims, floor_hand_case, shifted_diagonal_metric

pytestmark = pytest.mark.gpu

TOL1, TOL20 = 1e-11, 1e-9


@pytest.fixture(scope="module")
def binding():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2510_18968_b200 import binding as b
    b.load()
    return b


def _compare(g, o, n, dx_min, tol, what=""):
    Pg, Po = interior(g.get_prims(), n), interior(o.get_prims(), n)
    Ug, Uo = interior(g.get_cons(), n), interior(o.get_cons(), n)
    assert np.isfinite(Pg).all() and np.isfinite(Ug).all(), what
    eP = rel_linf(Pg, Po, prim_group_scales(Po, dx_min))
    eU = rel_linf(Ug, Uo, cons_group_scales(Uo, dx_min))
    assert eP.max() <= tol and eU.max() <= tol, (what, eP, eU)
    return max(eP.max(), eU.max())


def _both(binding, par, metric, prims, variant=0, omp=True):
    o = oracle.Oracle(par, omp=omp)
    g = binding.Rgrmhd(par)
    g.set_rhs_variant(variant)
    for h in (o, g):
        h.set_metric(metric); h.set_prims(prims)
    return g, o


# ----------------------------------------------------------------------------------------------
# conductivity models
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gamma_exp", [6, 12])
def test_e2_shocktube_power_law_conductivity(binding, gamma_exp):
    """The paper's E2: sigma = 1e6 D^gamma, 400 cells, minmod; sigma spans ~12 decades."""
    w = wl.shocktube_paper(gamma_exp=gamma_exp)
    f = w.fields()
    g = binding.from_workload(w, fields=f)
    o = oracle.from_workload(w, fields=f)
    for s in range(20):
        g.step(w.dt, w.recon); o.step(w.dt, w.recon)
        if s == 0:
            _compare(g, o, w.n, w.dx[0], TOL1, "e2 step 1")
    _compare(g, o, w.n, w.dx[0], TOL20, "e2 step 20")
    assert g.stats()["c2p_failures"] == 0 and o.stats()["c2p_failures"] == 0


def test_e2_shocktube_to_t04(binding):
    """E2 with gamma = 6 in full: 640 steps to t = 0.4 (bound: the 20-step one scaled linearly, as for config 1)."""
    w = wl.shocktube_paper(gamma_exp=6)
    f = w.fields()
    g = binding.from_workload(w, fields=f)
    o = oracle.from_workload(w, fields=f)
    for _ in range(w.nsteps):
        g.step(w.dt, w.recon); o.step(w.dt, w.recon)
    _compare(g, o, w.n, w.dx[0], (w.nsteps / 20) * TOL20, "e2 t=0.4")
    # the conductivity really is non-uniform: sigma0 D^6 spans many decades across the tube
    D = interior(g.get_cons(), w.n)[0]
    assert (D.max() / D.min()) ** 6 > 1e4


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_sigma_atmo_model_tov_subblock(binding, variant):
    """Eq. 61: sigma = sigma0 max(1 - D_atmo/D, 0)^2 on a block across the stellar surface of the
    config-5 star: zero conductivity in the atmosphere, sigma0 inside."""
    w = wl.tov_like()
    i_surf = int(round((8.125 + 12.0) / w.dx[0]))
    n, bc = (40, 12, 10), (wl.BC_OUTFLOW,) * 3
    f = w.fields((i_surf - 20, 256 - 6, 256 - 5), n)
    over = dict(sigma_model=wl.SIGMA_ATMO, sigma0=1e6, sigma_dref=1e-10)
    o = oracle.from_workload(w, fields=f, omp=True, n=n, bc=bc, **over)
    g = binding.from_workload(w, fields=f, n=n, bc=bc, **over)
    g.set_rhs_variant(variant)
    for s in range(10):
        g.step(w.dt, w.recon); o.step(w.dt, w.recon)
        if s == 0:
            _compare(g, o, n, w.dx[0], TOL1, "atmo step 1")
    _compare(g, o, n, w.dx[0], TOL20, "atmo step 10")
    sg, so = g.stats(), o.stats()
    assert sg["floor_resets"] == so["floor_resets"] > 0 and sg["c2p_failures"] == so["c2p_failures"] == 0


def test_sigma_atmo_model_face_ohm(binding):
    """The same model through charge mode A, where the flux kernel itself evaluates sigma(D) of the two cells."""
    rng = np.random.default_rng(5)
    from test_oracle_scheme import _pad_periodic, _periodic_problem
    n = (20, 10, 8)
    metric, P = _periodic_problem(24, rng, True)
    sl = (slice(None), slice(0, n[2]), slice(0, n[1]), slice(0, n[0]))
    metric, P = _pad_periodic(np.ascontiguousarray(metric[sl])), _pad_periodic(np.ascontiguousarray(P[sl]))
    for model, extra in ((wl.SIGMA_ATMO, dict(sigma0=40.0, sigma_dref=0.95)),
                         (wl.SIGMA_POWER_D, dict(sigma0=25.0, sigma_exp=3.0, sigma_dref=1.1))):
        par = dict(n=n, dx=(1 / 24,) * 3, bc=(0, 0, 0), gamma_eos=5 / 3, sigma_model=model, kappa=1.0,
                   charge_mode=wl.CHARGE_FACE_OHM, **extra)
        for variant in (0, 1):
            g, o = _both(binding, par, metric, P, variant)
            for _ in range(3):
                g.step(0.2 / 24, wl.RECON_MC); o.step(0.2 / 24, wl.RECON_MC)
            _compare(g, o, n, 1 / 24, TOL20, "face-ohm sigma model %d" % model)


# ----------------------------------------------------------------------------------------------
# E3: the paper's 2D cylindrical explosion
# ----------------------------------------------------------------------------------------------
def test_e3_explosion2d_full_200x200(binding):
    w = wl.explosion2d()
    f = w.fields()
    g = binding.from_workload(w, fields=f)
    o = oracle.from_workload(w, fields=f, omp=True)
    for s in range(20):
        g.step(w.dt, w.recon); o.step(w.dt, w.recon)
        if s == 0:
            _compare(g, o, w.n, w.dx[0], TOL1, "e3 step 1")
    _compare(g, o, w.n, w.dx[0], TOL20, "e3 step 20")
    assert g.stats()["c2p_failures"] == 0


# ----------------------------------------------------------------------------------------------
# atmosphere rule against hand-typed values, both recovery routes
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("route", ["flushed", "fused"])
def test_floor_rule_hand_case_gpu(binding, route):
    """tests/test_oracle_closed_forms.floor_hand_case: the expected primitives AND the written-back D, S_i, tau are
    typed by hand there.  'flushed' runs the final recovery as its own launch (k_c2p<3>) after every step, 'fused'
    lets the next step's first launch do it (k_c2p<4>)."""
    par, m, P, dt, expect, (lo, hi) = floor_hand_case()
    g = binding.Rgrmhd(par)
    g.set_metric(m); g.set_prims(P)
    for nsteps in (1, 2):
        g.step(dt, wl.RECON_WENO5)
        if route == "flushed" or nsteps == 2:
            g.flush()
        if route == "fused" and nsteps == 1:
            continue                                            # keep the recovery pending: step 2 fuses it
        Pg = interior(g.get_prims(), par["n"])[:, 0, 0, :]
        Ug = interior(g.get_cons(), par["n"])[:, 0, 0, :]
        prim, cons = expect(nsteps)
        for f in range(14):
            assert np.allclose(Pg[f, lo], prim[f], rtol=1e-13, atol=1e-18), (route, nsteps, f, Pg[f, lo], prim[f])
            assert np.allclose(Ug[f, lo], cons[f], rtol=1e-13, atol=1e-18), (route, nsteps, f, Ug[f, lo], cons[f])
        Pi = interior(P, par["n"])[:, 0, 0, :]
        assert np.allclose(Pg[:, hi], Pi[:, hi], rtol=1e-12, atol=1e-16)       # above the threshold: untouched
    st = g.stats()
    assert st["c2p_failures"] == 0 and st["floor_resets"] >= 3 * 2 * 12


# ----------------------------------------------------------------------------------------------
# a7 with a shift
# ----------------------------------------------------------------------------------------------
def test_max_speed_with_shift_gpu(binding):
    n, dx = (37, 21, 9), (0.1, 0.2, 0.15)
    par = dict(n=n, dx=dx, bc=(1, 1, 1), gamma_eos=2.0)
    g = binding.Rgrmhd(par)
    m = shifted_diagonal_metric(g.shape, n, dx)
    g.set_metric(m)
    mi = interior(m, n)
    exp = max(np.max((mi[0] / np.sqrt(mi[q]) + np.abs(mi[1 + k])) / dx[k]) for k, q in enumerate((4, 7, 9)))
    o = oracle.Oracle(par)
    o.set_metric(m)
    assert g.max_speed() == pytest.approx(exp, rel=1e-14)
    assert abs(g.max_speed() - o.max_speed()) <= 1e-15 * exp
    m0 = m.copy(); m0[1:4] = 0
    g.set_metric(m0)
    assert g.max_speed() < 0.95 * exp                              # the |beta^k| term is live


# ----------------------------------------------------------------------------------------------
# face fix-ups
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_face_fixup_stencil(binding, variant):
    """A profile on which WENO5 undershoots below zero in rho and p (tests/test_oracle_closed_forms pins the oracle's
    fallback values): 1D, and replicated along y and z so that the tiled kernels and their halo warps take the same
    decision; a wrong or missing fallback changes the fluxes at O(1)."""
    P1 = fixup_stencil_prims()
    for n in ((24, 1, 1), (24, 18, 6)):
        shape = tuple(m + 6 if m > 1 else 1 for m in (n[2], n[1], n[0]))
        P = np.ascontiguousarray(np.broadcast_to(P1, (14,) + shape[:2] + (30,)))
        m = np.zeros((16,) + shape); m[0] = 1.0; m[4] = m[7] = m[9] = 1.0
        par = dict(n=n, dx=(0.1, 0.1, 0.1), bc=(1, 1, 1), gamma_eos=5 / 3, sigma0=10.0)
        g, o = _both(binding, par, m, P, variant)
        dt = 0.02
        g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)
        assert o.stats()["face_fixups"] > 0
        _compare(g, o, n, 0.1, TOL1, "fix-up stencil n=%s" % (n,))
        for _ in range(4):
            g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)
        _compare(g, o, n, 0.1, TOL20, "fix-up stencil 5 steps n=%s" % (n,))


# ----------------------------------------------------------------------------------------------
# charge mode C: q = nabla_i E^i
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_charge_mode_div_e(binding, variant):
    """Curved periodic block (shift, K_ij, off-diagonal metric), a config-4 sub-block with outflow walls, and a 1D
    block: the charge of every stage and of the new state comes from the centred divergence of calE."""
    from test_oracle_scheme import _pad_periodic, _periodic_problem
    rng = np.random.default_rng(17)
    n = (38, 21, 9)
    metric, P = _periodic_problem(40, rng, True)
    sl = (slice(None), slice(0, n[2]), slice(0, n[1]), slice(0, n[0]))
    metric, P = _pad_periodic(np.ascontiguousarray(metric[sl])), _pad_periodic(np.ascontiguousarray(P[sl]))
    par = dict(n=n, dx=(1 / 40,) * 3, bc=(0, 0, 0), gamma_eos=5 / 3, sigma_model=0, sigma0=30.0, kappa=1.0,
               charge_mode=wl.CHARGE_DIV_E)
    g, o = _both(binding, par, metric, P, variant)
    dt = 0.2 / 40
    g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)
    _compare(g, o, n, 1 / 40, TOL1, "div E 1 step")
    for s in range(4):
        g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)
        if s == 1:
            g.stats()                        # flushes the pending recovery mid-run: the charge is still due on output
    _compare(g, o, n, 1 / 40, TOL20, "div E 5 steps")
    w = wl.blast_curved()
    nb, bc = (40, 36, 20), (wl.BC_OUTFLOW,) * 3
    f = w.fields((120, 138, 100), nb)
    o = oracle.from_workload(w, fields=f, omp=True, n=nb, bc=bc, charge_mode=wl.CHARGE_DIV_E)
    g = binding.from_workload(w, fields=f, n=nb, bc=bc, charge_mode=wl.CHARGE_DIV_E)
    g.set_rhs_variant(variant)
    for _ in range(20):
        g.step(w.dt, w.recon); o.step(w.dt, w.recon)
    _compare(g, o, nb, w.dx[0], TOL20, "div E cfg4 block 20 steps")
    assert g.stats()["c2p_failures"] == 0
    w1 = wl.shocktube(n=64, sigma0=1e3)
    f1 = w1.fields()
    f1["prims"][wl.BZ] = 0.3                                     # non-coplanar: the charge sector is live
    o = oracle.from_workload(w1, fields=f1, charge_mode=wl.CHARGE_DIV_E)
    g = binding.from_workload(w1, fields=f1, charge_mode=wl.CHARGE_DIV_E)
    for _ in range(10):
        g.step(w1.dt, wl.RECON_MC); o.step(w1.dt, wl.RECON_MC)
    _compare(g, o, w1.n, w1.dx[0], TOL20, "div E 1D")
    assert np.abs(interior(g.get_prims(), w1.n)[13]).max() > 1e-3


# ----------------------------------------------------------------------------------------------
# f1: state-dependent HLLE wave speeds
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_wave_speed_mode_mhd_inside(binding, variant):
    """Ideal-GRMHD characteristic speeds where both face states are denser than the switch, light speed elsewhere:
    (i) a curved periodic block with every state 'inside' (shift, K_ij, off-diagonal metric; even and odd row pitch),
    (ii) the config-5 block across the stellar surface, where the switch separates star and atmosphere;
    the CFL reduction becomes a per-step, state-dependent one and must agree too."""
    from test_oracle_scheme import _pad_periodic, _periodic_problem
    rng = np.random.default_rng(23)
    for n in ((38, 21, 9), (37, 11, 9)):
        metric, P = _periodic_problem(40, rng, True)
        sl = (slice(None), slice(0, n[2]), slice(0, n[1]), slice(0, n[0]))
        metric, P = _pad_periodic(np.ascontiguousarray(metric[sl])), _pad_periodic(np.ascontiguousarray(P[sl]))
        for switch in (0.0, 1.0):                      # everything inside / the switch cuts through the data (rho ~ 1 +- 0.2)
            par = dict(n=n, dx=(1 / 40,) * 3, bc=(0, 0, 0), gamma_eos=5 / 3, sigma_model=0, sigma0=30.0, kappa=1.0,
                       wave_speed_mode=wl.WAVE_MHD_INSIDE, wave_rho_switch=switch)
            g, o = _both(binding, par, metric, P, variant)
            assert abs(g.max_speed() - o.max_speed()) <= 1e-14 * o.max_speed()
            dt = 0.2 / 40
            g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)
            _compare(g, o, n, 1 / 40, TOL1, "mhd speeds 1 step")
            for _ in range(4):
                g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)
            _compare(g, o, n, 1 / 40, TOL20, "mhd speeds 5 steps")
            g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)   # leaves the final recovery pending
            l0 = g.launch_count()
            ms_g, ms_o = g.max_speed(), o.max_speed()                # the pending final recovery is flushed first ...
            assert g.launch_count() - l0 == 1                        # ... and reduces the CFL speed itself: one launch
            assert abs(ms_g - ms_o) <= 1e-12 * ms_o
            assert g.max_speed() == ms_g and g.launch_count() - l0 == 1          # still valid: no launch at all
            g.set_prims(g.get_prims())                               # same state, fused value forgotten:
            assert g.max_speed() == ms_g                             # the stand-alone kernel gives the same bits
    w = wl.tov_like()
    i_surf = int(round((8.125 + 12.0) / w.dx[0]))
    nb, bc = (40, 12, 10), (wl.BC_OUTFLOW,) * 3
    f = w.fields((i_surf - 20, 256 - 6, 256 - 5), nb)
    over = dict(wave_speed_mode=wl.WAVE_MHD_INSIDE, wave_rho_switch=1e-9)
    o = oracle.from_workload(w, fields=f, omp=True, n=nb, bc=bc, **over)
    g = binding.from_workload(w, fields=f, n=nb, bc=bc, **over)
    g.set_rhs_variant(variant)
    for _ in range(10):
        g.step(w.dt, w.recon); o.step(w.dt, w.recon)
    _compare(g, o, nb, w.dx[0], TOL20, "mhd speeds cfg5 block")
    assert g.stats()["floor_resets"] == o.stats()["floor_resets"] > 0
    # the result differs from the light-speed solver (the mode is live), and a switch nothing exceeds is bit-identical to it
    gl = binding.from_workload(w, fields=f, n=nb, bc=bc)
    goff = binding.from_workload(w, fields=f, n=nb, bc=bc, wave_speed_mode=wl.WAVE_MHD_INSIDE, wave_rho_switch=1e30)
    for h in (gl, goff):
        h.set_rhs_variant(variant)
        for _ in range(10):
            h.step(w.dt, w.recon)
    assert np.array_equal(gl.get_prims(), goff.get_prims())
    assert not np.array_equal(gl.get_prims(), g.get_prims())


# ----------------------------------------------------------------------------------------------
# f2: the other IMEX-RK schemes through the general tableau driver (Eq. 32-34)
# ----------------------------------------------------------------------------------------------
TIME_SCHEMES = {"ssp2_332": wl.TIME_SSP2_332, "ssp3_332": wl.TIME_SSP3_332, "ssp3_433": wl.TIME_SSP3_433,
                "ssp2_222_general": wl.TIME_SSP2_222_GENERAL}


@pytest.mark.parametrize("name", sorted(TIME_SCHEMES))
def test_imex_tableau_driver(binding, name):
    """Each scheme against the oracle's literal Eq. 32 on (i) a curved periodic block (all three flux kernels),
    (ii) a config-4 sub-block, (iii) the config-5 block across the stellar surface (floor resets with write-back in the
    final kernel), (iv) a 1D shocktube, (v) charge mode DIV_E."""
    from test_oracle_scheme import _pad_periodic, _periodic_problem
    ts = TIME_SCHEMES[name]
    rng = np.random.default_rng(41)
    n = (38, 21, 9)
    metric, P = _periodic_problem(40, rng, True)
    sl = (slice(None), slice(0, n[2]), slice(0, n[1]), slice(0, n[0]))
    metric, P = _pad_periodic(np.ascontiguousarray(metric[sl])), _pad_periodic(np.ascontiguousarray(P[sl]))
    dt = 0.2 / 40
    for variant in (0, 1, 2):
        for charge in (wl.CHARGE_CELL_CURRENT, wl.CHARGE_DIV_E) if variant == 0 else (wl.CHARGE_CELL_CURRENT,):
            par = dict(n=n, dx=(1 / 40,) * 3, bc=(0, 0, 0), gamma_eos=5 / 3, sigma_model=0, sigma0=30.0, kappa=1.0,
                       charge_mode=charge)
            g, o = _both(binding, par, metric, P, variant)
            g.step(dt, wl.RECON_WENO5 | ts); o.step(dt, wl.RECON_WENO5 | ts)
            _compare(g, o, n, 1 / 40, TOL1, "%s 1 step variant %d charge %d" % (name, variant, charge))
            for _ in range(4):
                g.step(dt, wl.RECON_WENO5 | ts); o.step(dt, wl.RECON_WENO5 | ts)
            _compare(g, o, n, 1 / 40, TOL20, "%s 5 steps" % name)
            assert g.stats()["c2p_failures"] == 0 and g.stats()["c2p_solves"] == o.stats()["c2p_solves"]
    w = wl.blast_curved()
    nb, bc = (40, 36, 20), (wl.BC_OUTFLOW,) * 3
    f = w.fields((120, 138, 100), nb)
    o = oracle.from_workload(w, fields=f, omp=True, n=nb, bc=bc)
    g = binding.from_workload(w, fields=f, n=nb, bc=bc)
    for _ in range(10):
        g.step(w.dt, w.recon | ts); o.step(w.dt, w.recon | ts)
    _compare(g, o, nb, w.dx[0], TOL20, name + " cfg4 block")
    w = wl.tov_like()
    i_surf = int(round((8.125 + 12.0) / w.dx[0]))
    nb = (40, 12, 10)
    f = w.fields((i_surf - 20, 256 - 6, 256 - 5), nb)
    o = oracle.from_workload(w, fields=f, omp=True, n=nb, bc=bc)
    g = binding.from_workload(w, fields=f, n=nb, bc=bc)
    for _ in range(5):
        g.step(w.dt, w.recon | ts); o.step(w.dt, w.recon | ts)
    _compare(g, o, nb, w.dx[0], TOL20, name + " cfg5 block")
    assert g.stats()["floor_resets"] == o.stats()["floor_resets"] > 0
    w1 = wl.shocktube(n=100)
    f1 = w1.fields()
    o = oracle.from_workload(w1, fields=f1)
    g = binding.from_workload(w1, fields=f1)
    for _ in range(20):
        g.step(w1.dt, w1.recon | ts); o.step(w1.dt, w1.recon | ts)
    _compare(g, o, w1.n, w1.dx[0], TOL20, name + " 1D")


def test_general_driver_reproduces_the_tuned_ssp2_222_path(binding):
    """SSP2(2,2,2) through the general driver and through the production kernels (regrouped stage algebra, deferred
    final recovery): same scheme, agreement to round-off; and mixing the two on one handle is allowed."""
    w = wl.blast_curved()
    nb, bc = (40, 36, 20), (wl.BC_OUTFLOW,) * 3
    f = w.fields((120, 138, 100), nb)
    ga = binding.from_workload(w, fields=f, n=nb, bc=bc)
    gb = binding.from_workload(w, fields=f, n=nb, bc=bc)
    gc = binding.from_workload(w, fields=f, n=nb, bc=bc)
    for s in range(6):
        ga.step(w.dt, w.recon)
        gb.step(w.dt, w.recon | wl.TIME_SSP2_222_GENERAL)
        gc.step(w.dt, w.recon | (wl.TIME_SSP2_222_GENERAL if s % 2 else wl.TIME_SSP2_222))
    Pa, Pb, Pc = (interior(h.get_prims(), nb) for h in (ga, gb, gc))
    sc = prim_group_scales(Pa, w.dx[0])
    assert rel_linf(Pb, Pa, sc).max() <= 1e-13 and rel_linf(Pc, Pa, sc).max() <= 1e-13
    assert ga.stats()["c2p_solves"] == gb.stats()["c2p_solves"] == gc.stats()["c2p_solves"]


# ----------------------------------------------------------------------------------------------
# failure paths of the recovery
# ----------------------------------------------------------------------------------------------
def test_recovery_failure_paths_terminate_and_follow_the_conventions(binding):
    """(i) Tiny iteration caps: every solve stops at the cap, is counted as failed, and the step still completes
    (round 2 found that a lane WITHOUT a physical bracket left the solver's loop early while the warp vote still named
    it: a deadlock as soon as one cell of a warp had D^ <= 0; such states only arise after failed solves).
    (ii) A time step far beyond the CFL limit makes the stage vector unphysical in part of the block (no bracket):
    both sides count the same failures and, following the same conventions (keep the guess, E from the guess
    velocity), agree on the outcome of that one step."""
    w = wl.blast_curved()
    n, bc = (48, 40, 24), (wl.BC_OUTFLOW,) * 3
    f = w.fields((100, 108, 100), n)
    for cap in (1, 2, 3):
        g = binding.from_workload(w, fields=f, n=n, bc=bc, c2p_max_iter=cap)
        for _ in range(4):
            g.step(w.dt, w.recon)
        st = g.stats()
        assert st["c2p_max_evals"] <= cap and st["c2p_failures"] > 0 and st["c2p_solves"] == 12 * 48 * 40 * 24
        g.get_prims()
    dt = 40 * w.dt
    g = binding.from_workload(w, fields=f, n=n, bc=bc)
    o = oracle.from_workload(w, fields=f, omp=True, n=n, bc=bc)
    g.step(dt, w.recon); o.step(dt, w.recon)
    sg, so = g.stats(), o.stats()
    assert so["c2p_failures"] > 0, so
    assert sg["c2p_failures"] == so["c2p_failures"], (sg, so)
    Pg, Po = interior(g.get_prims(), n), interior(o.get_prims(), n)
    assert np.isfinite(Pg).all() == np.isfinite(Po).all()
    if np.isfinite(Po).all():
        e = rel_linf(Pg, Po, prim_group_scales(Po, w.dx[0]))
        assert e.max() <= 1e-8, e


def test_set_metric_twice_reallocates_the_static_source_fields(binding):
    """set_metric sizes the slab of static source coefficients by the fields that are not identically zero on the
    grid (none in flat space, 15 for a conformally flat metric, all 34 with shift and K_ij).  Replacing the metric on a
    live handle must give the same results as a fresh handle."""
    from test_oracle_scheme import _pad_periodic, _periodic_problem
    rng = np.random.default_rng(3)
    n = (20, 18, 6)
    metric, P = _periodic_problem(24, rng, True)
    sl = (slice(None), slice(0, n[2]), slice(0, n[1]), slice(0, n[0]))
    metric, P = _pad_periodic(np.ascontiguousarray(metric[sl])), _pad_periodic(np.ascontiguousarray(P[sl]))
    flat = np.zeros_like(metric); flat[0] = 1; flat[4] = flat[7] = flat[9] = 1
    par = dict(n=n, dx=(1 / 24,) * 3, bc=(0, 0, 0), gamma_eos=5 / 3, sigma0=20.0)
    fresh = binding.Rgrmhd(par)
    fresh.set_metric(metric); fresh.set_prims(P)
    reused = binding.Rgrmhd(par)
    reused.set_metric(flat); reused.set_prims(P)
    reused.step(0.005, wl.RECON_WENO5)                   # flat space: no source field allocated
    reused.set_metric(metric); reused.set_prims(P)       # now all of them
    for h in (fresh, reused):
        for _ in range(3):
            h.step(0.005, wl.RECON_WENO5)
    assert np.array_equal(fresh.get_prims(), reused.get_prims())
    reused.set_metric(flat); reused.set_prims(P)         # and back
    ref = binding.Rgrmhd(par)
    ref.set_metric(flat); ref.set_prims(P)
    reused.step(0.005, wl.RECON_WENO5); ref.step(0.005, wl.RECON_WENO5)
    assert np.array_equal(ref.get_prims(), reused.get_prims())


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_superluminal_shift_upwinding(binding, variant):
    """A shift beyond the light cone in every direction, of either sign: one of lambda+- is clipped to zero and HLLE is
    pure upwinding (pinned for the oracle in tests/test_oracle_closed_forms.py); the CFL speed is alpha sqrt(g^kk) + |beta^k|."""
    rng = np.random.default_rng(77)
    n = (38, 21, 9)
    shape = tuple(m + 6 for m in (n[2], n[1], n[0]))
    m = np.zeros((16,) + shape); m[0] = 1.0; m[4] = m[7] = m[9] = 1.0
    m[1], m[2], m[3] = 1.5, -1.4, 1.3
    from test_oracle_scheme import _pad_periodic, _periodic_problem
    _, P = _periodic_problem(40, rng, False)
    sl = (slice(None), slice(0, n[2]), slice(0, n[1]), slice(0, n[0]))
    P = _pad_periodic(np.ascontiguousarray(P[sl]))
    par = dict(n=n, dx=(1 / 40,) * 3, bc=(0, 0, 0), gamma_eos=5 / 3, sigma0=30.0)
    g, o = _both(binding, par, m, P, variant)
    assert g.max_speed() == pytest.approx(2.5 * 40, rel=1e-15) and g.max_speed() == o.max_speed()
    dt = 0.2 / (2.5 * 40)
    g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)
    _compare(g, o, n, 1 / 40, TOL1, "superluminal shift 1 step")
    for _ in range(4):
        g.step(dt, wl.RECON_WENO5); o.step(dt, wl.RECON_WENO5)
    _compare(g, o, n, 1 / 40, TOL20, "superluminal shift 5 steps")
