"""The three readings of the charge sector (reading R3): A = FACE_OHM (Ohm's law on
the reconstructed face states), B = CELL_CURRENT (default), C = DIV_E (q = nabla_i E^i).  Pins of mode C
and the committed version of the comparison that froze B as the default.  CPU only (OpenMP oracle)."""
import numpy as np
import pytest

import oracle
from helpers import interior
from paper_2510_18968_b200 import workloads as wl


def _padded_coords(n, dx):
    ax = [(np.arange(-3, m + 3) + 0.5) * d for m, d in zip(n, dx)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return X, Y, Z


def test_div_e_charge_is_the_centred_divergence_of_calE_exact_on_quadratics():
    """Mode C after one step of a configuration in which calE is constant in time (sigma = 0, v = 0, B = 0, psi = 0: no
    current, no curl, no cleaning flux): q^{n+1} = d_i(calE^i)/sqrt(gamma).  With calE^i QUADRATIC in the coordinates the
    second-order centred difference is exact, so q is known in closed form on a curved (conformally flat) metric:
    pins the densitisation, the stencil and the 1/(2 dx) of reading R15."""
    n, dx = (10, 8, 6), (0.1, 0.15, 0.2)
    par = dict(n=n, dx=dx, bc=(1, 1, 1), gamma_eos=2.0, sigma0=0.0, charge_mode=wl.CHARGE_DIV_E)
    o = oracle.Oracle(par)
    X, Y, Z = _padded_coords(n, dx)
    f = 1.0 + 0.2 * np.sin(X + 0.5 * Y) + 0.1 * np.cos(Z)                  # gamma_ij = f delta_ij, sqrt(gamma) = f^1.5
    m = np.zeros((16,) + o.shape)
    m[0] = 1.0; m[4] = m[7] = m[9] = f
    cE = [0.3 * X * X + 0.1 * X * Y - 0.2 * Z, 0.05 * Y * Y - 0.3 * X * Z + 0.1, -0.15 * Z * Z + 0.2 * Y * Z + 0.1 * X]
    div = (0.6 * X + 0.1 * Y) + (0.1 * Y) + (-0.3 * Z + 0.2 * Y)           # d_x cE^x + d_y cE^y + d_z cE^z
    P = np.zeros((14,) + o.shape)
    P[0] = 1.0; P[1] = 1.0
    for i in range(3):
        P[5 + i] = 1e-3 * cE[i] / f ** 1.5
    P[13] = 7.0                                                            # whatever the caller passes as q is replaced
    o.set_metric(m); o.set_prims(P)
    o.step(1e-12, wl.RECON_MC)      # the HLLE dissipation of the quadratic profile moves calE by O(dt dx calE''): negligible
    q = interior(o.get_prims(), n)[13]
    Q = interior(o.get_cons(), n)[13]
    expQ = interior(1e-3 * div[None], n)[0]
    # outflow ghosts copy E^i of the nearest interior cell: the closed form holds one cell away from the block faces
    inner = (slice(1, -1),) * 3
    assert np.allclose(Q[inner], expQ[inner], rtol=0, atol=2e-15)
    assert np.allclose(q[inner], (expQ / interior(f[None], n)[0] ** 1.5)[inner], rtol=0, atol=2e-15)


def test_div_e_total_charge_telescopes_to_zero_on_a_periodic_block():
    from test_oracle_scheme import _pad_periodic, _periodic_problem
    rng = np.random.default_rng(8)
    metric, P = _periodic_problem(8, rng, True)
    par = dict(n=(8, 8, 8), dx=(1 / 8,) * 3, bc=(0, 0, 0), gamma_eos=5 / 3, sigma0=20.0, charge_mode=wl.CHARGE_DIV_E)
    o = oracle.Oracle(par)
    o.set_metric(_pad_periodic(metric)); o.set_prims(_pad_periodic(P))
    for _ in range(3):
        o.step(0.02, wl.RECON_WENO5)
    Q = interior(o.get_cons(), (8, 8, 8))[13]
    assert abs(Q.sum()) <= 1e-13 * np.abs(Q).sum() and np.abs(Q).max() > 1e-3
    assert o.stats()["c2p_failures"] == 0


@pytest.mark.slow
def test_charge_modes_compared_on_config3_and_config4():
    """The comparison SURVEY.md Sec. 7 step 2 asked for before freezing the mode (reading R3):
    config 3 (32^3, sigma = 1e8, 20 steps): the literal face evaluation (A) multiplies reconstruction mismatch by sigma,
    max|q| > 100; the cell-current reading (B) and q = div E (C) keep |q| < 1e-2 and agree with each other in B and v
    ('no significant differences');
    a config-4 sub-block (random sigma in [1, 1e6]): A loses finiteness within 30 steps, B and C stay finite with no
    failed solve."""
    w = wl.alfven3d(n=32)
    f = w.fields()
    out = {}
    for mode in (wl.CHARGE_FACE_OHM, wl.CHARGE_CELL_CURRENT, wl.CHARGE_DIV_E):
        o = oracle.from_workload(w, fields=f, omp=True, charge_mode=mode)
        for _ in range(20):
            o.step(w.dt, w.recon)
        out[mode] = o.get_prims()
        assert np.isfinite(out[mode]).all()
        assert mode == wl.CHARGE_FACE_OHM or o.stats()["c2p_failures"] == 0     # (A also makes the recovery fail)
    qmax = {k: float(np.abs(v[13]).max()) for k, v in out.items()}
    assert qmax[wl.CHARGE_FACE_OHM] > 100 and qmax[wl.CHARGE_CELL_CURRENT] < 1e-2 and qmax[wl.CHARGE_DIV_E] < 1e-2, qmax
    B, C = out[wl.CHARGE_CELL_CURRENT], out[wl.CHARGE_DIV_E]
    assert np.abs(B[8:11] - C[8:11]).max() < 1e-5 and np.abs(B[2:5] - C[2:5]).max() < 1e-5
    w = wl.blast_curved()
    n = (40, 36, 20)
    f = w.fields((120, 138, 100), n)
    finite_steps = {}
    for mode in (wl.CHARGE_FACE_OHM, wl.CHARGE_CELL_CURRENT, wl.CHARGE_DIV_E):
        o = oracle.from_workload(w, fields=f, omp=True, n=n, bc=(wl.BC_OUTFLOW,) * 3, charge_mode=mode)
        k = 0
        for k in range(1, 31):
            o.step(w.dt, w.recon)
            if not np.isfinite(o.get_prims()).all():
                break
        else:
            k = 31
        finite_steps[mode] = k
        if mode != wl.CHARGE_FACE_OHM:
            assert o.stats()["c2p_failures"] == 0
    assert finite_steps[wl.CHARGE_FACE_OHM] <= 30, finite_steps
    assert finite_steps[wl.CHARGE_CELL_CURRENT] == 31 and finite_steps[wl.CHARGE_DIV_E] == 31, finite_steps
