"""GPU tests (-m gpu) of the slab decomposition with halo exchange: a block cut
into 2 or 3 z-slabs, each an ordinary handle with an EXTERNAL z direction, stepped part by part in one process on one
GPU with the halo planes moved between them, must reproduce the undivided block BIT FOR BIT (the same kernels see the
same stencils); and the undivided block matches the oracle in the other tests."""
import numpy as np
import pytest

from helpers import interior
from paper_2510_18968_b200 import slab, workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2510_18968_b200 import binding as b
    b.load()
    return b


CASES = {
    "alfven_periodic": lambda: wl.alfven3d(n=24),                       # periodic in z: the end slabs exchange with each other
    "blast_outflow": lambda: wl.blast_curved(n=40),                     # curved metric, random sigma, outflow walls
    "tov_floor": lambda: wl.tov_like(n=36),                             # atmosphere resets, POWER_D conductivity
}


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("nslabs", [2, 3])
@pytest.mark.parametrize("case", sorted(CASES))
def test_slabs_reproduce_the_undivided_block(binding, case, nslabs, variant):
    w = CASES[case]()
    one = binding.from_workload(w)
    one.set_rhs_variant(variant)
    many = slab.LocalSlabs(binding, w, nslabs, rhs_variant=variant)
    assert many.max_speed() == one.max_speed()
    dt = w.cfl / one.max_speed()
    for _ in range(4):
        one.step(dt, w.recon)
        many.step(dt, w.recon)
    P1, U1 = interior(one.get_prims(), w.n), interior(one.get_cons(), w.n)
    assert np.isfinite(P1).all()
    assert np.array_equal(many.gather_prims(), P1)
    assert np.array_equal(many.gather_cons(), U1)
    s1 = one.stats()
    sm = [s.g.stats() for s in many.slabs]
    for key in ("c2p_solves", "c2p_evals", "c2p_failures", "floor_resets"):
        assert sum(s[key] for s in sm) == s1[key], key
    if case == "tov_floor":
        assert s1["floor_resets"] > 0


def test_split_step_api_rules(binding):
    """A handle with an EXTERNAL direction steps only in the split form; while a split step is in flight the state
    cannot be read; the split form on an ordinary block equals rgrmhd_step."""
    w = wl.alfven3d(n=12)
    f = w.fields()
    g = binding.from_workload(w, fields=f)
    h = binding.from_workload(w, fields=f)
    for _ in range(3):
        g.step(w.dt, w.recon)
        h.step_begin(w.dt, w.recon)
        with pytest.raises(binding.RgrmhdError) as e:
            h.get_prims()
        assert e.value.code == -2
        with pytest.raises(binding.RgrmhdError):
            h.step(w.dt, w.recon)
        assert h.step_continue() is True
        assert h.step_continue() is False
        with pytest.raises(binding.RgrmhdError):
            h.step_continue()
    assert np.array_equal(g.get_prims(), h.get_prims())
    par = w.params(bc=(wl.BC_PERIODIC, wl.BC_PERIODIC, wl.BC_EXTERNAL))
    x = binding.Rgrmhd(par)
    x.set_metric(f["metric"]); x.set_prims(f["prims"])
    with pytest.raises(binding.RgrmhdError) as e:
        x.step(w.dt, w.recon)
    assert e.value.code == -1
    assert x.halo_doubles(2) == 17 * 3 * 18 * 18
    with pytest.raises(binding.RgrmhdError):
        binding.Rgrmhd(dict(par, charge_mode=wl.CHARGE_DIV_E))
