"""GPU test (-m gpu) of ``rgrmhd_max_speed_static``: the CFL reduction for callers that may not allocate (scratch in a
fixed ``__device__`` array of the library, no handle, no cudaMalloc; include/rgrmhd.h).  Its result is compared with the
existing path (``rgrmhd_max_speed`` of a handle) within the tolerance the other max-speed tests use (1e-14 relative;
the two are in fact the same per-cell function and an exact maximum), on calls in a row that share the scratch array.

The file name sorts last on purpose: the suite runs with ``pytest -x``, and a failure here must not hide other tests.
"""
import numpy as np
import pytest

from paper_2510_18968_b200 import workloads as wl

pytestmark = pytest.mark.gpu

RTOL = 1e-14


@pytest.fixture(scope="module")
def binding():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2510_18968_b200 import binding as b
    b.load()
    return b


def _cases():
    """(name, params, metric (16 padded fields), prims (14 padded fields) or None): sizes from 4 to 432 CTAs of the static
    kernel, ragged extents, a shift, and the state-dependent mode with the switch cutting through the data."""
    from test_oracle_closed_forms import shifted_diagonal_metric
    from test_oracle_scheme import _pad_periodic, _periodic_problem
    out = []
    w = wl.blast_curved(n=96)
    f = w.fields()
    out.append(("cfg4 96^3, light", w.params(), f["metric"], None))
    n, dx = (37, 21, 9), (0.1, 0.2, 0.15)
    shape = tuple(m + 6 for m in (n[2], n[1], n[0]))
    out.append(("shift 37x21x9, light", dict(n=n, dx=dx, bc=(1, 1, 1), gamma_eos=2.0), shifted_diagonal_metric(shape, n, dx), None))
    rng = np.random.default_rng(23)
    n = (38, 21, 9)
    metric, P = _periodic_problem(40, rng, True)
    sl = (slice(None), slice(0, n[2]), slice(0, n[1]), slice(0, n[0]))
    metric, P = _pad_periodic(np.ascontiguousarray(metric[sl])), _pad_periodic(np.ascontiguousarray(P[sl]))
    par = dict(n=n, dx=(1 / 40,) * 3, bc=(0, 0, 0), gamma_eos=5 / 3, sigma_model=0, sigma0=30.0,
               wave_speed_mode=wl.WAVE_MHD_INSIDE, wave_rho_switch=1.0)
    out.append(("periodic 38x21x9, mhd inside", par, metric, P))
    return out


def _existing_path(binding, par, metric, prims):
    g = binding.Rgrmhd(par)
    g.set_metric(metric)
    if prims is not None:
        g.set_prims(prims)
    v = g.max_speed()
    g.close()
    return v


def test_static_max_speed_matches_existing_path_on_calls_in_a_row(binding):
    import torch
    cases = _cases()
    expected = [_existing_path(binding, par, m, P) for _, par, m, P in cases]
    assert len(set(expected)) == len(expected)                    # different answers: a stale result would show
    dev = [(torch.from_numpy(np.ascontiguousarray(m[:10])).cuda(), None if P is None else torch.from_numpy(P).cuda())
           for _, _, m, P in cases]
    # two rounds over all cases, enqueued back to back on one stream WITHOUT host synchronisation in between: every call
    # finds the scratch array as the previous one left it (more partial slots written than it uses itself, or fewer)
    order = list(range(len(cases))) + list(reversed(range(len(cases))))
    outs = [torch.full((1,), -1.0, dtype=torch.float64, device="cuda") for _ in order]
    for o, c in zip(outs, order):
        _, par, _, _ = cases[c]
        md, pd = dev[c]
        binding.max_speed_static(par["n"], par["dx"], md, pd, par["gamma_eos"], par.get("wave_speed_mode", wl.WAVE_LIGHT),
                                 par.get("wave_rho_switch", 0.0), o)
    torch.cuda.synchronize()
    for o, c in zip(outs, order):
        got = float(o.item())
        assert abs(got - expected[c]) <= RTOL * expected[c], (cases[c][0], got, expected[c])
    # the same call twice in a row gives the same bits
    a = torch.zeros(1, dtype=torch.float64, device="cuda")
    b = torch.zeros(1, dtype=torch.float64, device="cuda")
    _, par, _, _ = cases[0]
    for o in (a, b):
        binding.max_speed_static(par["n"], par["dx"], dev[0][0], None, par["gamma_eos"], wl.WAVE_LIGHT, 0.0, o)
    torch.cuda.synchronize()
    assert float(a.item()) == float(b.item())


def test_static_max_speed_size_limit(binding):
    """Exactly RGRMHD_STATIC_MAX_CELLS = 256^3 cells is accepted (flat metric through two shared fields: closed form
    1/dx); one more plane is rejected with the error of its own, before anything is touched."""
    import torch
    n = (256, 256, 256)
    assert n[0] * n[1] * n[2] == binding.STATIC_MAX_CELLS
    one = torch.ones((262, 262, 262), dtype=torch.float64, device="cuda")
    zero = torch.zeros_like(one)
    metric = [one, zero, zero, zero, one, zero, zero, one, zero, one]     # alpha, beta^i, gamma xx xy xz yy yz zz
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    binding.max_speed_static(n, (1 / 256,) * 3, metric, None, 4 / 3, wl.WAVE_LIGHT, 0.0, out)
    torch.cuda.synchronize()
    assert abs(float(out.item()) - 256.0) <= RTOL * 256.0
    out.fill_(-1.0)
    with pytest.raises(binding.RgrmhdError) as e:
        binding.max_speed_static((256, 256, 257), (1 / 256,) * 3, metric, None, 4 / 3, wl.WAVE_LIGHT, 0.0, out)
    assert e.value.code == binding.E_TOO_LARGE and "RGRMHD_STATIC_MAX_CELLS" in str(e.value)
    torch.cuda.synchronize()
    assert float(out.item()) == -1.0                                      # nothing was launched
    # and the array is still usable after the rejected call
    binding.max_speed_static((8, 8, 8), (0.5, 0.25, 0.125), metric, None, 4 / 3, wl.WAVE_LIGHT, 0.0, out)
    torch.cuda.synchronize()
    assert abs(float(out.item()) - 8.0) <= RTOL * 8.0
