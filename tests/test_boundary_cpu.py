"""CPU-side checks of the C-ABI boundary and of the host logic (no compute call, no GPU):

* ``librgrmhd.so`` loads and exports every function ``include/rgrmhd.h`` declares, and nothing the
  header does not declare carries the ``rgrmhd_`` prefix;
* the ctypes mirror of ``rgrmhd_params`` / ``rgrmhd_stats`` has the layout the C compiler gives the
  header's structs (checked by compiling a probe with gcc);
* enum values mirrored in ``workloads.py`` equal the header's;
* the product path has no CPU fallback and never imports ``oracle``;
* argument validation that happens before any CUDA call.
"""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "rgrmhd.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rgrmhd_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2510_18968_b200 import build, binding
    build.build()
    return binding.load()


def test_library_exports_every_declared_symbol(lib):
    from paper_2510_18968_b200 import binding
    decl = _declared_functions()
    assert len(decl) >= 14
    for name in decl:
        assert hasattr(lib, name), "declared in include/rgrmhd.h but not exported: " + name
    assert sorted(binding.SYMBOLS) == decl
    out = subprocess.run(["nm", "-D", "--defined-only", binding._LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = sorted(set(re.findall(r" T (rgrmhd_[a-z0-9_]+)", out)))
    assert exported == decl, (set(exported) ^ set(decl))


def test_struct_layout_matches_the_c_compiler(tmp_path):
    from paper_2510_18968_b200 import binding
    probe = tmp_path / "probe.c"
    fields_p = [f for f, _ in binding.Params._fields_]
    fields_s = [f for f, _ in binding.Stats._fields_]
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "rgrmhd.h"', 'int main(void){',
             'printf("%zu\\n", sizeof(rgrmhd_params));']
    lines += ['printf("%%zu\\n", offsetof(rgrmhd_params, %s));' % f for f in fields_p]
    lines += ['printf("%zu\\n", sizeof(rgrmhd_stats));']
    lines += ['printf("%%zu\\n", offsetof(rgrmhd_stats, %s));' % f for f in fields_s]
    lines += ['printf("%d %d %d %d %d\\n", RGRMHD_OK, RGRMHD_E_INVALID, RGRMHD_E_STATE, RGRMHD_E_CUDA, RGRMHD_E_NOMEM);',
              'return 0;}']
    probe.write_text("\n".join(lines))
    exe = tmp_path / "probe"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(probe), "-o", str(exe)],
                   check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split("\n")
    it = iter(out)
    assert int(next(it)) == C.sizeof(binding.Params)
    for f in fields_p:
        assert int(next(it)) == getattr(binding.Params, f).offset, f
    assert int(next(it)) == C.sizeof(binding.Stats)
    for f in fields_s:
        assert int(next(it)) == getattr(binding.Stats, f).offset, f
    assert next(it).split() == ["0", "-1", "-2", "-3", "-4"]


def test_enum_values_mirrored_in_workloads():
    from paper_2510_18968_b200 import workloads as wl
    src = open(HEADER).read()
    vals = dict((k, int(v)) for k, v in re.findall(r"\b(RGRMHD_[A-Z0-9_]+)\s*=\s*(-?\d+)\b(?!\s*<<)", src))
    for k in ("BC_PERIODIC", "BC_OUTFLOW", "SIGMA_UNIFORM", "SIGMA_ARRAY", "SIGMA_POWER_D", "SIGMA_ATMO",
              "RECON_MINMOD", "RECON_MC", "RECON_WENO5", "CHARGE_FACE_OHM", "CHARGE_CELL_CURRENT", "CHARGE_DIV_E",
              "WAVE_LIGHT", "WAVE_MHD_INSIDE"):
        assert vals["RGRMHD_" + k] == getattr(wl, k), k


def test_defaults_and_validation_before_any_cuda_call(lib):
    from paper_2510_18968_b200 import binding
    p = binding.params_default()
    assert p.ng == 3 and p.kappa == 1.0 and p.charge_mode == 1 and list(p.n) == [1, 1, 1]
    h = C.c_void_p()
    assert lib.rgrmhd_params_default(None) == -1
    assert lib.rgrmhd_create(None, C.byref(p)) == -1
    assert lib.rgrmhd_create(C.byref(h), None) == -1
    p.n[:] = [8, 1, 1]; p.dx[:] = [0.1, 0.1, 0.1]
    for field, bad in (("ng", 2), ("gamma_eos", 1.0), ("sigma_model", 7), ("charge_mode", 5), ("rho_floor", -1.0)):
        good = getattr(p, field)
        setattr(p, field, bad)
        assert lib.rgrmhd_create(C.byref(h), C.byref(p)) == -1, field
        assert not h.value
        setattr(p, field, good)
    p.n[0] = 2                                     # active directions need >= 3 cells (periodic wrap of 3 ghosts)
    assert lib.rgrmhd_create(C.byref(h), C.byref(p)) == -1
    p.n[0] = 8; p.bc[1] = 9
    assert lib.rgrmhd_create(C.byref(h), C.byref(p)) == -1
    for fn in ("rgrmhd_destroy", "rgrmhd_reset_stats"):
        assert getattr(lib, fn)(None) == -1
    assert lib.rgrmhd_step(None, 0.1, 2) == -1
    assert lib.rgrmhd_max_speed(None, None) == -1
    assert b"ok" == lib.rgrmhd_strerror(0) and b"unknown" in lib.rgrmhd_strerror(-99)
    assert lib.rgrmhd_last_cuda_error(None) == b""


def test_no_cpu_fallback_without_a_device(lib):
    """On a box without a GPU create() must fail with E_CUDA (it never computes on the host)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2510_18968_b200 import binding
    with pytest.raises(binding.RgrmhdError) as e:
        binding.Rgrmhd(dict(n=(8, 1, 1), dx=(0.1,) * 3, bc=(1, 1, 1), gamma_eos=2.0))
    assert e.value.code == -3
    out = C.c_double()
    assert lib.rgrmhd_measure_fp64_peak(0, 1, C.byref(out)) < 0


def test_product_path_never_imports_the_oracle():
    code = ("import sys; import paper_2510_18968_b200; from paper_2510_18968_b200 import binding, workloads, build;"
            "binding.load(); assert 'oracle' not in sys.modules; print('ok')")
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, cwd=ROOT)
    assert r.returncode == 0 and r.stdout.strip() == "ok", r.stderr
    pkg = os.path.join(ROOT, "paper_2510_18968_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), fn
                assert "rgrmhd_oracle" not in txt, fn


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_2510_18968_b200 import binding
    monkeypatch.setattr(binding, "_LIB", None)
    monkeypatch.setattr(binding, "_LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(ImportError):
        binding.load()


def test_workload_generators_are_seeded_and_subblocks_agree():
    from paper_2510_18968_b200 import workloads as wl
    w = wl.blast_curved()
    a = w.fields((100, 90, 80), (9, 8, 7))
    b = w.fields((100, 90, 80), (9, 8, 7))
    for k in ("prims", "metric", "sigma"):
        assert np.array_equal(a[k], b[k])
    big = w.fields((98, 88, 78), (13, 12, 11))
    # interior of the small block = the same global cells of the bigger block
    assert np.array_equal(a["sigma"][3:-3, 3:-3, 3:-3], big["sigma"][5:5 + 7, 5:5 + 8, 5:5 + 9])
    assert np.array_equal(a["metric"][:, 3:-3, 3:-3, 3:-3], big["metric"][:, 5:5 + 7, 5:5 + 8, 5:5 + 9])
    s = a["sigma"][3:-3, 3:-3, 3:-3]
    assert s.min() >= 1.0 and s.max() <= 1e6
    u = wl.splitmix64_uniform(4, np.arange(100000))
    assert 0.0 <= u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 5e-3
