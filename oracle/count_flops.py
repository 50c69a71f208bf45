"""Instrumented flop count of one zone-cycle from the oracle (TEST / MEASUREMENT INFRASTRUCTURE).

    python -m oracle.count_flops            # prints a table and rewrites oracle/flop_count.json

Builds rgrmhd_oracle.cpp with -DORACLE_COUNT_FLOPS (a counting scalar replaces `double`: add/sub, mul, div, sqrt each
count 1, so an FMA counts 2), runs ONE step of a sub-block of every BASELINE config (the robust solver, whose
evaluation counts are those of the CUDA path's algorithm) and tallies the operations per region of the step and per
interior cell.  Calls only oracle/ and the input generators.

How to read it.  The oracle is written for legibility, not economy: every face reconstructs its two cells from
scratch (each cell's pair of face values is evaluated twice per direction where once suffices, in the Jiang-Shu form
with three divisions per face value), prim->cons is evaluated again inside every face state's flux, the Levi-Civita
and Christoffel sums run over all index triples including the zeros, the metric derivatives are differenced in every
stage although the metric is fixed, and face metrics are inverted in full.  The counts below are therefore an UPPER
bound of the algorithmic work; the total with every reconstruction counted once is reported next to the raw figure.  bench.py prints both this count and its own minimal-operation hand count."""
from __future__ import annotations

import ctypes as C
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2510_18968_b200 import workloads as wl  # noqa: E402

REGIONS = ["other", "recon", "riemann", "divergence", "sources", "c2p_setup", "c2p_eval", "combine", "p2c"]
OPS = ["add", "mul", "div", "sqrt"]


def count(w, lo, n, bc):
    L = oracle.lib("count")
    f = w.fields(lo, n)
    o = oracle.from_workload(w, fields=f, omp="count", n=n, bc=bc, solver="robust")
    L.oracle_flops_reset()
    o.step(w.dt, w.recon)
    out = (C.c_longlong * (len(REGIONS) * len(OPS)))()
    calls = (C.c_longlong * len(REGIONS))()
    L.oracle_flops_get(out, calls)
    ncell = int(np.prod(n))
    a = np.array(out[:], dtype=np.float64).reshape(len(REGIONS), len(OPS))
    st = o.stats()
    per_cell = {r: float(a[i].sum()) / ncell for i, r in enumerate(REGIONS)}
    res = {"workload": w.name, "sub_block": {"lo": list(lo), "n": list(n)}, "cells": ncell,
           "flops_per_zone_cycle_by_region": per_cell,
           "ops_per_zone_cycle": {op: float(a[:, j].sum()) / ncell for j, op in enumerate(OPS)},
           "c2p_evals_per_solve": st["c2p_evals"] / st["c2p_solves"],
           "flops_per_c2p_eval": float(a[REGIONS.index("c2p_eval")].sum()) / max(st["c2p_evals"], 1),
           "flops_per_recon_call": float(a[REGIONS.index("recon")].sum()) / max(calls[REGIONS.index("recon")], 1),
           "recon_calls_per_cell_rhs": calls[REGIONS.index("recon")] / ncell / 2.0,
           "riemann_flops_per_face": float(a[REGIONS.index("riemann")].sum()) / max(calls[REGIONS.index("riemann")], 1)}
    # a cell's reconstruction pair (both faces of one variable in one direction) is needed once; the oracle's
    # recon_cell computes the pair, and is called twice per cell and face side
    ndir = sum(1 for m in n if m > 1)
    nvar = 15 if w.charge_mode != wl.CHARGE_FACE_OHM else 14
    res["recon_min_flops_per_zone_cycle"] = 2 * ndir * nvar * res["flops_per_recon_call"]
    res["total_flops_per_zone_cycle_oracle"] = float(a.sum()) / ncell
    res["total_flops_per_zone_cycle_recon_once"] = (res["total_flops_per_zone_cycle_oracle"] - per_cell["recon"]
                                                      + res["recon_min_flops_per_zone_cycle"])
    return res


def main():
    out = {}
    cases = [("cfg1", wl.shocktube(), (0, 0, 0), (400, 1, 1), None),
             ("cfg2", wl.current_sheet(), (0, 0, 0), (800, 1, 1), None),
             ("cfg3", wl.alfven3d(n=32), (0, 0, 0), (32, 32, 32), None),
             ("cfg4", wl.blast_curved(), (112, 112, 112), (32, 32, 32), (wl.BC_OUTFLOW,) * 3),
             ("cfg5", wl.tov_like(), (400, 240, 240), (32, 32, 32), (wl.BC_OUTFLOW,) * 3)]
    for name, w, lo, n, bc in cases:
        r = count(w, lo, n, bc)
        out[name] = r
        print("%s  oracle total %.0f flops/zone-cycle (recon counted once: %.0f); per region: %s; %.1f evals/solve, %.0f "
              "flops/eval, %.0f flops per WENO/TVD pair, %.0f per face Riemann solve" % (
                  name, r["total_flops_per_zone_cycle_oracle"], r["total_flops_per_zone_cycle_recon_once"],
                  {k: round(v) for k, v in r["flops_per_zone_cycle_by_region"].items()}, r["c2p_evals_per_solve"],
                  r["flops_per_c2p_eval"], r["flops_per_recon_call"], r["riemann_flops_per_face"]))
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "flop_count.json"), "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
        f.write("\n")


if __name__ == "__main__":
    main()
