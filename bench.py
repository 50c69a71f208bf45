#!/usr/bin/env python
"""bench.py -- zone-cycles/s of one full IMEX-RK2 step of resistive GRMHD (FP64) on B200.

Contract (task prompt): ``python bench.py --gpus N --steps K --warmup W`` does W untimed steps, times
exactly K steps (barrier + synchronize on both sides, CUDA events, max over ranks) and prints ONE JSON
line on rank 0.  A "step" is one pass of the whole hot path (a6 a1 a2-a5 a6 a1 a2-a5
a6) over the workload.  Inputs are seeded and synthetic (paper_2510_18968_b200/workloads.py).

* ``value``     zone-cycles/s with the state resident in HBM (whole job: all ranks' zones / max time)
* ``e2e``       the same metric through the C-ABI with HOST buffers: every step uploads the primitives
                from pinned host memory (set_prims), steps, and reads the primitives back (get_prims)
* ``roofline``  the dominant kernel (the TMA-staged flux-divergence kernel) against the measured FP64 DFMA
                peak or the measured HBM copy bandwidth, whichever bounds it
* ``cpu_baseline``  the CPU oracle, as it stands (single thread), on a bounded sample of the same workload

``--impl reference`` times the oracle instead (the paper ships no code; the oracle is the reference arm).
The path does not shard (north_star: one GPU, no collectives): ``--gpus N`` runs N independent replicas
("replicas only"); scaling is weak.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2510_18968_b200 import workloads as wl  # noqa: E402

METRIC = "zone-cycles/sec per IMEX-RK2 step (FP64)"
UNIT = "zone-cycles/s"

# Algorithmic work of the dominant kernel (flux divergence: reconstruct + HLLE + divergence + update of the
# stage target), per interior cell and launch -- derivation in DESIGN.md Sec. 7.
RHS_FLOPS = {wl.RECON_WENO5: 5500.0, wl.RECON_MC: 1900.0, wl.RECON_MINMOD: 1800.0}
RHS_DOUBLES = 41.0      # reads P 14 + jc 3 + alpha, beta, gamma_ij 10, writes the increment dU 14
SRC_FLOPS = 350.0       # explicit sources + point-wise stage combine (inside the recovery kernel), per stage
C2P_SETUP_FLOPS, C2P_EVAL_FLOPS = 250.0, 100.0   # per solve / per residual evaluation
STEP_DOUBLES = 253.0    # algorithmic traffic of one zone-cycle
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 DFMA/clk x 2 x 1.965 GHz = 37.2


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


def roof_kernel(variant: int) -> str:
    return {0: "k_flux_tma", 1: "k_rhs_simple", 2: "k_rhs_pencil"}[variant]


def oracle_flop_count(cfg: str):
    """The instrumented count of the oracle's own arithmetic for one zone-cycle of `cfg` (oracle/flop_count.json,
    written by `python -m oracle.count_flops`; a data file: nothing under oracle/ is executed here), or None."""
    p = os.path.join(ROOT, "oracle", "flop_count.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        return json.load(f).get(cfg)


def ncu_traffic(kernel: str, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture
    (profiles/ncu_traffic.md), or None if that kernel / workload was not captured."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.md")
    if not os.path.exists(p):
        return None
    for line in open(p):
        c = [x.strip() for x in line.strip().strip("|").split("|")]
        if len(c) == 3 and c[0] == kernel and c[1] == workload:
            try:
                return float(c[2])
            except ValueError:
                return None
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            c = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(c[0])); smax = float(c[1])
            except Exception:
                continue
            for nm, v in zip(names, c[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


def get_workload(name: str):
    return wl.get(name)


# ----------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py touches oracle/)
# ----------------------------------------------------------------------------------------------
ORACLE_RATE = 7.0e4   # single-thread oracle zone-cycles/s (order of magnitude, used only to size samples)


def oracle_sample(w, cells_budget: float):
    """A bounded sample of workload w for the single-thread oracle: the whole grid if it has at most
    cells_budget cells, else a centred cubic sub-block (outflow boundaries) of about that many cells."""
    if w.ncells <= cells_budget:
        return (0, 0, 0), tuple(w.n), tuple(w.bc)
    ndim = sum(1 for m in w.n if m > 1)
    side = int(round(cells_budget ** (1.0 / ndim)))
    side = max(16, min(side, min(m for m in w.n if m > 1)))
    shape = tuple(side if m > 1 else 1 for m in w.n)
    lo = tuple((m - s) // 2 if m > 1 else 0 for m, s in zip(w.n, shape))
    return lo, shape, (wl.BC_OUTFLOW,) * 3


def time_oracle(w, steps: int, warmup: int, seconds_per_step: float):
    import oracle  # test infrastructure: cpu_baseline / --impl reference legs only
    lo, shape, bc = oracle_sample(w, ORACLE_RATE * seconds_per_step)
    f = w.fields(lo, shape)
    o = oracle.from_workload(w, fields=f, omp=False, n=shape, bc=bc)
    for _ in range(warmup):
        o.step(w.dt, w.recon)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(w.dt, w.recon)
    dt = time.perf_counter() - t0
    ncell = int(np.prod(shape))
    sample = "%s sub-block lo=%s shape=%s, %d steps, single-thread oracle (g++ -O2 -ffp-contract=off)" % (
        w.name, list(lo), list(shape), steps)
    return ncell * steps / dt, dt / steps * 1e3, sample, ncell


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = get_workload(args.config)
    # each step is one oracle step on the bounded sample; sized so the whole run ends within minutes
    total = max(1, args.steps + args.warmup)
    value, ms, sample, ncell = time_oracle(w, steps=args.steps, warmup=args.warmup,
                                           seconds_per_step=min(10.0, max(0.5, 90.0 / total)))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n": list(w.n), "recon": int(w.recon), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------------
# rank plumbing ("replicas only": the path does not shard, so the only cross-rank operations are the
# barrier around the timed region and the max of the per-rank times)
# ----------------------------------------------------------------------------------------------
class Ranks:
    """torch.distributed wrapper used by bench.py: NCCL on the GPU box, gloo in the CPU test."""

    def __init__(self, world: int, backend: str, local: int = 0):
        self.world, self.backend, self.dist = world, backend, None
        if world > 1:
            import torch
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            if backend == "nccl":
                dist.init_process_group("nccl", device_id=torch.device("cuda", local))
            else:
                dist.init_process_group(backend)
            self.dist = dist

    def barrier(self):
        import torch
        if self.dist is not None:
            self.dist.barrier()
        if self.backend == "nccl":
            torch.cuda.synchronize()

    def max_over_ranks(self, x: float) -> float:
        if self.dist is None:
            return x
        import torch
        t = torch.tensor([x], dtype=torch.float64, device="cuda" if self.backend == "nccl" else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate(self, units_per_rank: int, steps: int, ms_local: float) -> float:
        """Whole-job throughput: units all ranks processed / max-over-ranks time."""
        return self.world * units_per_rank * steps / (self.max_over_ranks(ms_local) * 1e-3)

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


# ----------------------------------------------------------------------------------------------
# the CUDA path
# ----------------------------------------------------------------------------------------------
def measure_resident(g, w, dt, steps, warmup, stream, barrier, max_over_ranks, per_kernel=True):
    """W untimed warm-up steps, then exactly K steps between CUDA events on the launching stream (barrier +
    synchronize on both sides); state resident in HBM; per-kernel-class device times from the library's own events."""
    import torch
    for _ in range(warmup):
        g.step(dt, w.recon)
    g.flush()                                          # the warm-up's deferred final recovery stays outside
    g.get_timing()
    g.reset_stats()
    l0 = g.launch_count()
    g.set_timing(per_kernel)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        g.step(dt, w.recon)
    g.flush()                                          # the last step's final recovery is part of the K steps
    e1.record(stream)
    barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    launches = g.launch_count() - l0
    timing = g.get_timing()
    g.set_timing(False)
    stats = g.stats()
    finite = bool(np.isfinite(g.get_prims()).all())
    return {"ms_total": ms_total, "launches": launches, "timing": timing, "stats": stats, "finite": finite}


def step_roofline(w, stats, zc_per_s_per_gpu, fp64_peak, hbm_gbs):
    """north_star: the slower of the algorithmic bytes at HBM bandwidth and the algorithmic FP64 flops at peak."""
    evals_per_solve = stats["c2p_evals"] / max(stats["c2p_solves"], 1)
    ndir = sum(1 for m in w.n if m > 1)
    step_flops = (2 * RHS_FLOPS[w.recon] * ndir / 3.0 + 2 * SRC_FLOPS + 3 * C2P_SETUP_FLOPS +
                  3 * evals_per_solve * C2P_EVAL_FLOPS)
    step_bytes = STEP_DOUBLES * 8.0
    t = max(step_flops / (fp64_peak * 1e12), step_bytes / (hbm_gbs * 1e9))
    return {"zone_cycles_per_s_at_roofline": 1.0 / t, "frac": zc_per_s_per_gpu * t, "flops_per_zone_cycle": step_flops,
            "bytes_per_zone_cycle": step_bytes, "c2p_evals_per_solve": evals_per_solve,
            "flop_count": "minimal-operation hand count of the scheme's formulas (DESIGN.md Sec. 7.5)"}


EXTRA_STEPS = {"cfg1": 200, "cfg2": 200, "cfg3": 20, "cfg4": 10, "cfg5": 5}


def measure_extra_config(binding, name, local, stream, fp64_peak, hbm_gbs):
    """The other BASELINE configs, measured in the same run with the same code (state resident, W = 3)."""
    w = wl.get(name)
    g = binding.from_workload(w, device=local)
    g.set_stream(stream.cuda_stream)
    dt = w.cfl / g.max_speed()
    steps = EXTRA_STEPS[name]
    sync = lambda: __import__("torch").cuda.synchronize()
    m = measure_resident(g, w, dt, steps, 3, stream, sync, lambda x: x)
    if w.ncells < (1 << 20):
        # launch-bound block: the per-kernel event brackets (two events per launch) cost more than the kernels; time the
        # steps again without them and keep the per-kernel split of the first pass
        m["ms_total"] = measure_resident(g, w, dt, steps, 3, stream, sync, lambda x: x, per_kernel=False)["ms_total"]
    ms = m["ms_total"] / steps
    zc = w.ncells * steps / (m["ms_total"] * 1e-3)
    out = {"n": list(w.n), "steps": steps, "ms_per_step": ms, "zone_cycles_per_s": zc,
           "kernel_ms_per_step": {k: v[0] / steps for k, v in m["timing"].items()},
           "gpu_launches": int(m["launches"]), "rhs_kernel": roof_kernel(g.get_rhs_variant()), "finite": m["finite"],
           "c2p_failures": m["stats"]["c2p_failures"], "floor_resets": m["stats"]["floor_resets"]}
    sr = step_roofline(w, m["stats"], zc, fp64_peak, hbm_gbs)
    out["step_roofline_frac"] = sr["frac"] if w.ncells >= 1 << 20 else None     # launch-bound below: absolute numbers only
    out["c2p_evals_per_solve"] = sr["c2p_evals_per_solve"]
    g.close()
    return out


def run_slabs(args, w, ranks, rank, world, local):
    """--slabs with N > 1: ONE copy of the workload cut into N z-slabs, one per rank, with the halo exchange of
    paper_2510_18968_b200/slab.py after each stage: strong scaling.  Not the default: the
    north_star fixes one GPU and replicas; this build's GPU box has one GPU, so this path is
    exercised by the single-GPU slab tests and the gloo exchange test only."""
    import torch
    from paper_2510_18968_b200 import binding, slab
    s = slab.DistSlab(binding, w, device=local, rhs_variant=args.rhs_variant)
    dt = w.cfl / s.max_speed()
    for _ in range(args.warmup):
        s.step(dt, w.recon)
    s.g.flush()
    l0 = s.g.launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    ranks.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record()
    for _ in range(args.steps):
        s.step(dt, w.recon)
    s.g.flush()
    e1.record()
    ranks.barrier()
    t1 = time.time()
    ms_total = ranks.max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop(t0, t1) if sampler else None
    launches = s.g.launch_count() - l0
    finite = bool(np.isfinite(s.interior_prims()).all())
    if rank == 0:
        line = {"metric": METRIC, "value": w.ncells * args.steps / (ms_total * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.name, "n": list(w.n), "parallelism": "z-slabs x%d, halo exchange per stage" % world,
                           "slab_planes": s.n[2], "halo_bytes_per_face_and_exchange": s.g.halo_doubles(2) * 8},
                "clocks": clocks, "gpu_launches": int(launches), "finite": finite, "e2e": None, "roofline": None,
                "cpu_baseline": None}
        print(json.dumps(line), flush=True)
    ranks.close()
    return 0 if finite else 1


def run_ours(args):
    import torch
    from paper_2510_18968_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    ranks = Ranks(world, "nccl", local)
    barrier, max_over_ranks = ranks.barrier, ranks.max_over_ranks
    dist = ranks.dist

    w = get_workload(args.config)
    if args.slabs and world > 1:
        return run_slabs(args, w, ranks, rank, world, local)
    f = w.fields()                                     # every replica: the same seeded workload
    g = binding.from_workload(w, fields=f, device=local)
    g.set_rhs_variant(args.rhs_variant)
    stream = torch.cuda.current_stream()
    g.set_stream(stream.cuda_stream)
    dt = w.cfl / g.max_speed()                         # a7: the library's own CFL reduction
    hbm_gbs, peak_kind = load_peaks()

    # ---- device-resident timing ------------------------------------------------------------------
    sampler = ClockSampler(local) if rank == 0 else None
    t0 = time.time()
    m = measure_resident(g, w, dt, args.steps, args.warmup, stream, barrier, max_over_ranks)
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms_total, launches, timing, stats, finite = m["ms_total"], m["launches"], m["timing"], m["stats"], m["finite"]
    value = world * w.ncells * args.steps / (ms_total * 1e-3)
    variant_used = g.get_rhs_variant()

    # ---- end to end through the C-ABI with host buffers ------------------------------------------
    e2e = None
    if not args.no_e2e:
        pin_in = torch.from_numpy(f["prims"]).pin_memory()
        pin_out = torch.empty_like(pin_in).pin_memory()
        nbytes = pin_in.numel() * 8
        k_e2e = max(1, min(args.steps, args.e2e_steps))
        for _ in range(1):
            g.set_prims(pin_in); g.step(dt, w.recon); g.get_prims(pin_out)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(k_e2e):
            g.set_prims(pin_in)
            g.step(dt, w.recon)
            g.get_prims(pin_out)
        e1.record(stream)
        barrier()
        ms_e2e = max_over_ranks(e0.elapsed_time(e1))
        e2e = {"value": world * w.ncells * k_e2e / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": k_e2e, "ms_per_step": ms_e2e / k_e2e,
               "what": "set_prims(pinned host) + step + get_prims(pinned host) per step"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel ----------------------------------------------------------
    fp64_peak = binding.measure_fp64_peak(local, 5)
    rhs_ms, rhs_n = timing["rhs"]
    rhs_avg_s = rhs_ms * 1e-3 / max(rhs_n, 1)
    flops = RHS_FLOPS[w.recon] * w.ncells
    nbytes_alg = RHS_DOUBLES * 8.0 * w.ncells
    t_alu, t_hbm = flops / (fp64_peak * 1e12), nbytes_alg / (hbm_gbs * 1e9)
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": flops / rhs_avg_s / 1e12, "peak": fp64_peak, "unit": "TFLOP/s",
                "peak_kind": "measured DFMA microbenchmark (rgrmhd_measure_fp64_peak); nominal %.1f" % FP64_NOMINAL_TFLOPS}
    else:
        roof = {"bound": "hbm", "achieved": nbytes_alg / rhs_avg_s / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                "peak_kind": "%s copy bandwidth (MEASURED_PEAKS.json)" % peak_kind}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["kernel"] = roof_kernel(variant_used)          # the kernel rgrmhd_step actually launched (fallbacks included)
    roof["traffic"] = ncu_traffic(roof["kernel"], w.name)
    roof["traffic_source"] = "static: ncu --set full capture of this kernel on this workload (profiles/ncu_traffic.md)"
    roof["avg_launch_ms"] = rhs_avg_s * 1e3
    roof["alg_flops_per_cell"] = RHS_FLOPS[w.recon]
    roof["alg_bytes_per_cell"] = RHS_DOUBLES * 8.0
    roof["hbm_gbs_algorithmic"] = nbytes_alg / rhs_avg_s / 1e9
    step_ms = ms_total / args.steps
    shares = {k: (v[0] / args.steps) / step_ms for k, v in timing.items()}
    roof["share_of_step"] = shares["rhs"]
    step_roof = step_roofline(w, stats, value / world, fp64_peak, hbm_gbs)
    # the oracle's own, instrumented operation count for this config (an upper bound: the oracle recomputes freely)
    oc = oracle_flop_count(args.config)
    if oc is not None:
        f_or = oc["total_flops_per_zone_cycle_recon_once"]
        t_or = max(f_or / (fp64_peak * 1e12), STEP_DOUBLES * 8.0 / (hbm_gbs * 1e9))
        step_roof["oracle_instrumented"] = {
            "flops_per_zone_cycle": f_or, "flops_per_zone_cycle_as_executed": oc["total_flops_per_zone_cycle_oracle"],
            "by_region": oc["flops_per_zone_cycle_by_region"], "frac_if_used": value / world * t_or,
            "note": "python -m oracle.count_flops (counting scalar, FMA = 2, div = sqrt = 1, 32^3 sub-block); the oracle's "
                    "formulas are written for legibility, so this is an upper bound of the algorithmic work and `frac` "
                    "above keeps the smaller hand count"}

    # ---- the other BASELINE configs, same run, same code ---------------------------------------------
    configs = {args.config: {"n": list(w.n), "steps": args.steps, "ms_per_step": step_ms,
                             "zone_cycles_per_s": value / world,
                             "kernel_ms_per_step": {k: v[0] / args.steps for k, v in timing.items()},
                             "step_roofline_frac": step_roof["frac"], "rhs_kernel": roof["kernel"],
                             "c2p_evals_per_solve": step_roof["c2p_evals_per_solve"]}}
    if world == 1 and not args.no_extra_configs:
        g.close()
        del f
        for name in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5"):
            if name == args.config:
                continue
            if name == "cfg5":
                free, _ = torch.cuda.mem_get_info()
                if free < 135e9:
                    configs[name] = {"skipped": "needs 126 GB of device memory, %.0f GB free" % (free / 1e9)}
                    continue
            try:
                configs[name] = measure_extra_config(binding, name, local, stream, fp64_peak, hbm_gbs)
            except Exception as e:  # a failed extra config must not lose the headline line
                configs[name] = {"error": str(e)[:200]}

    cpu = None
    if not args.no_cpu_baseline:
        v, _, sample, _ = time_oracle(w, steps=2, warmup=0, seconds_per_step=args.cpu_seconds / 2.0)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n": list(w.n), "recon": ["minmod", "mc", "weno5"][w.recon],
                       "time": "imex_ssp2_222", "dt": dt, "parallelism": "replicas only x%d" % world,
                       "l2": "inputs larger than L2 (%.0f MB of fields per kernel vs 126 MB)" %
                             (RHS_DOUBLES * 8 * w.ncells / 1e6),
                       "rhs_variant": variant_used},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof,
            "step_roofline": step_roof, "kernel_ms_per_step": {k: v[0] / args.steps for k, v in timing.items()},
            "configs": configs,
            "cpu_baseline": cpu, "finite": finite, "c2p": stats}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0 if finite else 1


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg4", choices=sorted(wl.CONFIGS))
    ap.add_argument("--rhs-variant", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--slabs", action="store_true",
                    help="N > 1 only: cut ONE copy of the workload into N z-slabs with a halo exchange per stage "
                         "(strong scaling) instead of N replicas")
    ap.add_argument("--no-extra-configs", action="store_true",
                    help="skip the `configs` object (the other BASELINE configs measured in the same run)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                     # timing rule: W >= 3
    sys.exit(run_reference(args) if args.impl == "reference" else run_ours(args))


if __name__ == "__main__":
    main()
