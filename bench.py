#!/usr/bin/env python
"""bench.py -- throughput of the B200 mom_step hot path (libwl) on BASELINE.json's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2|C3|C4|C5] [--impl reference]

One "step" is one pass of the whole hot path of SURVEY.md 8(a) through the C ABI: wl_step =
measure (moving body only) + mom_step (predictor + corrector, two multigrid projections) + the
CFL reduction, on a synthetic BASELINE config.  The default workload is
C4 (torus, 512x256x256 = 33.5 M cells): BASELINE.json quotes its metric ("ns per cell per time
step (3D fp32) and achieved HBM GB/s") and its target (">= 60 % of HBM roofline on the >= 16 M-cell
3D cases") on the large 3-D cases; C2 (configs[1], 2 M cells) fits in the 126 MB L2 and is reported
under "also" together with C3 and C5.

Prints ONE JSON line (rank 0).  Keys: the driver contract (metric/value/unit/n_gpus/steps/warmup/
ms_per_step/higher_is_better/scaling/vs_baseline/dtype/data/config/clocks/e2e/gpu_launches) plus
"roofline" (dominant kernel class, CUDA-event timed inside this run) and "cpu_baseline" (the fp64
oracle timed on this box's host cores on a bounded sample).

Multi-GPU: the path does not shard (BASELINE.json north_star: one GPU, no collectives; DESIGN.md
section 9) => "replicas only": every rank runs an independent simulation of the same workload;
value = time / (cells x steps x ranks), time = max over ranks.

--impl reference times the oracle itself (oracle/wl_oracle.c, as it stands) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import wl_inputs as wi  # noqa: E402

WORKLOADS = {"C2": 1, "C3": 2, "C4": 3, "C5": 4}
METRIC = "ns per cell per time step (3D fp32)"
UNIT = "ns/cell/step"

# Algorithmic bytes per fine-grid cell of each kernel class (fp32, every array read/written once
# per pass, halos ignored) ON BODY-FREE TILES, where face coefficients and 1/D are analytic and not
# loaded: DESIGN.md section 6 restates SURVEY.md 8(d)'s table for the kernels as they are fused in
# libwl.  These are the smallest counts (tiles cut by a body also read L and iD), so the achieved
# GB/s computed from them is a lower bound.
ALG_BYTES = {
    "conv_diff_bdim": None,   # mean of predictor and corrector: computed below
    "residual": 4 * (3 + 1 + 2),            # u, p -> x, r
    "pcg_matvec": 4 * (2 + 2),              # pass A: e, r -> e', q (first iteration: r -> e', q)
    "pcg_update": 4 * (4 + 2),              # pass B / the last sweep of the one-sweep form: x, r, e', q -> x, r
    "pcg_fused": 4 * (4 + 4),               # one-sweep iteration (wl_pcgfused.cu): x, r, e, q -> x, r', e', q'
    "restrict": 4 * (1 + 2 / 8),            # r -> r_c, x_c
    "prolong": 4 * (2 + 1 / 8 + 2),         # x, r, x_c -> x, r
    "apply_gradient": 4 * (3 + 1 + 3 + 1),  # u, x -> u, p
    "cfl": 4 * 3,
    "measure": 4 * (3 + 9),
}


# DRAM traffic per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the fine-level kernels on C4, from the
# ncu --set full captures summarised in profiles/r1c_stages_c4_ncu.md and (pcg_fused) profiles/r1e_pcg_fused_c4_ncu.md
# (bytes; other workloads: not captured)
NCU_TRAFFIC_C4 = {"pcg_fused": 1200e6, "pcg_update": 793e6, "pcg_matvec": 593e6, "residual": 882e6, "prolong": 577e6,
                  "apply_gradient": 1088e6, "cfl": 420e6, "restrict": 160e6, "conv_diff_bdim": 1430e6}


def conv_alg_bytes(cfg) -> float:
    """conv_diff+BDIM tile kernel, mean of the predictor (w, mu0 -> u) and corrector (w, u0, mu0 -> u)
    passes; mu1 is read only on the band list (k_cd_band), V is three scalars."""
    return 4 * ((3 + 3 + 3) + (3 + 3 + 3 + 3)) / 2


def ncells(cfg) -> int:
    n = 1
    for d in cfg["dims"][: cfg["ndim"]]:
        n *= int(d)
    return n


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.strip().lower() == "active":
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------- oracle legs
def oracle_sample(cfg_full: dict, k: int, budget_s: float = 15.0) -> dict:
    """Time the fp64 oracle (as it stands) on a bounded sample of workload k: the same config at
    half the linear size (same shape, same Reynolds number), 1 warm-up + n timed steps."""
    from oracle import wl_oracle as wo
    cfg = wi.baseline_config(k, scale=2)
    n = ncells(cfg)
    o = wo.OracleSim(cfg)
    moving = cfg["motion"] != wi.MOTION_STATIC
    if cfg["body_kind"] == wi.BODY_NONE:
        o.init_tgv(1)
        dt = o.cfl()
    else:
        dt = cfg["dt0"]
    t = 0.0

    def one(dt, t):
        if moving:
            o.measure(t + dt)
        o.mom_step(dt)
        return o.cfl(), t + dt

    t0 = time.perf_counter()
    dt, t = one(dt, t)
    first = time.perf_counter() - t0
    steps = max(1, min(20, int(budget_s / max(first, 1e-3)) - 1))
    t0 = time.perf_counter()
    for _ in range(steps):
        dt, t = one(dt, t)
    el = time.perf_counter() - t0
    threads = wo.num_threads()
    o.close()
    return {"value": el / steps / n * 1e9, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{wi.WORKLOAD_NAMES[k]} at 1/2 linear scale ({'x'.join(map(str, cfg['dims']))} = {n} cells, "
                      f"same shape and Re), fp64, 1 warm-up + {steps} timed steps, {el:.1f} s wall",
            "steps": steps, "seconds": el, "cells": n}


def _oracle_run(k: int, scale: int, nsteps: int, state=None):
    """Advance the oracle `nsteps` steps of workload k at 1/scale linear size; returns (seconds, state)."""
    from oracle import wl_oracle as wo
    if state is None:
        cfg = wi.baseline_config(k, scale=scale)
        o = wo.OracleSim(cfg)
        if cfg["body_kind"] == wi.BODY_NONE:
            o.init_tgv(1)
            dt = o.cfl()
        else:
            dt = cfg["dt0"]
        state = {"o": o, "cfg": cfg, "dt": dt, "t": 0.0}
    o, cfg = state["o"], state["cfg"]
    moving = cfg["motion"] != wi.MOTION_STATIC
    t0 = time.perf_counter()
    for _ in range(nsteps):
        if moving:
            o.measure(state["t"] + state["dt"])
        o.mom_step(state["dt"])
        state["t"] += state["dt"]
        state["dt"] = o.cfl()
    return time.perf_counter() - t0, state


def run_reference(args) -> None:
    """The reference arm of this tier is the oracle, as it stands, on the host cores.  A step is
    one oracle time step on a bounded sample of the workload: the same config at 1/scale linear
    size, scale chosen (2, 4 or 8) so that W + K steps end within a few minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import wl_oracle as wo
    k = WORKLOADS[args.workload]
    cfg = wi.baseline_config(k)
    total = args.warmup + args.steps
    scale, state, warm_done = 2, None, 0
    while True:
        el, state = _oracle_run(k, scale, 1)            # first step of this sample size (counts as warm-up)
        warm_done = 1
        if el * total <= 200.0 or scale >= 8:
            break
        state["o"].close()
        scale, state = scale * 2, None
    if args.warmup > warm_done:
        _oracle_run(k, scale, args.warmup - warm_done, state)
    el, state = _oracle_run(k, scale, args.steps, state)
    scfg = state["cfg"]
    n = ncells(scfg)
    state["o"].close()
    val = el / args.steps / n * 1e9
    threads = wo.num_threads()
    sample = (f"{wi.WORKLOAD_NAMES[k]} at 1/{scale} linear scale ({'x'.join(map(str, scfg['dims'][:scfg['ndim']]))} = {n} cells, "
              f"same shape and Re), fp64 oracle, {max(args.warmup, warm_done)} warm-up + {args.steps} timed steps, {el:.1f} s wall")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg, args.workload, k, note="oracle timed on a bounded sample: " + sample),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def config_dict(cfg, wl_name, k, note=None) -> dict:
    d = {"workload": wi.WORKLOAD_NAMES[k], "baseline_config_index": k, "dims": list(cfg["dims"][: cfg["ndim"]]),
         "cells": ncells(cfg), "body": ["none", "sphere", "torus"][cfg["body_kind"]],
         "moving_body": bool(cfg["motion"]), "nu": cfg["nu"], "dt": "CFL-adaptive, device-resident",
         "mg": {"fixed_vcycles": cfg["fixed_vcycles"], "smooth_iters": cfg["smooth_iters"]},
         "l2": "working set (>= 3 GB for C4/C5) is far larger than the 126 MB L2; no flush needed between steps"}
    if note:
        d["note"] = note
    return d


# ----------------------------------------------------------------------------- GPU arm
def make_sim(cfg, device):
    from paper_2407_16032_b200 import wl
    s = wl.Sim(cfg, device=device)
    if cfg["body_kind"] == wi.BODY_NONE and all(cfg["periodic"][: cfg["ndim"]]):
        s.init_tgv(1)
        dt0 = s.cfl()
    else:
        dt0 = cfg["dt0"]
    return s, dt0


def time_steps(torch, sim, dt0, steps, warmup, dist=None):
    """W untimed + K timed wl_step calls, device-timed with CUDA events on the sim's stream,
    bracketed by barrier + synchronize; returns ms (this rank)."""
    for i in range(warmup):
        sim.step(dt0 if i == 0 else 0.0, dt0, adaptive=True)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(sim._stream)
    for _ in range(steps):
        sim.step(0.0, dt0, adaptive=True)
    e1.record(sim._stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    return e0.elapsed_time(e1)


def aggregate(ms_local: float, cells: int, steps: int, world: int, reduce_max=None) -> dict:
    """Replicas-only aggregation: time = max over ranks; value = time / (cells*steps*world)."""
    ms = reduce_max(ms_local) if reduce_max is not None else ms_local
    total = cells * steps * world
    return {"ms": ms, "ns_per_cell_step": ms * 1e6 / total, "cells_steps_per_s": total / (ms * 1e-3)}


def run_gpu(args) -> None:
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libwl has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=torch.device(device))
        dist = dist_mod

    def reduce_max(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    k = WORKLOADS[args.workload]
    cfg = wi.baseline_config(k)
    cells = ncells(cfg)
    sim, dt0 = make_sim(cfg, device)
    peaks = {}
    try:
        peaks = json.load(open(ROOT / "MEASURED_PEAKS.json"))
    except (OSError, ValueError):
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md 6.65 TB/s)"

    # ---- timed region: K steps, device-timed, clocks sampled meanwhile
    l0 = sim.stats()["kernel_launches"]
    for i in range(args.warmup):
        sim.step(dt0 if i == 0 else 0.0, dt0, adaptive=True)
    l1 = sim.stats()["kernel_launches"]
    sampler = ClockSampler(local) if rank == 0 else None
    ms_local = time_steps(torch, sim, dt0, args.steps, 0, dist)
    clocks = sampler.stop() if sampler else None
    l2 = sim.stats()["kernel_launches"]
    agg = aggregate(ms_local, cells, args.steps, world, reduce_max)
    dt_now = sim.cfl()
    st = sim.stats()

    # ---- same K steps again with every launch bracketed by CUDA events: per-kernel-class times
    sim.prof_enable(True)
    ms_prof = time_steps(torch, sim, dt0, args.steps, 0, None)
    prof = sim.prof_read()
    sim.prof_enable(False)
    tot_prof = sum(v[0] for v in prof.values())
    alg = dict(ALG_BYTES)
    alg["conv_diff_bdim"] = conv_alg_bytes(cfg)
    if "pcg_fused" in prof:                           # one-sweep form: every fine-level pcg_matvec launch is a first sweep, r -> e', q
        alg["pcg_matvec"] = 4 * (1 + 2)
        # ... and of the two last sweeps of a solve (fixed two V-cycles) the second leaves r alone (x, e' -> x): mean of 24 and 12
        alg["pcg_update"] = (4 * (4 + 2) + 4 * (2 + 1)) / 2
    breakdown = {}
    for name, (ms, n) in sorted(prof.items(), key=lambda kv: -kv[1][0]):
        ent = {"ms_per_step": ms / args.steps, "launches_per_step": n / args.steps, "share": ms / tot_prof}
        if name in alg and alg[name]:                 # fine-level classes only (".coarse" = multigrid levels >= 1)
            ent["alg_gbs"] = alg[name] * cells * n / (ms * 1e-3) / 1e9
        breakdown[name] = ent
    # the dominant kernel with a roofline: the fine-level class that takes the most time
    dom = next((nm for nm in breakdown if alg.get(nm)), next(iter(breakdown)))
    dom_ms, dom_n = prof[dom]
    base = dom.split(".")[0]
    achieved = (alg.get(base) or 0) * cells * dom_n / (dom_ms * 1e-3) / 1e9 if not dom.endswith(".coarse") else None
    # step-level view: algorithmic bytes of all fine-level passes / step time
    step_bytes = sum((alg.get(nm) or 0) * cells * n for nm, (ms, n) in prof.items() if not nm.endswith(".coarse")) / args.steps
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
                "frac": (achieved / hbm_peak) if achieved else None, "frac_of_nominal_8TBs": (achieved / 8000.0) if achieved else None,
                "peak_source": peak_src,
                "traffic": NCU_TRAFFIC_C4.get(base) if args.workload == "C4" else None,
                "traffic_source": (("profiles/r1e_pcg_fused_c4_ncu.md" if base == "pcg_fused" else "profiles/r1c_stages_c4_ncu.md")
                                   + " (ncu --set full, one launch)") if args.workload == "C4" else None,
                "alg_bytes_per_cell_per_launch": alg.get(base), "avg_launch_us": dom_ms / dom_n * 1e3,
                "share_of_step": dom_ms / tot_prof,
                "step": {"alg_bytes_per_cell_per_step": step_bytes / cells,
                         "achieved_gbs": step_bytes / (agg["ms"] / args.steps * 1e-3) / 1e9 if world == 1 else None,
                         "frac": step_bytes / (agg["ms"] / args.steps * 1e-3) / 1e9 / hbm_peak if world == 1 else None},
                "profiled_ms_per_step": ms_prof / args.steps,
                "kernels": breakdown}

    # ---- end to end through the C ABI with HOST buffers: set_fields(host) + step + get_fields(host)
    e2e_steps = max(1, min(args.steps, 5))
    nd = cfg["ndim"]
    hu = torch.empty((nd,) + tuple(reversed(cfg["dims"][:nd])), dtype=torch.float32).pin_memory()
    hp = torch.empty(tuple(reversed(cfg["dims"][:nd])), dtype=torch.float32).pin_memory()
    sim.get_fields(u=hu, p=hp)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    t_e2e = 1.0e3
    for _ in range(e2e_steps):
        t_e2e += dt_now
        sim.set_fields(u=hu, p=hp)
        sim.step(t_e2e, dt_now, adaptive=False)
        sim.get_fields(u=hu, p=hp)
    torch.cuda.synchronize()
    e2e_ms = reduce_max((time.perf_counter() - t0) * 1e3)
    nbytes = (nd + 1) * cells * 4
    e2e = {"value": e2e_ms * 1e6 / (cells * e2e_steps * world), "unit": UNIT, "h2d_bytes_per_step": nbytes,
           "d2h_bytes_per_step": nbytes, "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
           "call": "wl_set_fields(host u,p) + wl_step + wl_get_fields(host u,p), pinned host memory, wall clock"}
    sim.close()
    del hu, hp

    # ---- the other 3-D BASELINE workloads, short runs (rank 0, N = 1 only)
    also = {}
    if world == 1 and not args.no_also:
        for name, kk in WORKLOADS.items():
            if name == args.workload:
                continue
            c2 = wi.baseline_config(kk)
            s2, d0 = make_sim(c2, device)
            ms = time_steps(torch, s2, d0, args.steps, args.warmup, None)
            also[wi.WORKLOAD_NAMES[kk]] = {"cells": ncells(c2), "ns_per_cell_step": ms * 1e6 / (ncells(c2) * args.steps),
                                           "ms_per_step": ms / args.steps}
            s2.close()
            torch.cuda.empty_cache()
        # the shape of the paper's headline figure (TGV 512^3, 134 M cells; here fully periodic and with
        # the fixed two V-cycles of the BASELINE configs): context beside the paper's 1.57 ns on an H100, not a config
        try:
            c2 = wi.tgv3d(512)
            s2, d0 = make_sim(c2, device)
            ms = time_steps(torch, s2, d0, min(args.steps, 10), 3, None)
            also["TGV3D_512_paper_headline_shape"] = {"cells": ncells(c2), "ns_per_cell_step": ms * 1e6 / (ncells(c2) * min(args.steps, 10)),
                                                      "ms_per_step": ms / min(args.steps, 10)}
            s2.close()
        except Exception as e:                       # not enough free memory on a shared box: skip the context line
            also["TGV3D_512_paper_headline_shape"] = {"skipped": str(e)[:120]}
        torch.cuda.empty_cache()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    cpu = oracle_sample(cfg, k) if (world == 1 and not args.no_cpu) else None
    line = {"metric": METRIC, "value": agg["ns_per_cell_step"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": agg["ms"] / args.steps, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": config_dict(cfg, args.workload, k, note="replicas only: every rank runs this workload" if world > 1 else None),
            "cells_steps_per_s": agg["cells_steps_per_s"],
            "clocks": clocks, "e2e": e2e, "gpu_launches": l2 - l1, "gpu_launches_per_step": (l2 - l1) / args.steps,
            "vcycles_per_solve": st["vcycles"], "nan_flag": st["nan_flag"], "dt_last": dt_now,
            "roofline": roofline, "cpu_baseline": cpu, "also": also,
            "context": "paper: 1.57 ns/DOF/step on H100 64GB, fp32, TGV 512^3 (PAPER.md:143); another machine and workload, not a target"}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", choices=sorted(WORKLOADS), default="C4")
    ap.add_argument("--impl", choices=["b200", "reference"], default="b200")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--no-also", action="store_true", help="skip the other workloads")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        print(f"bench.py: warning: --warmup {args.warmup} < 3 (timing rules ask for >= 3)", file=sys.stderr)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
