#!/usr/bin/env python
"""bench.py -- throughput of the B200 mom_step hot path (libwl) on BASELINE.json's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--repeats R] [--workload C2|C3|C4|C5|N1|N2|N3]
                    [--impl reference] [--no-cpu] [--no-also] [--no-tol] [--stages]

One "step" is one pass of the whole hot path of SURVEY.md 8(a) through the C ABI: wl_step = measure (moving body
only) + mom_step (predictor + corrector, two multigrid projections) + the CFL reduction, on a synthetic BASELINE
config.  The default workload is C4 (torus, 512x256x256 = 33.5 M cells): BASELINE.json quotes
its metric ("ns per cell per time step (3D fp32) and achieved HBM GB/s") and its target (">= 60 % of HBM roofline on
the >= 16 M-cell 3D cases") on the large 3-D cases; C2 (configs[1], 2 M cells) fits in the 126 MB L2 and is reported
under "also" together with C3, C5 and the SURVEY 8(f) workloads (N1: the paper's moving cylinder, 28.3 M cells; N2: its
pulsing jellyfish, a composite non-rigid body, 8.4 M cells; N3: its half-domain Taylor-Green vortex at 512^3, 134 M
cells -- the shape of its 1.57 ns/DOF/step headline).

Protocol: W warm-up steps, then R (default 5) timed blocks of K steps each, every block bracketed by
barrier + synchronize and timed with CUDA events on the simulation's stream; `value` is the MEDIAN block (min and max
are reported beside it).  Fixed two V-cycles per solve (the parity configuration); the tolerance mode (tol = 1e-4) is
timed separately with its mean number of V-cycles per solve.  C3 is timed with the pressure force read every step, as
BASELINE.json states it.

Prints ONE JSON line (rank 0).  Keys: the driver contract (metric/value/unit/n_gpus/steps/warmup/ms_per_step/
higher_is_better/scaling/vs_baseline/dtype/data/config/clocks/e2e/gpu_launches) plus "roofline" (dominant kernel
class, CUDA-event timed inside this run; `traffic` = the ncu DRAM bytes of that kernel from this round's capture,
profiles/r2_ncu_traffic_c4.csv), "cpu_baseline" (the fp64 oracle timed on this box's host cores on the workload
itself), "tolerance_mode" and "also".

Multi-GPU: the path does not shard (BASELINE.json north_star: one GPU, no collectives) =>
"replicas only": every rank runs an independent simulation of the same workload; value = time / (cells x steps x
ranks), time = max over ranks.

--impl reference times the oracle itself (oracle/wl_oracle.c, as it stands) on the host cores, same workload.
--stages launches every fine-level stage once inside a cudaProfilerStart/Stop range (for `ncu --profile-from-start
off --set full`, see profiles/); it prints no JSON line and times nothing.
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

WORKLOADS = {"C2": 1, "C3": 2, "C4": 3, "C5": 4, "N1": 5, "N3": 6, "N2": 7}
NAMES = wi.WORKLOAD_NAMES + ["N1_cylinder_2dof_576x384x128", "N3_tgv_half_512", "N2_jelly_128x128x512"]


def workload_config(k: int, scale: int = 1) -> dict:
    """BASELINE.json configs[k] for k < 5; k = 5, 6, 7: the SURVEY 8(f) NEXT-1 / NEXT-3 / NEXT-2 workloads."""
    if k < 5:
        return wi.baseline_config(k, scale=scale)
    if k == 5:
        return wi.cylinder_2dof(64 // scale)
    if k == 7:
        return wi.jelly(7 - {1: 0, 2: 1, 4: 2}[scale])
    return wi.tgv3d_half(512 // scale)


def is_tgv(cfg) -> bool:
    return cfg["body_kind"] == wi.BODY_NONE and tuple(cfg["U"][:3]) == (0.0, 0.0, 0.0)

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


TRAFFIC_FILE = ROOT / "profiles" / "r2_ncu_traffic_c4.csv"


def ncu_traffic(workload: str) -> dict:
    """{kernel class: DRAM bytes per launch (read + write)} from this round's `ncu --set full` capture of every
    fine-level kernel (profiles/r2_ncu_traffic_c4.md names the command); C4 only, {} when the file is absent."""
    if workload != "C4" or not TRAFFIC_FILE.exists():
        return {}
    out = {}
    for line in TRAFFIC_FILE.read_text().splitlines()[1:]:
        f = line.split(",")
        if len(f) >= 4 and f[0]:
            out[f[0]] = float(f[2]) + float(f[3])
    return out


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
def _oracle_run(k: int, scale: int, nsteps: int, state=None):
    """Advance the oracle `nsteps` steps of workload k at 1/scale linear size; returns (seconds, state)."""
    from oracle import wl_oracle as wo
    if state is None:
        cfg = workload_config(k, scale=scale)
        o = wo.OracleSim(cfg)
        if is_tgv(cfg):
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


def oracle_timed(k: int, warmup: int, steps: int, budget_s: float):
    """The fp64 oracle, as it stands, on workload k ITSELF (full size): `warmup` + `steps` steps.  Only if the first step
    shows that this would take longer than `budget_s` is the same config taken at 1/2 (then 1/4) linear size, and the
    sample says so.  Returns (seconds of the timed steps, steps, scale, cfg of the sample, threads)."""
    from oracle import wl_oracle as wo
    scale = 1
    while True:
        el, state = _oracle_run(k, scale, 1)                  # first step of this size: the warm-up step
        if el * (max(warmup, 1) + steps) <= budget_s or scale >= 4:
            break
        state["o"].close()
        scale *= 2
    if warmup > 1:
        _oracle_run(k, scale, warmup - 1, state)
    el, state = _oracle_run(k, scale, steps, state)
    cfg = state["cfg"]
    state["o"].close()
    return el, steps, scale, cfg, wo.num_threads()


def _sample_text(k, scale, cfg, warmup, steps, el):
    dims = "x".join(map(str, cfg["dims"][: cfg["ndim"]]))
    size = "the workload itself" if scale == 1 else f"the workload at 1/{scale} linear scale (same shape and Re)"
    return (f"{NAMES[k]}: {size}, {dims} = {ncells(cfg)} cells, fp64 oracle as it stands, "
            f"{max(warmup, 1)} warm-up + {steps} timed steps, {el:.1f} s wall")


def oracle_sample(k: int) -> dict:
    """cpu_baseline: 1 warm-up + 3 timed oracle steps of the workload itself (SURVEY 8(d) 'Oracle timed beside it')."""
    el, steps, scale, cfg, threads = oracle_timed(k, 1, 3, budget_s=120.0)
    n = ncells(cfg)
    return {"value": el / steps / n * 1e9, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": _sample_text(k, scale, cfg, 1, steps, el), "same_config": scale == 1,
            "steps": steps, "seconds": el, "cells": n}


def run_reference(args) -> None:
    """The reference arm of this tier is the oracle, as it stands, on the host cores, on the workload itself."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    k = WORKLOADS[args.workload]
    cfg = workload_config(k)
    el, steps, scale, scfg, threads = oracle_timed(k, args.warmup, args.steps, budget_s=400.0)
    n = ncells(scfg)
    val = el / steps / n * 1e9
    sample = _sample_text(k, scale, scfg, args.warmup, steps, el)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": el / steps * 1e3, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg, k, note="oracle timed on: " + sample),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                             "same_config": scale == 1},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def config_dict(cfg, k, note=None) -> dict:
    d = {"workload": NAMES[k], "baseline_config_index": k if k < 5 else None, "dims": list(cfg["dims"][: cfg["ndim"]]),
         "cells": ncells(cfg), "body": ["none", "sphere", "torus", "cylinder", "plane"][cfg["body_kind"]] + ("+%d more" % len(cfg["parts"]) if cfg.get("parts") else ""),
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
    if is_tgv(cfg):
        s.init_tgv(1)
        dt0 = s.cfl()
    else:
        dt0 = cfg["dt0"]
    return s, dt0


def time_steps(torch, sim, dt0, steps, warmup, dist=None, force=False):
    """W untimed + K timed wl_step calls, device-timed with CUDA events on the sim's stream,
    bracketed by barrier + synchronize; returns ms (this rank).  force: the pressure force is read every step."""
    def one(first):
        sim.step(dt0 if first else 0.0, dt0, adaptive=True)
        if force:
            sim.pressure_force()
    for i in range(warmup):
        one(i == 0)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(sim._stream)
    for _ in range(steps):
        one(False)
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


def alg_bytes_table(cfg, prof) -> dict:
    alg = dict(ALG_BYTES)
    alg["conv_diff_bdim"] = conv_alg_bytes(cfg)
    if "pcg_fused" in prof:                           # one-sweep form: every fine-level pcg_matvec launch is a first sweep, r -> e', q
        alg["pcg_matvec"] = 4 * (1 + 2)
        fv = int(cfg.get("fixed_vcycles", 2))
        if fv > 0 and "pcg_update" not in prof:
            # fixed V-cycles: no last sweep on level 0.  The final update of a smoother call is applied by its readers on the fly:
            # between two V-cycles restrict(0) reads q too (+4) and prolong(0) e and q (+8); apply_gradient reads e (+4)
            alg["restrict"] += 4 * (fv - 1) / fv
            alg["prolong"] += 8 * (fv - 1) / fv
            alg["apply_gradient"] += 4
        else:
            alg["pcg_update"] = 4 * (4 + 2)           # tolerance mode: every call ends with x, r, e', q -> x, r
    return alg


def profile_classes(torch, sim, cfg, dt0, steps, hbm_peak, ms_per_step, force=False):
    """The same steps again with every launch bracketed by CUDA events: per-kernel-class times, and the step-level view:
    algorithmic bytes of all fine-level passes per step against the step time."""
    cells = ncells(cfg)
    sim.prof_enable(True)
    ms_prof = time_steps(torch, sim, dt0, steps, 0, None, force=force)
    prof = sim.prof_read()
    sim.prof_enable(False)
    tot = sum(v[0] for v in prof.values())
    alg = alg_bytes_table(cfg, prof)
    kernels = {}
    for name, (ms, n) in sorted(prof.items(), key=lambda kv: -kv[1][0]):
        ent = {"ms_per_step": ms / steps, "launches_per_step": n / steps, "share": ms / tot}
        if alg.get(name):                             # fine-level classes only (".coarse" = multigrid levels >= 1)
            ent["alg_gbs"] = alg[name] * cells * n / (ms * 1e-3) / 1e9
            ent["frac_of_measured_peak"] = ent["alg_gbs"] / hbm_peak
        kernels[name] = ent
    step_bytes = sum((alg.get(nm) or 0) * cells * n for nm, (ms, n) in prof.items() if not nm.endswith(".coarse")) / steps
    gbs = step_bytes / (ms_per_step * 1e-3) / 1e9
    coarse_ms = sum(ms for nm, (ms, n) in prof.items() if nm.endswith(".coarse")) / steps
    step = {"alg_bytes_per_cell_per_step": step_bytes / cells, "achieved_gbs": gbs, "frac_of_measured_peak": gbs / hbm_peak,
            "frac_of_nominal_8TBs": gbs / 8000.0, "levels_ge_1_ms_per_step": coarse_ms, "profiled_ms_per_step": ms_prof / steps}
    return prof, alg, kernels, step


def run_stages(args) -> None:
    """--stages: every fine-level stage of the hot path launched ONCE on the full-size grid inside a cudaProfilerStart/Stop
    range, so that `ncu --profile-from-start off --set full` captures exactly one launch of each kernel (after a few
    warm-up steps, which are not captured)."""
    import torch
    k = WORKLOADS[args.workload]
    cfg = workload_config(k)
    s, dt0 = make_sim(cfg, "cuda:0")
    for i in range(max(args.warmup, 1)):
        s.step(dt0 if i == 0 else 0.0, dt0, adaptive=True)
    dt = s.cfl()
    torch.cuda.synchronize()
    torch.cuda.profiler.start()
    s.measure(1.0)
    s.dbg_save_u0()
    s.dbg_conv_diff_bdim(dt, 0)
    s.dbg_bc()
    if cfg["exit_bc"]:
        s.dbg_exit_bc(dt)
    s.dbg_conv_diff_bdim(dt, 1)
    s.dbg_residual()
    s.dbg_restrict(0)
    s.dbg_prolong(0)
    s.dbg_smooth(0, 3)
    s.dbg_residual()
    s.dbg_apply_gradient()
    s.cfl()
    s.energy()
    if cfg["body_kind"] != wi.BODY_NONE:
        s.pressure_force(1.0)
    torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    s.close()
    print("bench.py --stages: done", file=sys.stderr)


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
    cfg = workload_config(k)
    cells = ncells(cfg)
    force = (k == 2)                                   # BASELINE configs[2]: "pressure force each step"
    sim, dt0 = make_sim(cfg, device)
    peaks = {}
    try:
        peaks = json.load(open(ROOT / "MEASURED_PEAKS.json"))
    except (OSError, ValueError):
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md 6.65 TB/s)"

    # ---- timed region: R blocks of K steps, device-timed, clocks sampled meanwhile
    for i in range(args.warmup):
        sim.step(dt0 if i == 0 else 0.0, dt0, adaptive=True)
        if force:
            sim.pressure_force()
    l1 = sim.stats()["kernel_launches"]
    sampler = ClockSampler(local) if rank == 0 else None
    blocks = [reduce_max(time_steps(torch, sim, dt0, args.steps, 0, dist, force=force)) for _ in range(args.repeats)]
    clocks = sampler.stop() if sampler else None
    l2 = sim.stats()["kernel_launches"]
    ms_med = statistics.median(blocks)
    agg = aggregate(ms_med, cells, args.steps, world)
    dt_now = sim.cfl()
    st = sim.stats()

    prof, alg, kernels, step = profile_classes(torch, sim, cfg, dt0, args.steps, hbm_peak, agg["ms"] / args.steps, force=force)
    if world > 1:
        step["achieved_gbs"] = step["frac_of_measured_peak"] = step["frac_of_nominal_8TBs"] = None
    tot_prof = sum(v[0] for v in prof.values())
    # the dominant kernel with a roofline: the fine-level class that takes the most time
    dom = next((nm for nm in kernels if alg.get(nm)), next(iter(kernels)))
    dom_ms, dom_n = prof[dom]
    achieved = alg[dom] * cells * dom_n / (dom_ms * 1e-3) / 1e9 if alg.get(dom) else None
    traffic = ncu_traffic(args.workload)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
                "frac": (achieved / hbm_peak) if achieved else None, "frac_of_nominal_8TBs": (achieved / 8000.0) if achieved else None,
                "peak_source": peak_src,
                "traffic": traffic.get(dom),
                "traffic_source": "profiles/r2_ncu_traffic_c4.csv (ncu --set full, one launch of every fine-level kernel, this round)"
                                  if traffic.get(dom) else None,
                "traffic_all_kernels": traffic or None,
                "alg_bytes_per_cell_per_launch": alg.get(dom), "avg_launch_us": dom_ms / dom_n * 1e3,
                "share_of_step": dom_ms / tot_prof, "step": step, "kernels": kernels}

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
    torch.cuda.empty_cache()

    # ---- tolerance mode (reported separately, with the mean number of V-cycles per solve)
    tol_mode = None
    if world == 1 and not args.no_tol:
        ct = dict(cfg, fixed_vcycles=0, tol=1e-4, max_vcycles=32)
        s2, d0 = make_sim(ct, device)
        for i in range(args.warmup):
            s2.step(d0 if i == 0 else 0.0, d0, adaptive=True)
        torch.cuda.synchronize()
        nv, res = [], []
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(s2._stream)
        for _ in range(args.steps):
            s2.step(0.0, d0, adaptive=True)
            q = s2.stats()                             # host-side counters: no synchronisation
            nv += q["vcycles"]; res += q["res"]
        e1.record(s2._stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        tol_mode = {"tol": 1e-4, "max_vcycles": 32, "ns_per_cell_step": ms * 1e6 / (cells * args.steps), "ms_per_step": ms / args.steps,
                    "mean_vcycles_per_solve": sum(nv) / len(nv), "max_vcycles_seen": max(nv), "max_residual": max(res),
                    "not_converged": s2.stats()["noconv"],
                    "note": "each V-cycle ends with a host read of max|r| (the only host round trip of the path)"}
        s2.close()
        torch.cuda.empty_cache()

    # ---- the other workloads, one timed block each (rank 0, N = 1 only): BASELINE.md section 3's table
    also = {}
    if world == 1 and not args.no_also:
        for name, kk in WORKLOADS.items():
            if name == args.workload:
                continue
            try:
                c2 = workload_config(kk)
                s2, d0 = make_sim(c2, device)
                nst = args.steps if ncells(c2) < 100e6 else min(args.steps, 10)
                f2 = (kk == 2)
                ms = time_steps(torch, s2, d0, nst, args.warmup, None, force=f2)
                _, _, kern2, step2 = profile_classes(torch, s2, c2, d0, nst, hbm_peak, ms / nst, force=f2)
                top = next(iter(kern2))
                also[NAMES[kk]] = {"cells": ncells(c2), "steps": nst, "ns_per_cell_step": ms * 1e6 / (ncells(c2) * nst),
                                   "ms_per_step": ms / nst, "force_every_step": f2, **step2,
                                   "top_kernel": top, "top_kernel_share": kern2[top]["share"]}
                s2.close()
            except Exception as e:                       # e.g. not enough free memory on a shared box
                also[NAMES[kk]] = {"skipped": str(e)[:120]}
            torch.cuda.empty_cache()

    # ---- scalar types: the tuned fp32 kernels against the generic engine in fp64 and in fp64
    # dual numbers (value + d/d nu through every kernel) on C3 at 1/2 scale; the paper quotes +80 % for Dual over plain
    modes = None
    if world == 1 and not args.no_also:
        modes = {}
        cm = workload_config(2, scale=2)
        for name, extra in (("fp32_tuned", {}), ("fp64_generic", {"precision": 1}), ("tangent_fp64_dual", {"tangent": ("nu", 0)})):
            s2, d0 = make_sim(dict(cm, **extra), device)
            nst = 10
            ms = time_steps(torch, s2, d0, nst, 3, None)
            modes[name] = {"ns_per_cell_step": ms * 1e6 / (ncells(cm) * nst), "ms_per_step": ms / nst}
            s2.close()
            torch.cuda.empty_cache()
        modes["workload"] = "C3 at 1/2 scale (128x64x64)"
        modes["tangent_over_fp64"] = modes["tangent_fp64_dual"]["ms_per_step"] / modes["fp64_generic"]["ms_per_step"]

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    cpu = oracle_sample(k) if (world == 1 and not args.no_cpu) else None
    line = {"metric": METRIC, "value": agg["ns_per_cell_step"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": agg["ms"] / args.steps, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": config_dict(cfg, k, note="replicas only: every rank runs this workload" if world > 1 else None),
            "repeats": {"n": args.repeats, "statistic": "median", "ms_per_step_min": min(blocks) / args.steps,
                        "ms_per_step_median": ms_med / args.steps, "ms_per_step_max": max(blocks) / args.steps},
            "cells_steps_per_s": agg["cells_steps_per_s"], "force_every_step": force,
            "clocks": clocks, "e2e": e2e, "gpu_launches": l2 - l1, "gpu_launches_per_step": (l2 - l1) / (args.steps * args.repeats),
            "vcycles_per_solve": st["vcycles"], "nan_flag": st["nan_flag"], "dt_last": dt_now,
            "roofline": roofline, "cpu_baseline": cpu, "tolerance_mode": tol_mode, "also": also, "scalar_types": modes,
            "context": "paper: 1.57 ns/DOF/step on H100 64GB, fp32, half-domain TGV 512^3 (PAPER.md:143); another machine, not a target"}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--repeats", type=int, default=5, help="timed blocks of --steps steps; the median is reported")
    ap.add_argument("--workload", choices=sorted(WORKLOADS), default="C4")
    ap.add_argument("--impl", choices=["b200", "reference"], default="b200")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--no-also", action="store_true", help="skip the other workloads")
    ap.add_argument("--no-tol", action="store_true", help="skip the tolerance-mode leg")
    ap.add_argument("--stages", action="store_true", help="one launch per fine-level stage inside a profiler range (for ncu); no JSON")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200" and not args.stages:
        print(f"bench.py: warning: --warmup {args.warmup} < 3 (timing rules ask for >= 3)", file=sys.stderr)
    if args.impl == "reference":
        run_reference(args)
    elif args.stages:
        run_stages(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
