"""Launch every fine-level stage of the hot path once, inside a cudaProfilerStart/Stop range, so that
`ncu --profile-from-start off --set full` captures exactly one launch of each kernel on the full-size
grid (no warm-up launches, no coarse multigrid levels unless asked).

    python -m paper_2407_16032_b200.profile_stages [--workload C4] [--warm 3] [--coarse]

Used only to produce the ncu summaries under profiles/; bench.py does the timing.
"""
from __future__ import annotations

import argparse
import sys
from pathlib import Path

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))

import wl_inputs as wi  # noqa: E402


def main():
    import torch
    from paper_2407_16032_b200 import wl

    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="C4", choices=["C2", "C3", "C4", "C5"])
    ap.add_argument("--warm", type=int, default=3)
    ap.add_argument("--coarse", action="store_true", help="also launch the level-1 smoother once")
    ap.add_argument("--steps", type=int, default=0, help="instead of single stages, profile this many whole steps")
    a = ap.parse_args()
    k = {"C2": 1, "C3": 2, "C4": 3, "C5": 4}[a.workload]
    cfg = wi.baseline_config(k)
    s = wl.Sim(cfg)
    if cfg["body_kind"] == wi.BODY_NONE:
        s.init_tgv(1)
        dt0 = s.cfl()
    else:
        dt0 = cfg["dt0"]
    for i in range(a.warm):
        s.step(dt0 if i == 0 else 0.0, dt0, adaptive=True)
    dt = s.cfl()
    torch.cuda.synchronize()
    torch.cuda.profiler.start()
    if a.steps:
        for _ in range(a.steps):
            s.step(0.0, dt0, adaptive=True)
    else:
        s.measure(1.0)
        s.dbg_save_u0()
        s.dbg_conv_diff_bdim(dt, 0)
        s.dbg_bc()
        if cfg["exit_bc"]:
            s.dbg_exit_bc(dt)
        s.dbg_conv_diff_bdim(dt, 1)
        s.dbg_residual()
        s.dbg_restrict(0)
        if a.coarse:
            s.dbg_smooth(1, 2)
        s.dbg_prolong(0)
        s.dbg_smooth(0, 3)
        s.dbg_residual()
        s.dbg_apply_gradient()
        s.cfl()
        if cfg["body_kind"] != wi.BODY_NONE:
            s.pressure_force(1.0)
    torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    s.close()
    print("profile_stages: done")


if __name__ == "__main__":
    main()
