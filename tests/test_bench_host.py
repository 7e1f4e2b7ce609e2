"""Host-side logic of bench.py (no GPU): replicas-only aggregation over ranks with a world_size-2
gloo group, the algorithmic-byte table, and the reference arm's JSON line."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
def reduce_max(x):
    t = torch.tensor([x], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
ms_local = 10.0 * (rank + 1)            # rank 1 is the slow one
agg = bench.aggregate(ms_local, cells=1000, steps=4, world=world, reduce_max=reduce_max)
dist.barrier()
if rank == 0:
    print(json.dumps(agg))
dist.destroy_process_group()
"""


def test_replica_aggregation_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=str(ROOT)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29611", str(script)],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    agg = json.loads(line)
    assert agg["ms"] == pytest.approx(20.0)                       # max over ranks
    assert agg["ns_per_cell_step"] == pytest.approx(20.0e6 / (1000 * 4 * 2))
    assert agg["cells_steps_per_s"] == pytest.approx(1000 * 4 * 2 / 20.0e-3)


def test_aggregate_single_rank():
    sys.path.insert(0, str(ROOT))
    import bench
    agg = bench.aggregate(5.0, cells=100, steps=2, world=1)
    assert agg["ms"] == 5.0 and agg["ns_per_cell_step"] == pytest.approx(5.0e6 / 200)


def test_alg_bytes_table_matches_design():
    """DESIGN.md section 6 and bench.ALG_BYTES state the same per-cell figures."""
    sys.path.insert(0, str(ROOT))
    import bench
    import wl_inputs as wi
    assert bench.ALG_BYTES["pcg_matvec"] == 16 and bench.ALG_BYTES["pcg_update"] == 24 and bench.ALG_BYTES["pcg_fused"] == 32
    assert bench.ALG_BYTES["residual"] == 24 and bench.ALG_BYTES["apply_gradient"] == 32
    assert bench.conv_alg_bytes(wi.baseline_config(3)) == (36 + 48) / 2
    text = (ROOT / "DESIGN.md").read_text()
    for tok in ("| `pcg_matvec` (pass A) | e, r → e′, q | 16 |", "| `pcg_update` (pass B) | x, r, e′, q → x, r | 24 |",
                "| `pcg_fused` (one-sweep iteration, §6.2) | x, r, e, q → x, r′, e′, q′ | 32 |", "| `apply_gradient` |"):
        assert tok in text


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1",
                          "--workload", "C2"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "ns/cell/step" and line["higher_is_better"] is False
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
    # the reference arm times the workload itself (C2: 128^3), not a scaled sample
    assert line["cpu_baseline"]["same_config"] is True and line["config"]["cells"] == 128 ** 3
    assert "128x128x128" in line["cpu_baseline"]["sample"]


def test_traffic_table_is_read_from_profiles():
    """roofline.traffic comes from the committed ncu summary of this round, not from constants in bench.py"""
    sys.path.insert(0, str(ROOT))
    import bench
    assert "NCU_TRAFFIC" not in (ROOT / "bench.py").read_text()
    t = bench.ncu_traffic("C4")
    if bench.TRAFFIC_FILE.exists():
        assert t and all(v > 0 for v in t.values()) and "pcg_fused" in t
    assert bench.ncu_traffic("C3") == {}


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1"],
                         capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
