"""Host logic of bench.py that needs no GPU: the multi-rank aggregation (max time over ranks, sum of units) under
torch.distributed/gloo with world_size 2, the roofline denominator, and the reference-arm contract keys."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ms, units = bench.all_reduce_max_sum(100.0 * (rank + 1), 8.0 * 5, world)
dist.barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "units": units, "value": bench.throughput(units, ms)}))
dist.destroy_process_group()
"""


def test_replica_aggregation_world_size_2_gloo(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER % ROOT)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29547", str(w)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    out = json.loads(line)
    assert out["ms"] == 200.0           # max over ranks
    assert out["units"] == 80.0         # both replicas' bead evaluations
    assert out["value"] == pytest.approx(80.0 / 0.2)


def test_single_rank_aggregation_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.all_reduce_max_sum(12.5, 40.0, 1) == (12.5, 40.0)
    assert bench.fp32_peak_tflops(1965.0) == pytest.approx(74.45, abs=0.05)


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, timeout=120, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_roofline_traffic_comes_from_the_committed_ncu_capture():
    """roofline.traffic is read from profiles/ (the ncu capture of the S5 launch), not typed into bench.py."""
    sys.path.insert(0, ROOT)
    import bench
    traffic, src = bench.traffic_bytes_per_launch()
    assert src == bench.NCU_METRICS_FILE and os.path.exists(os.path.join(ROOT, src))
    vals = dict(l.strip().split(",") for l in open(os.path.join(ROOT, src)) if not l.startswith("#"))
    assert traffic == float(vals["dram__bytes_read.sum"]) + float(vals["dram__bytes_write.sum"])
    assert 1.0e7 < traffic < 1.0e10          # bytes per launch: tens to hundreds of MB
