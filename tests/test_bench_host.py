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


def test_both_arms_print_the_same_config_object():
    """The reference arm times the oracle on the GPU arm's `config`: one function builds it for both (the driver compares
    the two dicts key by key)."""
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    from paper_2501_11962_b200 import workloads as W
    s = W.config1(n_beads=16)
    a = argparse.Namespace(config=1, parallelism="blocks")
    c = bench.bench_config(a, s, 16, 1, False, 16, s.temperature, 0)
    assert sorted(c) == ["l2", "pair_list", "parallelism", "path", "workload"]
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert src.count('"config": bench_config(') == 2          # run_ours and run_reference


def test_folded_path_is_the_recursion_walked_back_and_forth():
    """workloads.folded_path (bench.py --gpus N, sweep.py): at most 32 recursion steps whatever the path length; every pair
    of neighbouring beads is one recursion step apart; a rank's slice equals the same beads of the whole path."""
    import numpy as np
    from paper_2501_11962_b200 import workloads as W
    s = W.config1(n_beads=16)
    calls = []

    def zero_force(X):
        calls.append(1)
        return np.zeros_like(X)

    R16 = W.folded_path(s, 16, zero_force, seed=3)
    assert np.array_equal(R16, W.brownian_path(s, 16, zero_force, seed=3))
    del calls[:]
    R70 = W.folded_path(s, 70, zero_force, seed=3)
    assert len(calls) == W.MAX_RECURSION_BEADS - 1 and R70.shape == (70, s.n_atoms, 3)
    R32 = W.brownian_path(s, 32, zero_force, seed=3)
    assert np.array_equal(R70[:32], R32) and np.array_equal(R70[32], R32[30]) and np.array_equal(R70[62], R32[0])
    assert np.array_equal(R70[63], R32[1])
    steps = {tuple(sorted((int(np.argmin([np.abs(R32[k] - R70[j]).max() for k in range(32)])),
                           int(np.argmin([np.abs(R32[k] - R70[j + 1]).max() for k in range(32)]))))) for j in range(69)}
    assert all(b - a == 1 for a, b in steps)
    assert np.array_equal(W.folded_path(s, 70, zero_force, seed=3, first=56), R70[56:])
    assert W.folded_path(s, 1, zero_force, seed=3).shape == (1, s.n_atoms, 3)
