"""Bead-block sharding, host side: the exchange logic of paper_2501_11962_b200/blocks.py under
torch.distributed/gloo on CPU tensors with world sizes 2 and 3 -- the same code moves CUDA tensors over NCCL.  The engine
here is a stand-in with the three block calls (a free polymer with a harmonic well on bead 1, in torch), so that every
rank's gradient block and the reduced V_eff can be checked against the closed form of the whole path."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch
import torch.distributed as dist
from paper_2501_11962_b200 import blocks

K, KW, Q, NPATH = 3.0, 0.7, 5, 7

class ToyEngine:
    # V = KW/2 |R^1|^2 + sum_n K/2 |R^{n+1} - R^n|^2  (eta^n = R^{n+1} - R^n: no physical force, H = 0)
    def __init__(self, first, n, npath):
        self.first, self.n, self.npath = first, n, npath
        self.nh = min(n, npath - 1 - first)
    def mop_block_pass1(self, R, R_right, keta_out):
        nxt = torch.cat([R[1:], R_right[None]]) if R_right is not None else R[1:]
        self.eta = nxt[:self.nh] - R[:self.nh]
        self.R = R
        if keta_out is not None:
            keta_out.copy_(K * self.eta[self.nh - 1])
    def mop_block_pass2(self, R):
        pass
    def mop_get_stats(self):
        return {"veff": self.v}
    def mop_block_assemble(self, keta_left, grad_out, sync=True):
        g = torch.zeros_like(self.R)
        g[:self.nh] -= K * self.eta
        g[1:self.nh + 1 if self.nh < self.n else self.n] += K * self.eta[:self.n - 1]
        if keta_left is not None:
            g[0] += keta_left
        v = 0.5 * K * float((self.eta ** 2).sum())
        if self.first == 0:
            g[0] += KW * self.R[0]
            v += 0.5 * KW * float((self.R[0] ** 2).sum())
        self.v = v
        return (v if sync else None), g

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
torch.manual_seed(0)
R = torch.randn(NPATH, Q, 3, dtype=torch.float64)          # the same path on every rank
first, n = blocks.partition(NPATH, world)[rank]
bp = blocks.BlockPath(ToyEngine(first, n, NPATH), Q, first, n, NPATH, dtype=torch.float64)
v, g = bp.eval(R[first:first + n].clone())
# closed form of the whole path
d = R[1:] - R[:-1]
G = torch.zeros_like(R)
G[:-1] -= K * d
G[1:] += K * d
G[0] += KW * R[0]
V = 0.5 * K * float((d ** 2).sum()) + 0.5 * KW * float((R[0] ** 2).sum())
err = float((g - G[first:first + n]).abs().max())
# the stepping form: no V_eff per evaluation (the assembly stays asynchronous), the energy read once afterwards
v2, g2 = bp.eval(R[first:first + n].clone(), sync=False)
assert v2 is None and float((g2 - g).abs().max()) == 0.0
out = torch.tensor([err, max(abs(v - V), abs(bp.veff() - V))], dtype=torch.float64)
dist.all_reduce(out, op=dist.ReduceOp.MAX)
if rank == 0:
    print(json.dumps({"grad_err": float(out[0]), "veff_err": float(out[1]), "world": world, "V": V}))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,port", [(2, 29551), (3, 29553)])
def test_block_exchange_gloo(tmp_path, world, port):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER % ROOT)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world), "--master-addr",
           "127.0.0.1", "--master-port", str(port), str(w)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-3000:]
    out = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    assert out["world"] == world
    assert out["grad_err"] < 1e-12 and out["veff_err"] < 1e-10 * abs(out["V"])


def test_partition():
    sys.path.insert(0, ROOT)
    from paper_2501_11962_b200 import blocks
    assert blocks.partition(8, 2) == [(0, 4), (4, 4)]
    assert blocks.partition(7, 3) == [(0, 3), (3, 2), (5, 2)]
    assert blocks.partition(8, 8) == [(k, 1) for k in range(8)]
    assert blocks.partition(64, 1) == [(0, 64)]
    with pytest.raises(ValueError):
        blocks.partition(3, 4)
