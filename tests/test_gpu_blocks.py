"""Bead-block mode on the GPU (mop.h "bead-block mode"): several contexts on ONE device, each
owning a contiguous block of beads of the same path, the halos handed over directly (no process group: the exchange
itself is covered by tests/test_blocks_host.py under gloo), must reproduce the whole-path evaluation -- V_eff to 1e-8
and the gradient to 1e-6 RMS (same kernels, same lists; only the order of the float atomics that build F differs, which
moves E_spring by ~1e-9 of itself from one run to the next: two evaluations by ONE context differ as much) -- and the oracle at
the usual bars.  Unmeasured on more than one GPU: this run has a single B200."""
import numpy as np
import pytest

from paper_2501_11962_b200 import blocks
from paper_2501_11962_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device: the library has no CPU fallback")
    from paper_2501_11962_b200 import binding
    binding.load()
    return binding


def run_blocks(B, s, R, parts):
    """Evaluate the path R [N][Q][3] with one context per (first, n) in parts; returns (V_eff, grad [N][Q][3])."""
    import torch
    N = R.shape[0]
    Rg = torch.tensor(R, device="cuda")
    ctx = [B.Mop(s, n, block=(f, N)) for f, n in parts]
    keta = [torch.zeros((s.n_atoms, 3), device="cuda") for _ in parts]
    for k, (f, n) in enumerate(parts):
        last = f + n == N
        ctx[k].mop_block_pass1(Rg[f:f + n], None if last else Rg[f + n].contiguous(), None if last else keta[k])
    for k, (f, n) in enumerate(parts):
        ctx[k].mop_block_pass2(Rg[f:f + n])
    v, g = 0.0, []
    for k, (f, n) in enumerate(parts):
        vk, gk = ctx[k].mop_block_assemble(None if k == 0 else keta[k - 1])
        v += vk
        g.append(gk.cpu().numpy())
    for c in ctx:
        c.close()
    return v, np.concatenate(g, 0)


@pytest.mark.parametrize("name,parts", [("c2", [(0, 4), (4, 4)]), ("c2", [(0, 3), (3, 4), (7, 1)]), ("c2", [(k, 1) for k in range(8)]),
                                        ("chain", [(0, 1), (1, 5)]), ("c1", [(0, 16)])])
def test_blocks_reproduce_the_whole_path(B, oracle, name, parts):
    if name == "c1":
        s = W.config1(n_beads=16)
    elif name == "c2":
        s = W.config2(n_beads=8)
    else:
        s = H.tiny_chain()
        s.n_beads = 6
    o = oracle.OracleSystem(s)
    R = W.brownian_path(s, s.n_beads, lambda X: oracle.bead(o, X, geom=0)["F"], seed=0)
    m = B.Mop(s, s.n_beads)
    v0, g0 = m.mop_eval_veff_grad(R)
    m.close()
    v, g = run_blocks(B, s, R, parts)
    assert abs(v - v0) <= 1e-8 * abs(v0)
    assert H.rms_rel(g, g0.cpu().numpy()) <= 1e-6
    v_ref, g_ref = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=s.n_atoms <= 3000)
    assert abs(v - v_ref) <= 1e-6 * abs(v_ref)
    H.assert_close(g, g_ref, 1e-4)


def test_block_context_rules_and_integrator(B, oracle):
    import torch
    s = W.config1(n_beads=4)
    o = oracle.OracleSystem(s)
    R = W.brownian_path(s, 4, lambda X: oracle.bead(o, X, geom=0)["F"], seed=0)
    Rg = torch.tensor(R, device="cuda")
    a = B.Mop(s, 2, block=(0, 4))
    with pytest.raises(B.MopError) as e:              # a partial block refuses the whole-path call
        a.mop_eval_veff_grad(Rg[:2])
    assert e.value.status == 1
    with pytest.raises(B.MopError):                   # pass 2 before pass 1
        a.mop_block_pass2(Rg[:2])
    with pytest.raises(B.MopError):                   # not the last block: the right halo is required
        a.mop_block_pass1(Rg[:2])
    with pytest.raises(B.MopError):                   # block outside the path
        B.Mop(s, 3, block=(2, 4))
    with pytest.raises(B.MopError) as e:              # no block context takes a bias (mop.h) ...
        a.mop_set_bias([0], [1], 0.01, 1.0)
    assert e.value.status == 1
    a.close()
    # a block that is the whole path takes the whole-path calls
    w = B.Mop(s, 4, block=(0, 4))
    with pytest.raises(B.MopError) as e:              # ... the one that holds the whole path included: mop_block_assemble
        w.mop_set_bias([0], [1], 0.01, 1.0)           # has no coordinates to form the CV from
    assert e.value.status == 1 and "bias" in str(e.value)
    m = B.Mop(s, 4)
    v1, g1 = w.mop_eval_veff_grad(Rg)
    v0, g0 = m.mop_eval_veff_grad(Rg)
    assert abs(v1 - v0) <= 1e-8 * abs(v0) and H.rms_rel(g1.cpu().numpy(), g0.cpu().numpy()) <= 1e-6
    # one velocity-Verlet step from the block integrator = mop_step(.., 1)
    rng = np.random.default_rng(3)
    sd = np.sqrt(W.KB * s.temperature / s.mass.astype(np.float64))
    V0 = torch.tensor((rng.normal(0, 1, R.shape) * sd[None, :, None]).astype(np.float32), device="cuda")
    Ra, Va = Rg.clone(), V0.clone()
    m.mop_step(Ra, Va, 0.001, 1)
    Rb, Vb = Rg.clone(), V0.clone()
    _, g = w.mop_eval_veff_grad(Rb)
    w.mop_block_integrate(Rb, Vb, g, 0.001, 0)
    _, g = w.mop_eval_veff_grad(Rb)
    w.mop_block_integrate(Rb, Vb, g, 0.001, 1)
    assert H.rms_rel((Rb - Rg).cpu().numpy(), (Ra - Rg).cpu().numpy()) <= 1e-5
    assert H.rms_rel(Vb.cpu().numpy(), Va.cpu().numpy()) <= 1e-5
    w.close()
    m.close()


@pytest.mark.parametrize("parts", [[(0, 2), (2, 2)], [(0, 1), (1, 2), (3, 1)]])
def test_sharded_langevin_step_replays_the_whole_path_noise(B, oracle, parts):
    """NVT on a sharded path (the configuration of the paper's scaling runs): block evaluation + the two
    mop_block_integrate halves + mop_block_thermostat per block reproduce mop_step_langevin on the whole path, velocities
    to 1e-5 RMS -- which they can only do if every block draws, for each of its coordinates, the random number the whole-path
    call draws (the thermostat term is the larger part of the velocity here: c = exp(-0.25) = 0.78)."""
    import torch
    s = W.config1(n_beads=4)
    o = oracle.OracleSystem(s)
    R = W.brownian_path(s, 4, lambda X: oracle.bead(o, X, geom=0)["F"], seed=0)
    rng = np.random.default_rng(3)
    sd = np.sqrt(W.KB * s.temperature / s.mass.astype(np.float64))
    V0 = (rng.normal(0, 1, R.shape) * sd[None, :, None]).astype(np.float32)
    dt, gamma, T, seed, step0 = 0.001, 250.0, s.temperature, 17, 5
    m = B.Mop(s, 4)
    Ra, Va = torch.tensor(R, device="cuda"), torch.tensor(V0, device="cuda")
    m.mop_step_langevin(Ra, Va, dt, 2, gamma, T, seed=seed, step0=step0)
    m.close()
    ctx = [B.Mop(s, n, block=(f, 4)) for f, n in parts]
    Rb = [torch.tensor(R[f:f + n], device="cuda") for f, n in parts]
    Vb = [torch.tensor(V0[f:f + n], device="cuda") for f, n in parts]
    keta = [torch.zeros((s.n_atoms, 3), device="cuda") for _ in parts]

    def grads():
        for k, (f, n) in enumerate(parts):
            last = f + n == 4
            ctx[k].mop_block_pass1(Rb[k], None if last else Rb[k + 1][0].contiguous(), None if last else keta[k])
        for k in range(len(parts)):
            ctx[k].mop_block_pass2(Rb[k])
        return [ctx[k].mop_block_assemble(None if k == 0 else keta[k - 1])[1] for k in range(len(parts))]

    g = grads()
    for it in range(2):
        for k in range(len(parts)):
            ctx[k].mop_block_integrate(Rb[k], Vb[k], g[k], dt, 0)
        g = grads()
        for k in range(len(parts)):
            ctx[k].mop_block_integrate(Rb[k], Vb[k], g[k], dt, 1)
            ctx[k].mop_block_thermostat(Vb[k], dt, gamma, T, seed=seed, step=step0 + it)
    Vs = torch.cat(Vb).cpu().numpy()
    Rs = torch.cat(Rb).cpu().numpy()
    assert H.rms_rel(Vs, Va.cpu().numpy()) <= 1e-5
    assert H.rms_rel(Rs - R, Ra.cpu().numpy() - R) <= 1e-5
    # a block that used its LOCAL coordinate index would draw bead 1's numbers again: the velocities would be far apart
    assert H.rms_rel(Vs[2:], Va.cpu().numpy()[:2]) > 0.1
    with pytest.raises(B.MopError):
        ctx[0].mop_block_thermostat(Vb[0], dt, -1.0, T)
    for c in ctx:
        c.close()


def test_block_path_driver_single_rank(B, oracle):
    """blocks.BlockPath with world = 1 (no process group): the driver bench.py uses, on the real engine."""
    import torch
    s = W.config1(n_beads=6)
    o = oracle.OracleSystem(s)
    R = W.brownian_path(s, 6, lambda X: oracle.bead(o, X, geom=0)["F"], seed=0)
    Rg = torch.tensor(R, device="cuda")
    eng = B.Mop(s, 6, block=(0, 6))
    bp = blocks.BlockPath(eng, s.n_atoms, 0, 6, 6, rank=0, world=1, device="cuda")
    v, g = bp.eval(Rg)
    v_ref, g_ref = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=True)
    assert abs(v - v_ref) <= 1e-6 * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, 1e-4)
    eng.close()


@pytest.mark.parametrize("ranks,config,beads,port", [(4, 2, 4, 29561), (8, 4, 8, 29563)])
def test_bench_block_arm_with_n_ranks_on_one_gpu(B, ranks, config, beads, port):
    """The code path `bench.py --gpus N` takes, run with N real ranks before any multi-GPU box does: N processes (torchrun),
    every one with its own bead-block context on cuda:0, the halos and the 8-byte reduction staged through host memory
    under gloo (NCCL wants one GPU per rank).  Same partition, same BlockPath, the real engine.  FUNCTIONAL, not a scaling
    number: the ranks share one GPU.  Rank 0's V_eff must be that of ONE context evaluating the same N x beads path --
    to 1e-6 only, because every rank generates the path itself with the library's force, whose float atomics differ in the
    last bits from process to process (a few coordinates round to the neighbouring FP32 value)."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(ranks), "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(root, "bench.py"), "--gpus", str(ranks), "--config", str(config),
           "--beads", str(beads), "--steps", "2", "--warmup", "3", "--dist-backend", "gloo", "--all-ranks-on-one-gpu",
           "--no-cpu-baseline"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=1500, cwd=root)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    out = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    n_path = ranks * beads
    assert out["n_gpus"] == ranks and "bead blocks: %d ranks x %d beads of one %d-bead path" % (ranks, beads, n_path) in \
        out["config"]["parallelism"] and "not a scaling number" in out["config"]["parallelism"]
    assert out["value"] > 0 and out["e2e"]["value"] > 0 and out["gpu_launches"] > 0
    s = W.CONFIGS[config](seed=0, n_beads=n_path)
    m1 = B.Mop(s, 1)
    R = W.folded_path(s, n_path, lambda X: m1.mop_force_hvp(X)[0].double().cpu().numpy(), seed=0)
    m1.close()
    m = B.Mop(s, n_path)
    v, _ = m.mop_eval_veff_grad(R, want_grad=False)
    m.close()
    assert abs(out["veff"] - v) <= 1e-6 * abs(v), (out["veff"], v)
