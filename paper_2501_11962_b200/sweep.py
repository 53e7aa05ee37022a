"""Bead-count sweep of BASELINE.json configs[4]: the 150,000-atom membrane-protein-shaped system at
N = 1, 4, 16, 64, 128 beads on one GPU.

    python -m paper_2501_11962_b200.sweep [--beads 1 4 16 64 128] [--steps 10] [--pmd-steps 20] [--config 4] [--r-buf 0.05]

Per N it prints one JSON line: ms per mop_eval_veff_grad (pair list rebuilt every evaluation, 256 MiB L2 flush
between timed evaluations, CUDA events), bead-gradient evaluations/s, in-range pair interactions/s, the
algorithmic FP32 fraction of the H.eta pair kernel, and mop_step throughput (velocity-Verlet PMD steps/s x N,
integrator kernels included; also with a buffered pair list, --r-buf), and the time of the paper's finite-difference form of the Hessian term
(mop_eval_veff_grad_fd, eps = 0.01) with its RMS deviation from the analytic gradient.  The path is the Brownian recursion of BASELINE.json with the force from the
library's own pass 1 (as in bench.py).  The explicit Euler recursion of the stiff three-site water is not stable
for much more than ~60 steps at dt = 2 fs (bare +0.41 e sites without LJ), so for N > 32 the
path is the 32-bead recursion traversed back and forth (every consecutive pair of beads is still one Brownian
step apart; throughput does not depend on it).  mop_step recomputes the gradient at the start of every call, so
ms_per_pmd_step = elapsed / pmd_steps carries 1/pmd_steps of one extra evaluation.
Needs a CUDA device: there is no CPU fallback.
"""
import argparse
import json

import numpy as np

FLOP_PER_PAIR_HVP = 55.0


def run(config, N, steps, pmd_steps, device=0, r_buf=0.0):
    import torch
    from . import binding, workloads as W
    dev = torch.device("cuda", device)
    s = W.CONFIGS[config](seed=0, n_beads=N)
    m1 = binding.Mop(s, 1, device=device)
    # N > 32: back and forth over the stable stretch of the recursion (workloads.folded_path)
    R = W.folded_path(s, N, lambda X: m1.mop_force_hvp(X)[0].double().cpu().numpy(), seed=0)
    m1.close()
    m = binding.Mop(s, N, device=device)
    Rd = torch.as_tensor(R, device=dev)
    Gd = torch.empty_like(Rd)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    for _ in range(3):
        m.mop_eval_veff_grad(Rd, sync=False, grad_out=Gd)
    torch.cuda.synchronize()
    st = m.mop_get_stats()
    pairs = [m.mop_debug_pairs(n, cap=0)[1] for n in range(m.nf)]
    n_hvp = m.nf if N > 1 else 0
    m.mop_set_timing(True)
    e0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    e1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    for k in range(steps):
        flush.zero_()
        e0[k].record()
        m.mop_eval_veff_grad(Rd, sync=False, grad_out=Gd)
        e1[k].record()
    torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(b) for a, b in zip(e0, e1)]))
    stages = m.mop_get_timing()
    m.mop_set_timing(False)
    # full path-MD steps (eq. 4, velocity Verlet, dt_pmd = 1 fs), integrator included
    V = torch.zeros_like(Rd)
    Rs = Rd.clone()
    m.mop_step(Rs, V, 1.0e-3, 1)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    m.mop_step(Rs, V, 1.0e-3, pmd_steps)
    b.record()
    torch.cuda.synchronize()
    ms_pmd = a.elapsed_time(b) / pmd_steps   # one evaluation + two half-kick kernels per step (plus the initial evaluation / pmd_steps)
    # the same PMD steps with a buffered list (r_buf > 0: the list is rebuilt only when an atom has moved r_buf / 2);
    # thermal velocities, so that atoms move as they do in a run
    ms_pmd_buf, rebuilds_buf = None, None
    if r_buf > 0:
        mb = binding.Mop(s, N, device=device, r_buf=r_buf)
        sd = np.sqrt(W.KB * s.temperature / s.mass.astype(np.float64))
        Vt = torch.as_tensor((np.random.default_rng(1).normal(0, 1, R.shape) * sd[None, :, None]).astype(np.float32), device=dev)
        Rs = Rd.clone()
        mb.mop_step(Rs, Vt, 1.0e-3, 1)
        torch.cuda.synchronize()
        r0 = mb.mop_get_stats()["rebuilds"]
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        mb.mop_step(Rs, Vt, 1.0e-3, pmd_steps)
        b.record()
        torch.cuda.synchronize()
        ms_pmd_buf = a.elapsed_time(b) / pmd_steps
        rebuilds_buf = int(mb.mop_get_stats()["rebuilds"] - r0)
        mb.close()
    # the paper's finite-difference form (three force passes per bead), eps = 0.01
    ms_fd, fd_vs_analytic = None, None
    if N > 1:
        Gf = torch.empty_like(Rd)
        m.mop_eval_veff_grad_fd(Rd, 0.01, sync=False, grad_out=Gf)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(3):
            m.mop_eval_veff_grad_fd(Rd, 0.01, sync=False, grad_out=Gf)
        b.record()
        torch.cuda.synchronize()
        ms_fd = a.elapsed_time(b) / 3
        fd_vs_analytic = float(((Gf - Gd).double().pow(2).sum() / Gd.double().pow(2).sum()).sqrt())
    mem = torch.cuda.max_memory_allocated(dev)
    free, total = torch.cuda.mem_get_info(dev)
    t_h = stages["S5_nb_hvp"] * 1e-3
    out = {"config": "configs[4] sweep on %s" % s.name, "atoms": s.n_atoms, "beads": N, "ms_per_eval": round(ms, 4),
           "bead_evals_per_sec": round(N / (ms * 1e-3), 1),
           "pair_interactions_per_sec": (sum(pairs) + sum(pairs[:n_hvp])) / (ms * 1e-3),
           "stage_ms": {k: round(v, 4) for k, v in stages.items() if k != "evals"},
           "hvp_tflops_algorithmic": (sum(pairs[:n_hvp]) * FLOP_PER_PAIR_HVP / t_h / 1e12) if t_h > 0 else None,
           "ms_per_pmd_step": round(ms_pmd, 4), "pmd_bead_steps_per_sec": round(N / (ms_pmd * 1e-3), 1),
           "r_buf": r_buf, "ms_per_pmd_step_buffered_list": None if ms_pmd_buf is None else round(ms_pmd_buf, 4),
           "list_rebuilds_in_those_steps": rebuilds_buf,
           "ms_per_eval_fd_form": None if ms_fd is None else round(ms_fd, 4), "fd_vs_analytic_grad_rms_rel": fd_vs_analytic,
           "device_memory_used_gb": round((total - free) / 2 ** 30, 2), "veff": st["veff"]}
    m.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--beads", type=int, nargs="+", default=[1, 4, 16, 64, 128])
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--pmd-steps", type=int, default=20)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--r-buf", type=float, default=0.05, help="Verlet buffer (nm) of the buffered-list PMD measurement; 0: skip")
    a = ap.parse_args()
    for N in a.beads:
        print(json.dumps(run(a.config, N, a.steps, a.pmd_steps, r_buf=a.r_buf)), flush=True)


if __name__ == "__main__":
    main()
