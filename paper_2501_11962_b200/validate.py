"""Fig. 4 analogue: energy conservation of path MD in the microcanonical ensemble and temperature
stability under the Langevin thermostat, on a synthetic config of BASELINE.json (default: configs[1], the 3,000-atom
water-like box with N = 64 beads; the paper's own run is 512 beads x ~150k atoms on the JUWELS Cluster).

    python -m paper_2501_11962_b200.validate [--config 2] [--beads 64] [--steps 2000] [--dt 0.0005]

At the paper's PMD step (--dt 0.001) the Lennard-Jones config 1 runs (profiles/r03_validate_fig4.txt); the
unconstrained water stand-in of config 2 needs 0.5 fs, the default here (the paper constrains bonds to H, out of scope).

Prints one JSON line per ensemble.  NVE: velocity Verlet (mop_step) from thermal velocities; reports the standard
deviation and the drift of V_eff + E_kin relative to the mean kinetic energy.  NVT: mop_step_langevin with the paper's
damping (250 /ps) from rest; reports mean and standard deviation of the kinetic temperature after
equilibration.  Needs a CUDA device (there is no CPU fallback); the path is generated with the library's own force.
"""
import argparse
import json

import numpy as np


def run(config, N, steps, dt, device=0, block=50):
    import torch
    from . import binding, workloads as W
    dev = torch.device("cuda", device)
    s = W.CONFIGS[config](seed=0, n_beads=N)
    m1 = binding.Mop(s, 1, device=device)
    R = W.brownian_path(s, N, lambda X: m1.mop_force_hvp(X)[0].double().cpu().numpy(), seed=0)
    m1.close()
    m = binding.Mop(s, N, device=device)
    dof = R.size
    T = s.temperature
    out = []
    # ---- NVE
    sd = np.sqrt(W.KB * T / s.mass.astype(np.float64))
    Rg = torch.as_tensor(R, device=dev).clone()
    Vg = torch.as_tensor((np.random.default_rng(5).normal(0, 1, R.shape) * sd[None, :, None]).astype(np.float32), device=dev)
    tot, kin = [], []
    for _ in range(steps // block):
        m.mop_step(Rg, Vg, dt, block)
        st = m.mop_get_stats()
        tot.append(st["veff"] + st["E_kin"])
        kin.append(st["E_kin"])
    tot, kin = np.asarray(tot), np.asarray(kin)
    slope = np.polyfit(np.arange(len(tot)), tot, 1)[0] * len(tot)
    out.append({"ensemble": "NVE", "system": s.name, "atoms": s.n_atoms, "beads": N, "steps": len(tot) * block, "dt_ps": dt,
                "mean_E_kin": float(kin.mean()), "std_total_over_mean_E_kin": float(tot.std() / kin.mean()),
                "drift_total_over_mean_E_kin": float(slope / kin.mean()),
                "kinetic_temperature_mean_K": float(2 * kin.mean() / (dof * W.KB))})
    # ---- NVT
    Rg = torch.as_tensor(R, device=dev).clone()
    Vg = torch.zeros_like(Rg)
    gamma, done, tk = 250.0, 0, []
    for b in range(steps // block):
        m.mop_step_langevin(Rg, Vg, dt, block, gamma, T, seed=1, step0=done)
        done += block
        tk.append(2 * m.mop_get_stats()["E_kin"] / (dof * W.KB))
    tk = np.asarray(tk[len(tk) // 4:])
    out.append({"ensemble": "NVT", "system": s.name, "atoms": s.n_atoms, "beads": N, "steps": done, "dt_ps": dt,
                "gamma_per_ps": gamma, "target_K": T, "kinetic_temperature_mean_K": float(tk.mean()),
                "kinetic_temperature_std_K": float(tk.std()), "expected_std_K": float(T * np.sqrt(2.0 / dof))})
    m.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--beads", type=int, default=64)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--dt", type=float, default=0.0005)
    a = ap.parse_args()
    for line in run(a.config, a.beads, a.steps, a.dt):
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
