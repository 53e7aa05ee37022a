#!/usr/bin/env python
"""bench.py -- throughput of the MoP hot path (V_eff gradient of an N-bead path) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--beads 8] [--impl ours|reference]

A "step" is one mop_eval_veff_grad over the whole path (stages S0..S7 of DESIGN.md, pair list rebuilt every
step) on the synthetic 150,000-atom membrane-protein-shaped system of BASELINE.json configs[3] at N = 8 beads.
Prints ONE JSON line (rank 0).  metric = bead V_eff-gradient evaluations per second = beads * steps / time;
pair interactions per second and the fraction of the FP32 roofline of the dominant kernel ride along.

--gpus N > 1 (under torchrun): the path does not shard in this build (north_star: one GPU, no collectives), so
every rank runs an independent replica (own seed); value = units of all ranks / max-over-ranks time ("weak").

--impl reference: there is no reference code for this paper; the arm times the FP64 CPU oracle (oracle/), as it
stands, on the host cores, on a bounded sample of the same workload (see `sample` in the line it prints).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "bead_veff_gradient_evals_per_sec"
UNIT = "bead-evals/s"
# Algorithmic FP32 work per in-range, non-excluded atom pair: FMA = 2.
FLOP_PER_PAIR_FORCE = 31.0
FLOP_PER_PAIR_HVP = 55.0
# DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/), or None.
TRAFFIC_BYTES_PER_LAUNCH = 130.6e6   # profiles/r01_ncu_summary.md: dram read 119.9 MB + write 10.7 MB (cfg 4, N = 8)


def env_rank():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def fp32_peak_tflops(sm_mhz):
    """148 SMs x 4 SMSPs x 32 lanes x 2 flop (FMA) x f_SM: one FFMA warp instruction per SMSP per cycle
    (B300_MICROARCH.md 'Instruction issue'; 148 SMs, 1965 MHz: B200_PROFILING.md)."""
    return 148 * 128 * 2 * sm_mhz * 1e6 / 1e12


def all_reduce_max_sum(local_ms, local_units, world, device=None):
    """max over ranks of the time, sum over ranks of the units (torch.distributed; gloo or nccl)."""
    if world == 1:
        return local_ms, local_units
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(units_total, ms_max):
    return units_total / (ms_max * 1e-3)


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe).  NVML is
    polled from a thread every few ms (the timed region of the default run lasts ~0.1 s, shorter than one
    nvidia-smi -lms period); nvidia-smi is the fallback when the NVML binding is missing."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.rows, self.proc, self.thread, self.nvml, self.stop_flag = [], None, None, None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            idx = str(index)
            self.h = (pynvml.nvmlDeviceGetHandleByUUID(idx) if idx.startswith("GPU-")
                      else pynvml.nvmlDeviceGetHandleByIndex(int(idx)))
            self.nvml = pynvml
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _poll(self):
        nv = self.nvml
        bits = [(getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8), "hw_slowdown"),
                (getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40), "hw_thermal_slowdown"),
                (getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20), "sw_thermal_slowdown"),
                (getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4), "sw_power_cap")]
        while not self.stop_flag:
            try:
                sm = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.rows.append((time.perf_counter(), sm, self.smax, pw, [n for b, n in bits if r & b]))
            except Exception:
                pass
            time.sleep(0.003)

    def _read(self):
        for line in self.proc.stdout:
            f = [x.strip() for x in line.strip().split(",")]
            if len(f) < 7:
                continue
            try:
                self.rows.append((time.perf_counter(), float(f[0]), float(f[1]), float(f[2]),
                                  [n for n, v in zip(self.NAMES, f[3:7]) if v.lower().startswith("active")]))
            except ValueError:
                continue

    def stop(self, t0=None, t1=None):
        if self.nvml is None and self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "note": "neither NVML nor nvidia-smi available"}
        self.stop_flag = True
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
        elif self.thread is not None:
            self.thread.join(timeout=1)
        rows = [r for r in self.rows if t0 is None or t0 <= r[0] <= t1]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "note": "no sample fell inside the timed region"}
        reasons = sorted({n for r in rows for n in r[4]})
        return {"sm_mhz": float(np.median([r[1] for r in rows])), "sm_max_mhz": float(max(r[2] for r in rows)),
                "power_w_max": float(max(r[3] for r in rows)), "samples": len(rows), "reasons": reasons,
                "source": "nvml" if self.nvml is not None else "nvidia-smi"}


# ------------------------------------------------------------------------------------------------ workload
def build_system(config, beads, scale=1.0):
    from paper_2501_11962_b200 import workloads as W
    if config == 4:
        if scale >= 0.999:
            return W.config4(seed=0, n_beads=beads)
        f3 = scale ** 3
        n_prot = max(200, int(round(4000 * f3 / 10.0)) * 10)
        return W.config4(seed=0, n_beads=beads, n_total=int(round(150000 * f3)),
                         box=(10.5 * scale, 10.5 * scale, 13.5 * scale), n_protein=n_prot, slab=4.0 * scale, r_cut=1.2,
                         name="c4_membrane_scaled_%.3f" % scale)
    s = W.CONFIGS[config](seed=0, n_beads=beads)
    return s


def workload_name(config, s, beads):
    return "configs[%d] %s: %d atoms, box %.2fx%.2fx%.2f nm, r_cut %.1f nm, N=%d beads" % (
        config - 1, s.name, s.n_atoms, s.box[0], s.box[1], s.box[2], s.r_cut, beads)


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(a):
    import torch
    from paper_2501_11962_b200 import binding, workloads as W
    rank, local_rank, world = env_rank()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the MoP hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    binding.load()
    N = a.beads
    s = build_system(a.config, N)
    Q = s.n_atoms
    # the path: BASELINE.json's Brownian recursion, forces from the library's own pass 1 (not timed)
    m1 = binding.Mop(s, 1, device=local_rank)
    R = W.brownian_path(s, N, lambda X: m1.mop_force_hvp(X)[0].double().cpu().numpy(), seed=rank)
    m1.close()
    m = binding.Mop(s, N, device=local_rank)
    Rd = torch.as_tensor(R, device=dev)
    Gd = torch.empty_like(Rd)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def step():
        m.mop_eval_veff_grad(Rd, sync=False, grad_out=Gd)

    for _ in range(a.warmup):
        step()
    torch.cuda.synchronize()
    st0 = m.mop_get_stats()
    if not np.isfinite(st0["veff"]):
        raise RuntimeError("V_eff is not finite on the bench workload")
    pairs = [m.mop_debug_pairs(n, cap=0)[1] for n in range(m.nf)]   # in-range, non-excluded pairs per force bead
    n_hvp_beads = m.nf if N > 1 else 0
    pairs_force, pairs_hvp = float(sum(pairs)), float(sum(pairs[:n_hvp_beads]))
    launches0 = m.mop_get_stats()["launches"]

    # ---- timed region: K steps, per-step CUDA events on the launching stream, L2 flushed between steps
    m.mop_set_timing(True)
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(a.steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(a.steps)]
    clocks = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ
                          else os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank])
    time.sleep(0.3)
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(a.steps):
        flush.zero_()
        ev0[k].record()
        step()
        ev1[k].record()
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    t1 = time.perf_counter()
    clk = clocks.stop(t0, t1)
    ms_steps = [ev0[k].elapsed_time(ev1[k]) for k in range(a.steps)]
    local_ms = float(sum(ms_steps))
    stages = m.mop_get_timing()
    m.mop_set_timing(False)
    st1 = m.mop_get_stats()
    launches = int(round((st1["launches"] - launches0) / 1.0))
    ms_max, units = all_reduce_max_sum(local_ms, float(N * a.steps), world, dev)

    # ---- end to end: HOST buffers through mop_eval_veff_grad_host, copies inside the timed region
    Rh = torch.as_tensor(R).pin_memory()
    Gh = torch.empty_like(Rh).pin_memory()
    for _ in range(2):
        v_e2e = m.mop_eval_veff_grad_host(Rh, Gh)
    n_e2e = max(3, min(a.steps, 10))
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize()
    te = time.perf_counter()
    for _ in range(n_e2e):
        flush.zero_()
        v_e2e = m.mop_eval_veff_grad_host(Rh, Gh)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - te) * 1e3
    e2e_ms_max, e2e_units = all_reduce_max_sum(e2e_ms, float(N * n_e2e), world, dev)
    if not (np.isfinite(v_e2e) and abs(v_e2e - st1["veff"]) <= 1e-5 * abs(st1["veff"])):
        raise RuntimeError("host-buffer evaluation disagrees with the device-buffer one: %r vs %r" % (v_e2e, st1["veff"]))

    if rank != 0:
        m.close()
        return None
    peaks, peak_src = measured_peaks()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak_tf = fp32_peak_tflops(sm_max)
    t_hvp = stages["S5_nb_hvp"] * 1e-3
    t_force = stages["S2_nb_force"] * 1e-3
    ach = pairs_hvp * FLOP_PER_PAIR_HVP / t_hvp / 1e12 if t_hvp > 0 else 0.0
    ach_f = pairs_force * FLOP_PER_PAIR_FORCE / t_force / 1e12 if t_force > 0 else 0.0
    ms_per_step = ms_max / a.steps
    probe = binding.mop_probe_fp32(local_rank)   # FP32 pipe with and without register-file-limited operands
    out = {
        "metric": METRIC, "value": throughput(units, ms_max), "unit": UNIT, "n_gpus": world, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(a.config, s, N), "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "l2": "256 MiB buffer written between timed steps (L2 flush)", "pair_list": "rebuilt every step",
                   "path": "Brownian recursion, dt=2 fs, nu=50/ps, T=%g K, seed %d" % (s.temperature, rank)},
        "pair_interactions_per_sec": world * (pairs_force + pairs_hvp) / (ms_per_step * 1e-3),
        "pairs_in_range_per_bead": pairs_force / max(m.nf, 1),
        "pair_slots_evaluated_per_pass": st1["pair_slots"],
        "stage_ms": {k: round(v, 5) for k, v in stages.items() if k != "evals"},
        "roofline": {"bound": "alu", "kernel": "k_nonbonded<HVP> (S5, fused force-scalar + H.eta pair kernel)",
                     "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf,
                     "traffic": TRAFFIC_BYTES_PER_LAUNCH,
                     "peak_source": "148 SMs x 128 FP32 lanes x 2 x %.0f MHz (sm_max_mhz, %s MEASURED_PEAKS.json); "
                                    "no measured FP32 entry exists" % (sm_max, peak_src),
                     "flop_per_pair": FLOP_PER_PAIR_HVP, "pairs_per_launch": pairs_hvp, "ms_per_launch": stages["S5_nb_hvp"],
                     "fp32_probe_tflops": {k: round(v, 2) for k, v in probe.items() if k != "sms"},
                     "frac_of_3reg_ffma2_probe": ach / probe["ffma2_3reg_tflops"] if probe["ffma2_3reg_tflops"] > 0 else None,
                     "force_kernel": {"achieved": ach_f, "frac": ach_f / peak_tf, "flop_per_pair": FLOP_PER_PAIR_FORCE,
                                      "pairs_per_launch": pairs_force, "ms_per_launch": stages["S2_nb_force"]}},
        "e2e": {"value": throughput(e2e_units, e2e_ms_max), "unit": UNIT, "h2d_bytes_per_step": int(N) * Q * 12,
                "d2h_bytes_per_step": int(N) * Q * 12 + 8, "steps": n_e2e,
                "api": "mop_eval_veff_grad_host (pinned host R in, grad + V_eff out)"},
        "gpu_launches": launches,
        "clocks": clk,
        "veff": st1["veff"],
    }
    if world == 1 and not a.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(s, N)
    m.close()
    return out


# ------------------------------------------------------------------------------------------------ the oracle legs
def cpu_baseline(s, N):
    """The oracle as it stands on a bounded sample of the bench workload: beads 1-2 of a path over the SAME system
    (inputs from the oracle's own force, never from the CUDA path)."""
    from oracle import oracle as O
    from paper_2501_11962_b200 import workloads as W
    o = O.OracleSystem(s)
    R2 = W.brownian_path(s, 2, lambda X: O.bead(o, X, geom=0)["F"], seed=0)
    t = time.perf_counter()
    v, g, parts = O.veff_grad(o, R2.astype(np.float64), geom=1, want_parts=True)
    dt = time.perf_counter() - t
    nf = max(N - 1, 1)
    return {"value": N / (nf * dt), "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "beads 1-2 of the workload path on the full %d-atom system (one force bead: 1 force pass + 1 H.eta "
                      "pass, %d in-range pairs), %.1f s; scaled to %d force beads per %d-bead evaluation; the oracle "
                      "threads over beads only, so this sample ran on 1 of %d available threads"
                      % (s.n_atoms, parts["npairs"], dt, nf, N, O.num_threads()),
            "seconds": dt, "pair_interactions_per_sec": 2.0 * parts["npairs"] / dt}


def run_reference(a):
    """--impl reference: the FP64 oracle on the host cores; each step one V_eff-gradient evaluation of an N-bead
    path over a reduced copy of the workload (same recipe, density, cutoff), sized to finish within minutes."""
    rank, _, world = env_rank()
    if rank != 0:
        return None
    from oracle import oracle as O
    from paper_2501_11962_b200 import workloads as W
    O.build()
    threads = O.num_threads()
    N = a.beads
    nf = max(N - 1, 1)
    budget = 150.0 / max(a.steps + a.warmup, 1)          # seconds per step
    cost_per_atom = 2.0e-4 * -(-nf // max(min(threads, nf), 1))   # s per atom per evaluation (force + H.eta passes, measured here)
    f = min(1.0, (budget / (cost_per_atom * 150000.0)) ** (1.0 / 3.0)) if a.config == 4 else 1.0
    f = max(f, 0.3)
    s = build_system(a.config, N, scale=f)
    o = O.OracleSystem(s)
    R = W.brownian_path(s, N, lambda X: O.bead(o, X, geom=0)["F"], seed=0).astype(np.float64)
    full_atoms = 150000 if a.config == 4 else s.n_atoms
    for _ in range(a.warmup):
        O.veff_grad(o, R, geom=1)
    t = time.perf_counter()
    for _ in range(a.steps):
        v, g = O.veff_grad(o, R, geom=1)
    dt = time.perf_counter() - t
    units = N * a.steps * (s.n_atoms / float(full_atoms))      # bead evaluations in 150k-atom equivalents
    sample = ("each step = one oracle V_eff-gradient evaluation of an N=%d path over %s (%d atoms, box scale %.3f of "
              "the workload, same recipe/density/cutoff); value scaled linearly in atom count to %d atoms"
              % (N, s.name, s.n_atoms, f, full_atoms))
    val = units / dt
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": world, "steps": a.steps,
            "warmup": a.warmup, "ms_per_step": dt * 1e3 / a.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[%d] at N=%d beads (150,000-atom membrane-protein-shaped system)" % (a.config - 1, N)
                       if a.config == 4 else workload_name(a.config, s, N)},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": min(threads, nf), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "veff": v}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4])
    ap.add_argument("--beads", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    a = ap.parse_args()
    if a.beads is None:
        a.beads = {1: 16, 2: 64, 3: 32, 4: 8}[a.config]
    a.warmup = max(a.warmup, 3) if a.impl == "ours" else a.warmup
    _, _, world = env_rank()
    if a.gpus != world and world > 1:
        raise SystemExit("--gpus %d does not match WORLD_SIZE %d" % (a.gpus, world))
    if a.gpus > 1 and world == 1 and "RANK" not in os.environ:   # convenience: re-launch one rank per GPU
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(a.gpus),
               "--master-addr", "127.0.0.1", "--master-port", "29541", os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    out = run_reference(a) if a.impl == "reference" else run_ours(a)
    if out is not None:
        print(json.dumps(out))
    if world > 1 and a.impl == "ours":
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
