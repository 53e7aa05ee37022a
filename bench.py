#!/usr/bin/env python
"""bench.py -- throughput of the MoP hot path (V_eff gradient of an N-bead path) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--beads 8] [--impl ours|reference]

A "step" is one mop_eval_veff_grad over the whole path (stages S0..S7 of DESIGN.md, pair list rebuilt every
step) on the synthetic 150,000-atom membrane-protein-shaped system of BASELINE.json configs[3] at N = 8 beads.
Prints ONE JSON line (rank 0).  metric = bead V_eff-gradient evaluations per second = beads * steps / time;
pair interactions per second and the fraction of the FP32 roofline of the dominant kernel ride along.

--gpus N > 1 (under torchrun), default --parallelism blocks: the paper's layout -- ONE path of
8 N beads, every rank owns a block of 8 consecutive beads (mop.h "bead-block mode") and exchanges two halos per
evaluation with its neighbours over NCCL send/recv plus an 8-byte all-reduce of V_eff (paper_2501_11962_b200/blocks.py);
per-GPU work is fixed, so "scaling": "weak"; value = beads of the whole path * steps / max-over-ranks time.
--parallelism replicas: every rank runs an independent 8-bead replica (own seed), no communication.

--impl reference: there is no reference code for this paper; the arm times the FP64 CPU oracle (oracle/), as it
stands, on the host cores, on the same workload (see `sample` in the line it prints).
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
# The ncu capture of the dominant kernel (S5) on the bench workload, committed under profiles/: a two-column CSV
# "metric,value" for one launch, written from the .ncu-rep by the command in profiles/r02_ncu_summary.md.
NCU_METRICS_FILE = os.path.join("profiles", "r03_ncu_hvp_metrics.csv")


def traffic_bytes_per_launch():
    """dram__bytes_read.sum + dram__bytes_write.sum of one S5 launch from the committed ncu capture, or None."""
    path = os.path.join(ROOT, NCU_METRICS_FILE)
    if not os.path.exists(path):
        return None, None
    vals = {}
    with open(path) as f:
        for line in f:
            k, _, v = line.strip().partition(",")
            try:
                vals[k] = float(v)
            except ValueError:
                continue
    if "dram__bytes_read.sum" in vals and "dram__bytes_write.sum" in vals:
        return vals["dram__bytes_read.sum"] + vals["dram__bytes_write.sum"], NCU_METRICS_FILE
    return None, None


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
def build_system(config, beads):
    from paper_2501_11962_b200 import workloads as W
    return W.CONFIGS[config](seed=0, n_beads=beads)


def workload_name(config, s, beads):
    return "configs[%d] %s: %d atoms, box %.2fx%.2fx%.2f nm, r_cut %.1f nm, N=%d beads" % (
        config - 1, s.name, s.n_atoms, s.box[0], s.box[1], s.box[2], s.r_cut, beads)


def bench_config(a, s, N, world, blocks_mode, n_path, temperature, seed):
    """The `config` object of the JSON line.  Both arms print the same one (the reference arm times the oracle on the GPU
    arm's config): `workload`, `path` and `pair_list` hold for both; `parallelism` and `l2` describe how the GPU arm runs
    that workload (the oracle arm runs on the host cores and has no L2 to flush -- its own run is described in its
    `cpu_baseline.sample`)."""
    return {"workload": workload_name(a.config, s, N) if not blocks_mode else
            workload_name(a.config, s, n_path) + " (one path; %d beads per GPU)" % N,
            "parallelism": "1 GPU" if world == 1 else
            ("bead blocks: %d ranks x %d beads of one %d-bead path, halos by torch.distributed batch_isend_irecv "
             "(%s), V_eff all-reduced (mop.h bead-block mode)"
             % (world, N, n_path, "gloo through host memory, ALL RANKS ON ONE GPU: functional run, not a scaling number"
                if getattr(a, "all_ranks_on_one_gpu", False) else "NCCL point-to-point") if blocks_mode
             else "independent replicas"),
            "l2": "256 MiB buffer written between timed steps (L2 flush)", "pair_list": "rebuilt every step",
            "path": "Brownian recursion, dt=2 fs, nu=50/ps, T=%g K, seed %d" % (temperature, seed)}


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(a):
    import torch
    from paper_2501_11962_b200 import binding, workloads as W
    rank, local_rank, world = env_rank()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the MoP hot path has no CPU fallback")
    if a.all_ranks_on_one_gpu:      # functional run of the N-rank code path on a single GPU (not a scaling number)
        local_rank = 0
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    gloo = a.dist_backend == "gloo"
    rdev = None if gloo else dev    # where the small reduction tensors live
    if world > 1:
        import torch.distributed as dist
        if gloo:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=dev)
    binding.load()
    N = a.beads
    s = build_system(a.config, N)
    Q = s.n_atoms
    blocks_mode = a.parallelism == "blocks" and (world > 1 or a.blocks_on_one_gpu)
    # the path: BASELINE.json's Brownian recursion, forces from the library's own pass 1 (not timed)
    m1 = binding.Mop(s, 1, device=local_rank)
    if blocks_mode:
        # one path of N * world beads (same seed on every rank); this rank owns beads [first, first + N)
        from paper_2501_11962_b200 import blocks
        n_path = N * world
        first, nb = blocks.partition(n_path, world)[rank]
        # at most 32 recursion steps, walked back and forth for longer paths: the raw Euler recursion of the stiff water
        # diverges after ~60 steps, and rank 7 of --gpus 8 would need 63 of them
        R = W.folded_path(s, first + nb, lambda X: m1.mop_force_hvp(X)[0].double().cpu().numpy(), seed=0, first=first)
        m1.close()
        m = binding.Mop(s, nb, device=local_rank, block=(first, n_path))
        bp = blocks.BlockPath(m, Q, first, nb, n_path, rank=rank, world=world, device=dev, host_staging=gloo)
        n_hvp_local = min(nb, n_path - 1 - first)
    else:
        n_path = N
        R = W.brownian_path(s, N, lambda X: m1.mop_force_hvp(X)[0].double().cpu().numpy(), seed=rank)
        m1.close()
        m = binding.Mop(s, N, device=local_rank)
        n_hvp_local = m.nf if N > 1 else 0
    Rd = torch.as_tensor(np.ascontiguousarray(R), device=dev)
    Gd = torch.empty_like(Rd)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def step():
        if blocks_mode:
            bp.eval(Rd, grad_out=Gd, sync=False)   # halos over NCCL; like the whole-path arm, no V_eff read per step
        else:
            m.mop_eval_veff_grad(Rd, sync=False, grad_out=Gd)

    for _ in range(a.warmup):
        step()
    torch.cuda.synchronize()
    st0 = m.mop_get_stats()
    if not np.isfinite(st0["veff"]):
        raise RuntimeError("V_eff is not finite on the bench workload")
    n_force_local = max(n_hvp_local, 1) if not blocks_mode else n_hvp_local
    pairs = [m.mop_debug_pairs(n, cap=0)[1] for n in range(n_force_local)]   # in-range, non-excluded pairs per force bead
    pairs_force, pairs_hvp = float(sum(pairs)), float(sum(pairs[:n_hvp_local]))
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
    veff_job = bp.veff() if blocks_mode else st1["veff"]    # whole-path V_eff (blocks: one 8-byte all-reduce, all ranks)
    launches = int(round((st1["launches"] - launches0) / 1.0))
    # the headline above records stage events, which switches the CUDA-graph replay off; the same K steps with stage
    # timing off go through the graphs, the form a caller of mop_eval_veff_grad gets (reported beside, not instead)
    ms_graphs = None
    if not blocks_mode:
        eg0 = [torch.cuda.Event(enable_timing=True) for _ in range(a.steps)]
        eg1 = [torch.cuda.Event(enable_timing=True) for _ in range(a.steps)]
        for _ in range(2):
            step()
        for k in range(a.steps):
            flush.zero_()
            eg0[k].record()
            step()
            eg1[k].record()
        torch.cuda.synchronize()
        ms_graphs = float(sum(eg0[k].elapsed_time(eg1[k]) for k in range(a.steps))) / a.steps
    ms_max, units = all_reduce_max_sum(local_ms, float(Rd.shape[0] * a.steps), world, rdev)
    if world > 1:   # pair counts of all ranks (rank 0 reports the job's pair rate; the roofline stays rank 0's own kernel)
        pc = torch.tensor([pairs_force, pairs_hvp], dtype=torch.float64, device=rdev)
        torch.distributed.all_reduce(pc)
        pairs_force_job, pairs_hvp_job = float(pc[0]), float(pc[1])
    else:
        pairs_force_job, pairs_hvp_job = pairs_force, pairs_hvp

    # ---- the same step with a buffered pair list (r_buf = 0.05 nm) that is REUSED: S0/S1 are replaced by k_refresh and
    # one flag read; the pair passes walk the longer list of r_cut + r_buf.  Reported separately.
    reuse = None
    if world == 1 and not blocks_mode:
        mr = binding.Mop(s, N, device=local_rank, r_buf=0.05)
        for _ in range(a.warmup):
            mr.mop_eval_veff_grad(Rd, sync=False, grad_out=Gd)
        torch.cuda.synchronize()
        r0 = mr.mop_get_stats()
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(a.steps)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(a.steps)]
        for k in range(a.steps):
            flush.zero_()
            e0[k].record()
            mr.mop_eval_veff_grad(Rd, sync=False, grad_out=Gd)
            e1[k].record()
        torch.cuda.synchronize()
        r1 = mr.mop_get_stats()
        ms_r = float(sum(e0[k].elapsed_time(e1[k]) for k in range(a.steps))) / a.steps
        reuse = {"r_buf_nm": 0.05, "ms_per_step": ms_r, "value": N / (ms_r * 1e-3), "unit": UNIT,
                 "rebuilds_in_timed_region": int(r1["rebuilds"] - r0["rebuilds"]),
                 "reuses_in_timed_region": int(r1["reuses"] - r0["reuses"]),
                 "note": "same coordinates every step, so every timed step reuses the list; neighbour sets are then "
                         "exact up to FP32 rounding of r^2 at r_c (DESIGN.md), which is why the headline rebuilds"}
        mr.close()

    # ---- end to end: HOST buffers through mop_eval_veff_grad_host, copies inside the timed region
    Rh = torch.as_tensor(np.ascontiguousarray(R)).pin_memory()
    Gh = torch.empty_like(Rh).pin_memory()

    def e2e_step():
        if not blocks_mode:
            return m.mop_eval_veff_grad_host(Rh, Gh)
        Rd.copy_(Rh, non_blocking=True)             # this rank's block in, its gradient block out
        v, _ = bp.eval(Rd, grad_out=Gd)
        Gh.copy_(Gd, non_blocking=True)
        torch.cuda.synchronize()
        return v

    for _ in range(2):
        v_e2e = e2e_step()
    n_e2e = max(3, min(a.steps, 10))
    if world > 1:
        torch.distributed.barrier()
    # every call is host-synchronous (it returns V_eff), so its wall-clock time IS the end-to-end time of one step; the L2
    # flush runs, and is waited for, before the clock starts
    e2e_ms = 0.0
    for _ in range(n_e2e):
        flush.zero_()
        torch.cuda.synchronize()
        te = time.perf_counter()
        v_e2e = e2e_step()
        e2e_ms += (time.perf_counter() - te) * 1e3
    e2e_ms_max, e2e_units = all_reduce_max_sum(e2e_ms, float(Rd.shape[0] * n_e2e), world, rdev)
    if not blocks_mode and not (np.isfinite(v_e2e) and abs(v_e2e - st1["veff"]) <= 1e-5 * abs(st1["veff"])):
        raise RuntimeError("host-buffer evaluation disagrees with the device-buffer one: %r vs %r" % (v_e2e, st1["veff"]))
    if not np.isfinite(v_e2e):
        raise RuntimeError("V_eff is not finite in the end-to-end run")

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
    traffic, traffic_src = traffic_bytes_per_launch()
    out = {
        "metric": METRIC, "value": throughput(units, ms_max), "unit": UNIT, "n_gpus": world, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": bench_config(a, s, N, world, blocks_mode, n_path, s.temperature, rank),
        "ms_per_step_graphs": ms_graphs,
        "pair_interactions_per_sec": (pairs_force_job + pairs_hvp_job) / (ms_per_step * 1e-3),
        "pairs_in_range_per_bead": pairs_force / max(m.nf, 1),
        "pair_slots_admitted_by_patterns_per_pass": st1["pair_slots"],
        "pair_slots_evaluated_per_pass": st1["pair_slots_evaluated"],
        "evaluated_slots_per_in_range_pair": st1["pair_slots_evaluated"] / max(pairs_force, 1.0),
        "stage_ms": {k: round(v, 5) for k, v in stages.items() if k != "evals"},
        "roofline": {"bound": "alu", "kernel": "k_nonbonded<HVP> (S5, fused force-scalar + H.eta pair kernel)",
                     "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf,
                     "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": "148 SMs x 128 FP32 lanes x 2 x %.0f MHz (sm_max_mhz, %s MEASURED_PEAKS.json); "
                                    "no measured FP32 entry exists" % (sm_max, peak_src),
                     "flop_per_pair": FLOP_PER_PAIR_HVP, "pairs_per_launch": pairs_hvp, "ms_per_launch": stages["S5_nb_hvp"],
                     "force_kernel": {"achieved": ach_f, "frac": ach_f / peak_tf, "flop_per_pair": FLOP_PER_PAIR_FORCE,
                                      "pairs_per_launch": pairs_force, "ms_per_launch": stages["S2_nb_force"]}},
        "e2e": {"value": throughput(e2e_units, e2e_ms_max), "unit": UNIT, "h2d_bytes_per_step": int(n_path) * Q * 12,
                "d2h_bytes_per_step": int(n_path) * Q * 12 + 8 * world, "steps": n_e2e,
                "api": "mop_eval_veff_grad_host (pinned host R in, grad + V_eff out)" if not blocks_mode else
                       "per rank: pinned host block -> device, blocks.BlockPath.eval, gradient block -> pinned host"},
        "with_list_reuse": reuse,
        "gpu_launches": launches,
        "clocks": clk,
        "veff": veff_job,
    }
    if world == 1 and not a.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(s, N)
    m.close()
    return out


# ------------------------------------------------------------------------------------------------ the oracle legs
def cpu_baseline(s, N):
    """The oracle as it stands on the bench workload itself (inputs from the oracle's own force, never from the CUDA
    path).  The oracle threads over beads only (OpenMP over the force beads of each pass), so two figures:
    `value` = one whole N-bead evaluation on min(threads, force beads) threads; `one_thread` = beads 1-2 (one force
    bead) on one thread, scaled to the force beads of the evaluation."""
    from oracle import oracle as O
    from paper_2501_11962_b200 import workloads as W
    o = O.OracleSystem(s)
    threads = O.num_threads()
    nf = max(N - 1, 1)
    nb = min(N, 8)                                   # bounded sample: at most 8 beads of the path
    R = W.brownian_path(s, nb, lambda X: O.bead(o, X, geom=0)["F"], seed=0).astype(np.float64)
    t = time.perf_counter()
    v, g, parts = O.veff_grad(o, R, geom=1, want_parts=True)
    dt_all = time.perf_counter() - t
    nfb = max(nb - 1, 1)
    out = {"value": N * (nfb / float(nf)) / dt_all, "unit": UNIT, "cores": min(threads, nfb), "kind": "oracle",
           "sample": "one whole V_eff-gradient evaluation of the first %d beads of the workload path on the full %d-atom "
                     "system (%d force beads: force pass + H.eta pass each, %d in-range pairs in total), %.1f s on %d of "
                     "%d available threads%s; the path comes from the same recursion and seed as the GPU arm's but with the "
                     "oracle's FP64 force in it (the GPU arm's uses the library's pass 1), so the two arms time equal "
                     "workloads, not byte-identical inputs"
                     % (nb, s.n_atoms, nfb, parts["npairs"], dt_all, min(threads, nfb), threads,
                        "" if nb == N else "; scaled to %d force beads" % nf),
           "seconds": dt_all, "pair_interactions_per_sec": 2.0 * parts["npairs"] / dt_all}
    if nb >= 2:
        t = time.perf_counter()
        v2, g2, p2 = O.veff_grad(o, R[:2], geom=1, want_parts=True)
        dt1 = time.perf_counter() - t
        out["one_thread"] = {"value": N / (nf * dt1), "unit": UNIT, "cores": 1, "seconds": dt1,
                             "sample": "beads 1-2 (one force bead, %d in-range pairs) on one thread, scaled to %d force "
                                       "beads" % (p2["npairs"], nf)}
    return out


def run_reference(a):
    """--impl reference: there is no reference code, so this arm times the FP64 oracle on the host cores, on the bench
    workload itself (same system, same bead count: `config` equals the GPU arm's).  Each step is one whole oracle
    V_eff-gradient evaluation of the N-bead path (OpenMP over the force beads).  A wall-clock guard ends the run early
    (and says so: `steps` is what was done) if the host is much slower than the ~20 s per step measured here."""
    rank, _, world = env_rank()
    if rank != 0:
        return None
    from oracle import oracle as O
    from paper_2501_11962_b200 import workloads as W
    O.build()
    threads = O.num_threads()
    N = a.beads
    nf = max(N - 1, 1)
    t_start = time.perf_counter()
    budget_s = 1200.0
    s = build_system(a.config, N)
    o = O.OracleSystem(s)
    R = W.brownian_path(s, N, lambda X: O.bead(o, X, geom=0)["F"], seed=0).astype(np.float64)
    warm_done = 0
    for _ in range(a.warmup):
        if time.perf_counter() - t_start > 0.3 * budget_s:
            break
        O.veff_grad(o, R, geom=1)
        warm_done += 1
    t = time.perf_counter()
    done = 0
    for _ in range(a.steps):
        v, g, parts = O.veff_grad(o, R, geom=1, want_parts=True)
        done += 1
        if time.perf_counter() - t_start > budget_s:
            break
    dt = time.perf_counter() - t
    val = N * done / dt
    sample = ("each step = one whole oracle V_eff-gradient evaluation of the N=%d path over the full system (%d atoms, %d "
              "force beads: force pass + H.eta pass each, %d in-range pairs per evaluation) on %d of %d threads; %d of %d "
              "timed steps and %d of %d warm-up steps done" % (N, s.n_atoms, nf, parts["npairs"], min(threads, nf), threads,
                                                             done, a.steps, warm_done, a.warmup))
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": world, "steps": done,
            "warmup": warm_done, "ms_per_step": dt * 1e3 / done, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": bench_config(a, s, N, world, a.parallelism == "blocks" and world > 1, N * world, s.temperature, 0),
            "pair_interactions_per_sec": 2.0 * parts["npairs"] * done / dt,
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
    ap.add_argument("--blocks-on-one-gpu", action="store_true",
                    help="--gpus 1 through the bead-block driver (one block = the whole path): exercises that code path")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="gloo: halos and reductions staged through host memory (needed when several ranks share a GPU)")
    ap.add_argument("--all-ranks-on-one-gpu", action="store_true",
                    help="every rank uses cuda:0: runs the N-rank code path on one GPU (functional check, not a scaling "
                         "number; use with --dist-backend gloo -- NCCL needs one GPU per rank)")
    ap.add_argument("--parallelism", default="blocks", choices=["blocks", "replicas"],
                    help="--gpus N > 1: one path sharded by bead blocks with halo exchange (default), or independent replicas")
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
