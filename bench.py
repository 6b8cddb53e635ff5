#!/usr/bin/env python
"""bench.py -- chain-timesteps/s of the HI bead-rod BD hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c2] [--impl ours|reference]

A "step" is one pass of the whole hot path (noise, forces, RPY assembly,
Cholesky, L dW, drift, semi-implicit rod update, observables) over one ensemble of synthetic chains.
At N = 1 the workload is BASELINE.json configs[1] (c2: 1024 chains x 100 rods).  For N > 1 every rank
runs its own C chains (global chain ids rank*C ..), no data-path collective; the 26-double ensemble
accumulator is all-reduced once at the end (weak scaling).  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2208_06559_b200 import workloads as W  # noqa: E402

METRIC = "chain-timesteps/sec"
UNIT = "chain-steps/s"
FP64_PEAK_TFLOPS = 37.07      # measured DMMA m8n8k4 issue-rate ceiling on this pool's B200 (profiles/r01_fp64_peak.md)


def _peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        busy = [x for x in sm if x > 0.5 * (max(mx) if mx else 1.0)] or sm
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def _oracle_sample(w: W.Workload, seconds_target: float = 15.0):
    """the oracle, as it stands, on the host cores: a bounded sample of the same workload."""
    import oracle as O
    p = O.Params(n_rods=w.n_rods, dt=w.dt, hstar=w.hstar, b=w.b, kappa=w.kappa(), seed=w.noise_seed)
    cores = O.num_threads()
    chains = min(w.n_chains, max(cores, 1) * 2)
    r = O.init_random_walk(w.n_rods, w.b, w.init_seed, range(chains))
    t0 = time.perf_counter()
    r, info = O.step_ensemble(p, r, 0, 1)
    t1 = time.perf_counter() - t0
    steps = int(max(1, min(5000, seconds_target / max(t1, 1e-6))))
    t0 = time.perf_counter()
    r, info = O.step_ensemble(p, r, 1, steps)
    dt = time.perf_counter() - t0
    return {"value": chains * steps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{chains} chains x {steps} steps of {w.name} ({w.n_rods} rods), OpenMP over chains, {dt:.1f} s"}


def run_reference(args, w):
    """--impl reference: for this tier the reference arm is the CPU oracle (no reference code exists)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as O
    p = O.Params(n_rods=w.n_rods, dt=w.dt, hstar=w.hstar, b=w.b, kappa=w.kappa(), seed=w.noise_seed)
    cores = O.num_threads()
    chains = min(w.n_chains, max(cores, 1) * 2)
    r = O.init_random_walk(w.n_rods, w.b, w.init_seed, range(chains))
    for s in range(args.warmup):
        r, _ = O.step_ensemble(p, r, s, 1)
    t0 = time.perf_counter()
    for s in range(args.steps):
        r, _ = O.step_ensemble(p, r, args.warmup + s, 1)
        O.observables(p, r)
    dt = time.perf_counter() - t0
    val = chains * args.steps / dt
    sample = f"each step = {chains} of the {w.n_chains} chains of {w.name}, OpenMP over chains"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "n_chains": w.n_chains, "n_rods": w.n_rods, "M": w.M, "dt": w.dt, "flow": w.flow,
                   "Wi": w.Wi, "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c2", choices=sorted(W.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--path", type=int, default=0, help="bd_set_path: 0 auto, 1 staged kernels, 2 fused per-chain kernel")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = W.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    import torch.distributed as dist
    from paper_2208_06559_b200 import ensemble
    from paper_2208_06559_b200.binding import BD, NOBS

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libbd has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()

    C, K = w.n_chains, args.steps
    bd = BD(n_rods=w.n_rods, n_chains=C, dt=w.dt, hstar=w.hstar, b=w.b, kappa=w.kappa(), seed=w.noise_seed,
            chain_id0=ensemble.shard(rank, world, C), device=f"cuda:{local_rank}")
    bd.set_workspace()
    bd.set_path(args.path)
    r = bd.init_random_walk(w.init_seed)
    per, ens = bd.empty(C, NOBS), bd.empty(2, NOBS)

    def one_step(s):
        bd.step(r, first_step=s, n_steps=1)
        bd.lib.bd_observables(bd._ctx, r.data_ptr(), per.data_ptr(), ens.data_ptr())

    step_no = 0
    for _ in range(args.warmup):
        one_step(step_no); step_no += 1
    torch.cuda.synchronize()

    # ---------------- timed region: device-resident inputs -------------------------------------------
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    bd.profile(True)
    l0 = bd.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); torch.cuda.synchronize()
    e0.record()
    for _ in range(K):
        one_step(step_no); step_no += 1
    e1.record()
    torch.cuda.synchronize(); barrier()
    ms = e0.elapsed_time(e1)
    launches = bd.launch_count() - l0
    stage, nprof = bd.stage_ms()
    bd.profile(False)
    clocks = sampler.stop() if rank == 0 else None
    ms = ensemble.max_over_ranks(ms, device="cuda")         # device-timed, max over ranks
    ensemble.reduce_ensemble(ens)                           # the one exchange: ensemble accumulator (26 doubles)
    value = world * C * K / (ms * 1e-3)
    failed = bd.last_info()[0]

    # ---------------- end to end: host buffers, H2D + D2H inside the timed region ---------------------
    r_host = r.cpu().pin_memory()
    ens_host = torch.zeros(2, NOBS, dtype=torch.float64).pin_memory()
    for _ in range(2):
        bd.step_host(r_host, step_no, 1, ens_host); step_no += 1
    barrier(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0.record()
    for _ in range(K):
        bd.step_host(r_host, step_no, 1, ens_host); step_no += 1
    e1.record()
    torch.cuda.synchronize(); barrier()
    ms_e2e = max(e0.elapsed_time(e1), 1e3 * (time.perf_counter() - t0))
    ms_e2e = ensemble.max_over_ranks(ms_e2e, device="cuda")
    e2e = {"value": world * C * K / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": C * w.M * 8,
           "d2h_bytes_per_step": C * w.M * 8 + 2 * NOBS * 8}

    if rank == 0:
        peaks = _peaks()
        # dominant kernel: the FP64 Cholesky (a dense contraction -> tensor roofline, FP64 DMMA peak).  On the fused
        # short-chain path the whole step is ONE kernel (k_chain_step); its algorithmic flops are counted as the
        # Cholesky flops only (M^3/3 + M^2/2 + M/6 per chain), the rest of the step is not credited.
        fused = stage["fused"] > 0.0
        chol_ms = (stage["fused"] if fused else stage["cholesky"]) / max(nprof, 1)
        chol_tflops = w.cholesky_flops() * C / (chol_ms * 1e-3) / 1e12 if chol_ms > 0 else None
        traffic = None
        try:
            traffic = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(w.name)
        except Exception:
            pass
        roofline = {"bound": "tensor",
                    "kernel": "k_chain_step<3> (fused a0-a8, one launch per step)" if fused else
                              "bd_cholesky stage (k_potf2 + k_trsm + k_syrk DMMA)",
                    "achieved": chol_tflops, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": (chol_tflops / FP64_PEAK_TFLOPS) if chol_tflops else None, "traffic": traffic,
                    "peak_source": "measured FP64 DMMA ceiling on B200 (148 SM x 64 FMA/clk x 1.957 GHz); "
                                   "MEASURED_PEAKS.json has no FP64 entry (bf16 %.1f TF/s, HBM %.1f GB/s)" %
                                   ((peaks or {}).get("bf16_tflops", float("nan")), (peaks or {}).get("hbm_gbs", float("nan"))),
                    "flops_per_launch": w.cholesky_flops() * C, "ms_per_launch": chol_ms}
        hbm = (peaks or {}).get("hbm_gbs", 6650.0)
        asm_ms, trmv_ms = stage["assemble"] / max(nprof, 1), stage["brownian"] / max(nprof, 1)
        stages = {k: v / max(nprof, 1) for k, v in stage.items()}
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": w.name, "n_chains_per_gpu": C, "n_rods": w.n_rods, "M": w.M, "dt": w.dt, "hstar": w.hstar,
                       "flow": w.flow, "Wi": w.Wi, "l2": ("working set larger than L2 (fragment-major L scratch of the resident CTAs, %.0f MB per step)" %
                              (min(C, 2 * 148) * ((w.M + 7) // 8 * 8) ** 2 * 8 / 1e6)) if stage["fused"] > 0.0 else
                             ("inputs larger than L2 (D/L storage %.0f MB per step)" % (bd.workspace_bytes() / 1e6)),
                       "failed_chains": failed},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "stage_ms_per_step": stages,
            "hbm_stages": None if fused else {
                "assemble_GBps": (4.0 * w.M * w.M + 4.0 * w.M) * C / (asm_ms * 1e-3) / 1e9 if asm_ms > 0 else None,
                "brownian_GBps": 4.0 * w.M * w.M * C / (trmv_ms * 1e-3) / 1e9 if trmv_ms > 0 else None,
                "peak_GBps": hbm, "peak_source": "MEASURED_PEAKS.json" if peaks else "fallback"},
            "cholesky_tflops": chol_tflops,
        }
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = _oracle_sample(w)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
