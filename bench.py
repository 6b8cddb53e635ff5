#!/usr/bin/env python
"""bench.py -- chain-timesteps/s of the HI bead-rod BD hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c5] [--impl ours|reference]

A "step" is one pass of the whole hot path (noise, forces, RPY assembly,
Cholesky, L dW, drift, semi-implicit rod update, observables) over one ensemble of synthetic chains.

The headline line (value / ms_per_step / roofline / e2e) is measured on c5, the largest single-GPU configuration of
BASELINE.json (1 chain x 10000 rods, D = 30003^2 FP64), the one the target "Cholesky >= 60 % of FP64 peak for
3N >= 6000, assembly / update >= 70 % of HBM peak" is quoted on; `per_config` carries the same fields for c1-c4, so
that chain-steps/s vs N is one record.  `roofline.peak` is the FP64 DMMA issue rate measured in this process
(paper_2208_06559_b200/bench/fp64_peak.cu) just before the timed region.

For N > 1 every rank runs its own C chains (global chain ids rank*C ..), no data-path collective; the 26-double
ensemble accumulator is all-reduced once at the end (weak scaling).  `--gpus N` without a torchrun environment
re-executes itself under torch.distributed.run with N ranks.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import math
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
HEADLINE = "c5"
# kernel sources whose change invalidates the stored ncu DRAM-traffic figures (profiles/traffic.json)
TRAFFIC_SOURCES = ("potrf.cu", "potrf_tiles.cu", "potf2_blocked.cuh", "warp_chol.cuh", "chain_step.cu")


def _peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return None


def _sources_sha16() -> str:
    h = hashlib.sha256()
    for f in TRAFFIC_SOURCES:
        p = os.path.join(ROOT, "paper_2208_06559_b200", "csrc", f)
        if os.path.exists(p):
            h.update(open(p, "rb").read())
    return h.hexdigest()[:16]


def _traffic(name: str):
    """DRAM bytes of the dominant kernel(s) per launch / per step from the committed ncu capture, with the commit
    and the kernel-source hash it was measured at; None once the kernels have changed since."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    except Exception:
        return None, "profiles/traffic.json missing"
    e = t.get(name)
    if not isinstance(e, dict):
        return None, "no ncu capture for this config"
    if e.get("sources_sha16") != _sources_sha16():
        return None, f"stale: captured at commit {e.get('commit')} (kernel sources changed since)"
    return e.get("bytes"), f"ncu --set full at commit {e.get('commit')} ({e.get('file')})"


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
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def mark(self):
        return time.perf_counter()

    def window(self, t0: float, t1: float):
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 and len(r) >= 7]
        sm = [float(r[0]) for r in rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in rows if r[2].replace(".", "").isdigit()]
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = sorted({names[i] for r in rows for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm), "power_w_max": max(pw) if pw else None}

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()


# ---------------------------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference arm): ONE method for both
# ---------------------------------------------------------------------------------------------------------------------
def _oracle_plan(w: W.Workload):
    """How a bounded sample of workload w is taken (SURVEY.md 8(d) budget labels).  The oracle parallelises over
    chains only, so a C = 1 workload keeps one thread busy."""
    import oracle as O
    cores = O.num_threads()
    if w.M <= 2000:                                       # c1-c3: real chains of the workload, measured
        chains = min(w.n_chains, 2 * max(cores, 1))
        return {"label": "measured", "chains": chains, "n_rods": w.n_rods, "scale": 1.0, "threads": min(chains, cores)}
    if w.M <= 8000:                                       # c4: one real chain x one step, x C stated as scaled
        return {"label": "scaled", "chains": 1, "n_rods": w.n_rods, "scale": 1.0 / min(w.n_chains, max(cores, 1)), "threads": min(w.n_chains, max(cores, 1)),
                "concurrent": min(w.n_chains, max(cores, 1))}
    # c5: one step is 9e12 flop (~2 h on one core): a sub-chain of 1001 beads (M = 3003) is stepped for real and the
    # time extrapolated with the M^3 law of the Cholesky (checked against M = 1503 in the same call)
    return {"label": "extrapolated", "chains": 1, "n_rods": 1000, "scale": (w.M / 3003.0) ** 3, "threads": 1}


def _oracle_step_sample(w: W.Workload, plan, first_step: int, n_steps: int, state):
    """runs n_steps oracle steps of the plan's sample; returns seconds."""
    import oracle as O
    if state.get("r") is None:
        state["p"] = O.Params(n_rods=plan["n_rods"], dt=w.dt, hstar=w.hstar, b=w.b, kappa=w.kappa(), seed=w.noise_seed)
        state["r"] = O.init_random_walk(plan["n_rods"], w.b, w.init_seed, range(plan["chains"]))
    t0 = time.perf_counter()
    state["r"], info = O.step_ensemble(state["p"], state["r"], first_step, n_steps)
    return time.perf_counter() - t0


def _oracle_sample(w: W.Workload, seconds_target: float = 12.0):
    """cpu_baseline: the oracle, as it stands, on the host cores, over a bounded sample of workload w."""
    plan = _oracle_plan(w)
    state = {}
    t1 = _oracle_step_sample(w, plan, 0, 1, state)
    steps = int(max(1, min(5000, seconds_target / max(t1, 1e-6)))) if plan["label"] == "measured" else 1
    dt = _oracle_step_sample(w, plan, 1, steps, state) if plan["label"] == "measured" else t1
    value = plan["chains"] * steps / (dt * plan["scale"])
    return {"value": value, "unit": UNIT, "cores": plan["threads"], "kind": "oracle", "label": plan["label"],
            "sample": _oracle_sample_text(w, plan, steps, dt)}


def _oracle_sample_text(w, plan, steps, seconds):
    if plan["label"] == "measured":
        return (f"measured: {plan['chains']} of the {w.n_chains} chains x {steps} steps of {w.name} ({w.n_rods} rods), "
                f"OpenMP over chains, {seconds:.1f} s")
    if plan["label"] == "scaled":
        return (f"scaled: 1 chain x {steps} step(s) of {w.name} ({w.n_rods} rods, M = {w.M}) measured on one thread, "
                f"{seconds / max(steps, 1):.1f} s per step; value assumes {plan['concurrent']} of the {w.n_chains} chains run at "
                f"that speed side by side on the box's cores (OpenMP over chains; not run)")
    return (f"extrapolated: {steps} step(s) of a {plan['n_rods']}-rod sub-chain (M = {3 * plan['n_rods'] + 3}) on one thread, "
            f"{seconds / max(steps, 1):.2f} s per step, x (M / 3003)^3 = {plan['scale']:.0f} for {w.name} (M = {w.M}); "
            f"the oracle parallelises over chains only and {w.name} has one")


def _config(w: W.Workload, n_chains: int, l2: str):
    return {"workload": w.name, "n_chains_per_gpu": n_chains, "n_rods": w.n_rods, "M": w.M, "dt": w.dt, "hstar": w.hstar,
            "flow": w.flow, "Wi": w.Wi, "l2": l2}


def _l2_text(w: W.Workload, fused: bool, ws_bytes: int) -> str:
    if fused:
        return "working set larger than L2 (factor scratch of the resident CTAs)" if w.n_chains > 64 else \
            "latency case: one chain, working set in shared memory (nothing to flush)"
    return "inputs larger than L2 (D/L storage %.0f MB rewritten every step)" % (ws_bytes / 1e6)


def run_reference(args, w):
    """--impl reference: for this tier the reference arm is the CPU oracle (no reference code exists), timed with the
    same sampling plan as the cpu_baseline leg; each step = one oracle step of that bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    plan = _oracle_plan(w)
    state = {}
    for s in range(args.warmup if plan["label"] == "measured" else min(args.warmup, 1)):
        _oracle_step_sample(w, plan, s, 1, state)
    steps = args.steps if plan["label"] == "measured" else min(args.steps, 3)
    dt = 0.0
    for s in range(steps):
        dt += _oracle_step_sample(w, plan, args.warmup + s, 1, state)
    val = plan["chains"] * steps / (dt * plan["scale"])
    sample = _oracle_sample_text(w, plan, steps, dt) + (f"; {steps} of the requested {args.steps} steps run" if steps != args.steps else "")
    fusedlike = w.M <= 320
    ws_bytes = w.n_chains * ((w.M + 15) // 16 * 16) * ((w.M + 7) // 8 * 8) * 8
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt * plan["scale"] / steps / 1.0, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config(w, w.n_chains, _l2_text(w, fusedlike, ws_bytes)),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": plan["threads"], "kind": "oracle", "label": plan["label"], "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---------------------------------------------------------------------------------------------------------------------
def measure_config(w, K, warmup, rank, local_rank, world, path, sampler, peak_tflops, peak_source, hbm_peak, hbm_source):
    """one workload: device-resident timing, stage timing, end-to-end leg -> dict of the JSON fields."""
    import torch
    from paper_2208_06559_b200 import ensemble
    from paper_2208_06559_b200.binding import BD, NOBS
    import torch.distributed as dist

    def barrier():
        if world > 1:
            dist.barrier()

    C = w.n_chains
    bd = BD(n_rods=w.n_rods, n_chains=C, dt=w.dt, hstar=w.hstar, b=w.b, kappa=w.kappa(), seed=w.noise_seed,
            chain_id0=ensemble.shard(rank, world, C), device=f"cuda:{local_rank}")
    bd.set_workspace()
    bd.set_path(path)
    r = bd.init_random_walk(w.init_seed)
    per, ens = bd.empty(C, NOBS), bd.empty(2, NOBS)

    def one_step(s):
        bd.step(r, first_step=s, n_steps=1)
        bd.lib.bd_observables(bd._ctx, r.data_ptr(), per.data_ptr(), ens.data_ptr())

    step_no = 0
    for _ in range(warmup):
        one_step(step_no); step_no += 1
    torch.cuda.synchronize()

    # ---------------- timed region: device-resident inputs -------------------------------------------
    bd.profile(True)
    l0 = bd.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); torch.cuda.synchronize()
    t_begin = sampler.mark() if sampler else 0.0
    e0.record()
    for _ in range(K):
        one_step(step_no); step_no += 1
    e1.record()
    torch.cuda.synchronize(); barrier()
    t_end = sampler.mark() if sampler else 0.0
    ms = e0.elapsed_time(e1)
    launches = bd.launch_count() - l0
    stage, nprof = bd.stage_ms()
    bd.profile(False)
    ms = ensemble.max_over_ranks(ms, device="cuda")         # device-timed, max over ranks
    ensemble.reduce_ensemble(ens)                           # the one exchange: ensemble accumulator (26 doubles)
    value = world * C * K / (ms * 1e-3)
    failed = bd.last_info()[0]

    # ---------------- end to end: host buffers, H2D + D2H inside the timed region ---------------------
    r_host = r.cpu().pin_memory()
    ens_host = torch.zeros(2, NOBS, dtype=torch.float64).pin_memory()
    Ke = K if w.M < 20000 else min(K, 5)
    for _ in range(2):
        bd.step_host(r_host, step_no, 1, ens_host); step_no += 1
    barrier(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0.record()
    for _ in range(Ke):
        bd.step_host(r_host, step_no, 1, ens_host); step_no += 1
    e1.record()
    torch.cuda.synchronize(); barrier()
    ms_e2e = max(e0.elapsed_time(e1), 1e3 * (time.perf_counter() - t0))
    ms_e2e = ensemble.max_over_ranks(ms_e2e, device="cuda")
    e2e = {"value": world * C * Ke / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": C * w.M * 8,
           "d2h_bytes_per_step": C * w.M * 8 + 2 * NOBS * 8, "steps": Ke}

    # dominant kernel: the FP64 Cholesky (a dense contraction -> tensor roofline, FP64 DMMA peak).  On the fused
    # short-chain path the whole step is ONE kernel (k_chain_step); its algorithmic flops are counted as the
    # Cholesky flops only (M^3/3 + M^2/2 + M/6 per chain), the rest of the step is not credited.
    fused = stage["fused"] > 0.0
    nprof = max(nprof, 1)
    chol_ms = (stage["fused"] if fused else stage["cholesky"]) / nprof
    chol_tflops = w.cholesky_flops() * C / (chol_ms * 1e-3) / 1e12 if chol_ms > 0 else None
    traffic, traffic_source = _traffic(w.name)
    roofline = {"bound": "tensor",
                "kernel": "k_chain_step<3> (fused a0-a8, one launch per step)" if fused else
                          "bd_cholesky stage of bd_step = ONE launch of k_potrf_tiles (persistent tile Cholesky: TMA operands, FP64 DMMA)",
                "achieved": chol_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": (chol_tflops / peak_tflops) if (chol_tflops and peak_tflops) else None,
                "frac_datasheet_40": (chol_tflops / 40.0) if chol_tflops else None,
                "traffic": traffic, "traffic_source": traffic_source, "peak_source": peak_source,
                "flops_per_launch": w.cholesky_flops() * C, "ms_per_launch": chol_ms}
    asm_ms, trmv_ms = stage["assemble"] / nprof, stage["brownian"] / nprof
    asm_gbs = (4.0 * w.M * w.M + 4.0 * w.M) * C / (asm_ms * 1e-3) / 1e9 if asm_ms > 0 else None
    trmv_gbs = 4.0 * w.M * w.M * C / (trmv_ms * 1e-3) / 1e9 if trmv_ms > 0 else None
    out = {
        "value": value, "ms_per_step": ms / K, "steps": K,
        "config": _config(w, C, _l2_text(w, fused, bd.workspace_bytes())),
        "failed_chains": failed, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
        "stage_ms_per_step": {k: v / nprof for k, v in stage.items()},
        "hbm_stages": None if fused else {
            "assemble_GBps": asm_gbs, "assemble_frac": asm_gbs / hbm_peak if asm_gbs else None,
            "brownian_GBps": trmv_gbs, "brownian_frac": trmv_gbs / hbm_peak if trmv_gbs else None,
            "peak_GBps": hbm_peak, "peak_source": hbm_source},
        "cholesky_tflops": chol_tflops,
    }
    if sampler:
        out["clocks"] = sampler.window(t_begin, t_end)
    bd.close()
    del bd, r, per, ens
    torch.cuda.empty_cache()
    return out


def _respawn(args):
    """--gpus N > 1 outside torchrun: start N ranks on this node (one per GPU) and pass their output through."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default=HEADLINE, choices=sorted(W.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="only the --config workload (profiling runs)")
    ap.add_argument("--no-peak", action="store_true", help="skip the FP64 microbenchmark; use the committed figure")
    ap.add_argument("--path", type=int, default=0, help="bd_set_path: 0 auto, 1 staged kernels, 2 fused per-chain kernel")
    ap.add_argument("--backend", default="nccl", help="torch.distributed backend for N > 1 (tests use gloo on CPU)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = W.CONFIGS[args.config]
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(_respawn(args))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE = {world}; refusing to print n_gpus != --gpus")
    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libbd has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group(args.backend, device_id=torch.device("cuda", local_rank) if args.backend == "nccl" else None)

    sampler = None
    if rank == 0:
        sampler = ClockSampler(local_rank)
        sampler.start()
        time.sleep(0.3)

    # ---- roofline denominators, measured in this process -------------------------------------------------------------
    peaks = _peaks()
    hbm_peak = (peaks or {}).get("hbm_gbs", 6550.0)
    hbm_source = "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6550 GB/s (B200_PROFILING.md; MEASURED_PEAKS.json absent)"
    peak_tflops, peak_source = 37.07, "committed figure profiles/r01_fp64_peak.md (--no-peak)"
    if not args.no_peak:
        from paper_2208_06559_b200.bench import fp64_peak
        t0 = sampler.mark() if sampler else 0.0
        fp64_peak.measure("dmma", 16, 20000, 3)                                    # warm the clocks
        peak_tflops, peak_ms = fp64_peak.measure("dmma", 16, 200000, 5)            # ~50 ms per launch
        dfma_tflops, _ = fp64_peak.measure("dfma", 16, 200000, 3)
        pc = sampler.window(t0, sampler.mark()) if sampler else {}
        peak_source = ("FP64 DMMA m8n8k4 issue rate measured in this run (paper_2208_06559_b200/bench/fp64_peak.cu, 16 warps/SM, "
                       "register operands, best of 5): %.2f TFLOP/s at SM clock %s MHz (plain DFMA %.2f); MEASURED_PEAKS.json has no FP64 "
                       "entry (bf16 %.1f TF/s, HBM %.1f GB/s)" %
                       (peak_tflops, pc.get("sm_mhz"), dfma_tflops, (peaks or {}).get("bf16_tflops", float("nan")), hbm_peak))

    common = dict(rank=rank, local_rank=local_rank, world=world, path=args.path, sampler=sampler, peak_tflops=peak_tflops,
                  peak_source=peak_source, hbm_peak=hbm_peak, hbm_source=hbm_source)
    head = measure_config(w, args.steps, args.warmup, **common)

    per_config = []
    if not args.no_per_config and world == 1 and args.config == HEADLINE:
        for name in ("c1", "c2", "c3", "c4"):
            wi = W.CONFIGS[name]
            Ki = {"c1": 1000, "c2": 200, "c3": 40}.get(name, args.steps)           # >= 0.05 s of timed work each
            e = measure_config(wi, max(args.steps, Ki), args.warmup, **common)
            e.pop("clocks", None)
            per_config.append(e)

    if sampler:
        sampler.stop()
    if rank == 0:
        out = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": head["config"], "clocks": head.get("clocks"), "e2e": head["e2e"],
            "gpu_launches": head["gpu_launches"], "roofline": head["roofline"], "stage_ms_per_step": head["stage_ms_per_step"],
            "hbm_stages": head["hbm_stages"], "cholesky_tflops": head["cholesky_tflops"], "failed_chains": head["failed_chains"],
        }
        if per_config:
            out["per_config"] = per_config
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = _oracle_sample(w)
            for e in per_config:
                e["cpu_baseline"] = _oracle_sample(W.CONFIGS[e["config"]["workload"]], seconds_target=4.0)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
