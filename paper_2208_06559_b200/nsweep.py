"""N-sweep of the per-timestep hot path (BASELINE.json metric "chain-timesteps/sec vs N beads"; the paper's Fig. 7,
PAPER.md:297-299: N = 199 .. 6399 rods, one chain per GPU, step time ~ N^1.2 for short and N^2.2-2.86 for long chains).

    python -m paper_2208_06559_b200.nsweep [--chains 1 16] [--beads 200 400 ...] [--context]

For every (C, N_b) it times `bd_step` (+ observables) with CUDA events, reports ms per ensemble step, chain-steps/s and
the Cholesky stage in TFLOP/s, and fits the log-log slope of the step time.  `--context` adds bench-only comparator
rows that are NOT part of libbd: `torch.linalg.cholesky(D, out=preallocated)` (cuSOLVER potrf / potrfBatched through torch's
wrapper: the call is out of place, so it includes torch's dispatch and one M^2 copy per chain; "the paper's method on this
box") on the same matrices and an FP64 `torch.matmul` of 8192^3 (cuBLAS DGEMM).
Prints a markdown table; synthetic seeded random-walk chains (workloads.py recipe), h* = a = 0.25, dt = 1e-4, no flow.
"""
from __future__ import annotations

import argparse
import math

import torch

from .binding import BD, NOBS


def _time(fn, reps):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fn()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def sweep(chains, beads, context=False):
    rows = []
    for C in chains:
        for nb in beads:
            N, M = nb - 1, 3 * nb
            flops = M ** 3 / 3.0 + M ** 2 / 2.0 + M / 6.0
            bd = BD(n_rods=N, n_chains=C, dt=1e-4, seed=0)
            bd.set_workspace()
            r = bd.init_random_walk(1000)
            per, ens = bd.empty(C, NOBS), bd.empty(2, NOBS)
            step = [0]

            def one():
                bd.step(r, first_step=step[0], n_steps=1)
                bd.lib.bd_observables(bd._ctx, r.data_ptr(), per.data_ptr(), ens.data_ptr())
                step[0] += 1

            for _ in range(3):
                one()
            reps = max(3, min(200, int(2000.0 / max(_time(one, 1), 0.01))))
            bd.profile(True)
            ms = _time(one, reps)
            stage, nprof = bd.stage_ms()
            bd.profile(False)
            chol_ms = (stage["fused"] if stage["fused"] > 0 else stage["cholesky"]) / max(nprof, 1)
            row = {"C": C, "Nb": nb, "M": M, "ms": ms, "cps": C / (ms * 1e-3), "tf": flops * C / (chol_ms * 1e-3) / 1e12,
                   "fused": stage["fused"] > 0, "failed": bd.last_info()[0]}
            if context and C * M * M * 8.0 < 20e9:        # comparator only where two extra copies of D fit comfortably
                D = bd.assemble_hi(r)[:, :, :M].contiguous()
                Lout = torch.empty_like(D)                    # preallocated result: no allocation inside the timed call
                row["potrf_ms"] = _time(lambda: torch.linalg.cholesky(D, out=Lout), 3)
                del Lout
                row["potrf_tf"] = flops * C / (row["potrf_ms"] * 1e-3) / 1e12
                del D
            rows.append(row)
            del bd, r
            torch.cuda.empty_cache()
    return rows


def slope(rows, C, lo, hi):
    pts = [(math.log(r["Nb"]), math.log(r["ms"])) for r in rows if r["C"] == C and lo <= r["Nb"] <= hi]
    if len(pts) < 2:
        return float("nan")
    n = len(pts)
    sx, sy = sum(p[0] for p in pts), sum(p[1] for p in pts)
    sxx, sxy = sum(p[0] ** 2 for p in pts), sum(p[0] * p[1] for p in pts)
    return (n * sxy - sx * sy) / (n * sxx - sx * sx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--chains", type=int, nargs="+", default=[1, 16])
    ap.add_argument("--beads", type=int, nargs="+", default=[200, 400, 800, 1600, 3200, 6400, 10001])
    ap.add_argument("--context", action="store_true")
    args = ap.parse_args()
    rows = sweep(args.chains, args.beads, args.context)
    hdr = "| C | N_b | M | path | ms / ensemble step | chain-steps/s | Cholesky TFLOP/s |"
    sep = "|---|---|---|---|---|---|---|"
    if args.context:
        hdr += " torch.linalg.cholesky(out=) ms (TFLOP/s): cuSOLVER potrf / potrfBatched through torch's wrapper |"
        sep += "---|"
    print(hdr)
    print(sep)
    for r in rows:
        line = (f"| {r['C']} | {r['Nb']} | {r['M']} | {'fused' if r['fused'] else 'staged'} | {r['ms']:.4g} | {r['cps']:.4g} | "
                f"{r['tf']:.3g} |")
        if args.context:
            line += f" {r['potrf_ms']:.4g} ({r['potrf_tf']:.3g}) |" if "potrf_ms" in r else " - |"
        print(line)
    for C in args.chains:
        print(f"C = {C}: step time ~ N_b^{slope(rows, C, 200, 800):.2f} (N_b 200-800), ~ N_b^{slope(rows, C, 3200, 10001):.2f} (N_b 3200-10001)")
    if args.context:
        a = torch.randn(8192, 8192, dtype=torch.float64, device="cuda")
        ms = _time(lambda: torch.matmul(a, a), 3)
        print(f"context: FP64 torch.matmul 8192^3 (cuBLAS DGEMM): {ms:.2f} ms = {2 * 8192 ** 3 / (ms * 1e-3) / 1e12:.1f} TFLOP/s")


if __name__ == "__main__":
    main()
