"""Run one BASELINE.json config for its FULL step count and report throughput and ensemble observables.

    python -m paper_2208_06559_b200.run_config c2 [--steps N] [--chunk K]

c1 1000 steps, c2 10^4, c3 2000, c4 500, c5 50 (workloads.py).  Time stepping is `bd_step` in chunks of `--chunk` steps
per call (the fused path runs a whole chunk inside one kernel launch); after every chunk `bd_observables` reduces the
ensemble and the line shows <R^2>, stretch sqrt(<R^2>) / (N b), <R_x^2>, R_g, the largest rod-length deviation so far
and the number of failed chains (reading A10).  Prints a markdown table and a summary line.
"""
from __future__ import annotations

import argparse

import torch

from . import workloads as W
from .binding import BD, OBS_NAMES


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=sorted(W.CONFIGS))
    ap.add_argument("--steps", type=int, default=0)
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--rows", type=int, default=10)
    args = ap.parse_args()
    w = W.CONFIGS[args.config]
    steps = args.steps or w.steps
    chunk = args.chunk or max(1, steps // args.rows)
    bd = BD(n_rods=w.n_rods, n_chains=w.n_chains, dt=w.dt, hstar=w.hstar, b=w.b, kappa=w.kappa(), seed=w.noise_seed)
    bd.set_workspace()
    r = bd.init_random_walk(w.init_seed)
    bd.step(r.clone(), first_step=0, n_steps=1)                 # warm-up on a copy
    torch.cuda.synchronize()
    i = {n: k for k, n in enumerate(OBS_NAMES)}
    print(f"{w.name}: {w.n_chains} chains x {w.n_rods} rods, flow {w.flow} (Wi {w.Wi}, rate {w.rate:.4g}), dt {w.dt}, {steps} steps")
    print("| step | strain | <R^2> | stretch sqrt(<R^2>)/(N b) | <R_x^2> | R_g | max rod deviation | failed chains |")
    print("|---|---|---|---|---|---|---|---|")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    done, ms, worst = 0, 0.0, 0.0
    while done <= steps:
        per, ens = bd.observables(r)
        torch.cuda.synchronize()
        m = (ens[0] / w.n_chains).cpu().numpy()
        worst = max(worst, float(per[:, i["rod_dev_max"]].max()))
        print(f"| {done} | {done * w.dt * w.rate:.3g} | {m[i['R2']]:.4g} | {m[i['R2']] ** 0.5 / (w.n_rods * w.b):.4f} | {m[i['Rx2']]:.4g} | "
              f"{m[i['Rg2']] ** 0.5:.4g} | {worst:.3g} | {bd.last_info()[0]} |", flush=True)
        if done == steps:
            break
        n = min(chunk, steps - done)
        e0.record()
        bd.step(r, first_step=done, n_steps=n)
        e1.record()
        torch.cuda.synchronize()
        ms += e0.elapsed_time(e1)
        done += n
    print(f"{w.name}: {steps} steps in {ms / 1e3:.2f} s GPU time = {w.n_chains * steps / (ms * 1e-3):.4g} chain-steps/s, "
          f"{bd.last_info()[0]} failed chains, max |Q|-b = {worst:.3g} b")


if __name__ == "__main__":
    main()
