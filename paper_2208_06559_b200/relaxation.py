"""Relaxation time lambda(N) from equilibrium runs ("fitting the last
70 % of the auto-correlation function [of the end-to-end vector] to an exponential decay", :303 equilibrium runs with
dt = 0.001, K* = 1000, expected scaling R_ee, R_g ~ N^0.5 and lambda ~ N^1.5 with HI).

    python -m paper_2208_06559_b200.relaxation [--rods 10 20 40 80] [--chains 1024] [--hstar 0.5 0.0]

Instead of one chain for 100 relaxation times (the paper's single-chain-per-GPU protocol) an ENSEMBLE of independent
chains is followed for `--window` Rouse times from equilibrium random-walk starts and the normalised correlation
C(t) = <R(t).R(0)> / <R(0).R(0)> is averaged over the chains.  All time stepping is `bd_step` (many steps per launch);
the correlation sums come from `bd_end_to_end` / `bd_autocorr` (kernels of libbd, oracle counterpart orc_autocorr); numpy
is used for the least-squares fit on the host only.  This replaces the
Rouse stand-in lambda_s of workloads.py (reading A12) by measured values.
"""
from __future__ import annotations

import argparse
import math

import numpy as np
import torch

from .binding import BD, NOBS
from .workloads import rouse_lambda


def measure(n_rods: int, n_chains: int, hstar: float, dt: float, window: float, samples: int, seed: int = 0,
            resume: str | None = None, save: str | None = None, budget_s: float | None = None):
    """One ensemble run.  With `budget_s` the run stops after that many seconds of wall time, writes its state (positions,
    origin R(0), correlation sums, sample index) to `save` and returns None; `resume` continues from such a file.  The
    noise is counter based (chain id, step) and the kernels deterministic, so a resumed run is the uninterrupted run."""
    import time
    lam_r = rouse_lambda(n_rods + 1)
    total_steps = int(window * lam_r / dt)
    stride = max(1, total_steps // samples)
    bd = BD(n_rods=n_rods, n_chains=n_chains, dt=dt, hstar=hstar, seed=seed)       # K* = 1/dt, a = h* b (or a = b/2 if h* = 0)
    bd.set_workspace()
    sums = bd.empty(samples + 1, 3)                         # per sampling instant: sum R.R0, sum (R.R0)^2, sum R0.R0
    if resume:
        st = np.load(resume)
        assert int(st["n_rods"]) == n_rods and int(st["n_chains"]) == n_chains and int(st["stride"]) == stride
        r = torch.as_tensor(st["r"]).to(bd.device)
        R0 = torch.as_tensor(st["R0"]).to(bd.device)
        k0 = int(st["k"])
        sums[:k0 + 1] = torch.as_tensor(st["sums"][:k0 + 1]).to(bd.device)
    else:
        r = bd.init_random_walk(4242)
        R0 = bd.end_to_end(r)                               # origin R(0) of every chain, kept on the device
        bd.autocorr(r, R0, sums[0])
        k0 = 0
    step = k0 * stride
    t_start = time.perf_counter()
    for k in range(k0, samples):
        bd.step(r, first_step=step, n_steps=stride)
        step += stride
        bd.autocorr(r, R0, sums[k + 1])                     # k_autocorr in libbd (no torch arithmetic on the path)
        if budget_s is not None and k + 1 < samples:
            torch.cuda.synchronize()
            if time.perf_counter() - t_start > budget_s:
                assert bd.last_info() == (0, -1)
                np.savez(save, r=r.cpu().numpy(), R0=R0.cpu().numpy(), sums=sums.cpu().numpy(), k=k + 1, n_rods=n_rods,
                         n_chains=n_chains, stride=stride)
                return None
    sums_h = sums.cpu().numpy()                             # one read-back at the end
    t = np.arange(samples + 1) * stride * dt
    acf = sums_h[:, 0] / sums_h[0, 2]
    per, _ = bd.observables(r)
    torch.cuda.synchronize()
    assert bd.last_info() == (0, -1)
    per = per.cpu().numpy()
    lam, t_cut = fit_tail(t, acf, n_chains)
    return {"N": n_rods, "hstar": hstar, "lambda": lam, "lambda_rouse": lam_r, "Ree": math.sqrt(per[:, 0].mean()),
            "Rg": math.sqrt(per[:, 4].mean()), "steps": step, "acf_end": float(acf[-1]), "t_cut": t_cut}


def fit_tail(t, acf, n_chains):
    """lambda from "the last 70 % of the auto-correlation function", where the function ends at t_cut, the
    first time it drops below its own noise floor max(0.05, 3 / sqrt(chains)) (the standard error of C(t) over the
    ensemble is ~ 1 / sqrt(chains)); beyond that ln C is noise and a fit over it returns the window, not lambda (the
    first version fitted the whole recorded window: with HI the function is gone after a tenth of a Rouse time)."""
    floor = max(0.05, 3.0 / math.sqrt(n_chains))
    below = np.nonzero(acf < floor)[0]
    hi = int(below[0]) if len(below) else len(t)
    lo = int(0.3 * hi)
    if hi - lo < 3:
        return float("nan"), float(t[min(hi, len(t) - 1)])
    slope, _ = np.polyfit(t[lo:hi], np.log(acf[lo:hi]), 1)
    return -1.0 / slope, float(t[hi - 1])


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rods", type=int, nargs="+", default=[10, 20, 40, 80])
    ap.add_argument("--chains", type=int, default=1024)
    ap.add_argument("--hstar", type=float, nargs="+", default=[0.5, 0.0])
    ap.add_argument("--dt", type=float, default=1e-3)
    ap.add_argument("--window", type=float, default=2.0, help="length of the run in Rouse relaxation times (h* = 0)")
    ap.add_argument("--window-hi", type=float, default=0.5, help="the same for h* > 0 (relaxation with HI is several times faster)")
    ap.add_argument("--samples", type=int, default=200)
    ap.add_argument("--budget-s", type=float, default=None, help="stop after this many seconds, write --save, exit 3")
    ap.add_argument("--save", default=None, help="checkpoint file written when --budget-s runs out (one h*, one N)")
    ap.add_argument("--resume", default=None, help="continue from a checkpoint written by --save")
    args = ap.parse_args()
    print("| h* | N rods | steps | lambda (fit) | fitted up to t = | Rouse stand-in | R_ee | R_g | C(t_end) |")
    print("|---|---|---|---|---|---|---|---|---|")
    rows = []
    for h in args.hstar:
        for n in args.rods:
            row = measure(n, args.chains, h, args.dt, args.window if h == 0.0 else args.window_hi, args.samples,
                          resume=args.resume, save=args.save, budget_s=args.budget_s)
            if row is None:
                print(f"checkpoint written to {args.save}", flush=True)
                raise SystemExit(3)
            rows.append(row)
            print(f"| {h} | {n} | {row['steps']} | {row['lambda']:.4g} | {row['t_cut']:.4g} | {row['lambda_rouse']:.4g} | {row['Ree']:.4g} | {row['Rg']:.4g} | "
                  f"{row['acf_end']:.3f} |", flush=True)
    for h in args.hstar:
        sel = [r for r in rows if r["hstar"] == h]
        if len(sel) >= 2:
            ln = np.log([r["N"] for r in sel])
            for key in ("lambda", "Ree", "Rg"):
                e = np.polyfit(ln, np.log([r[key] for r in sel]), 1)[0]
                print(f"h* = {h}: {key} ~ N^{e:.2f}")


if __name__ == "__main__":
    main()
