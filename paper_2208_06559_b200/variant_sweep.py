"""Paper-variant runs on the GPU path: the settings the paper itself ran --
uniform noise (Eq. 2, `noise_kind = 1`), (dt, K*) = (1e-3, 1e3) -- in start-up of
uniaxial extension, for several h*.

    python -m paper_2208_06559_b200.variant_sweep [--rods 100] [--chains 256] [--Wi 3] [--strain 6] [--hstar 1e-5 0 0.5]

The check of PAPER.md:262 / Fig. 6 (:419): a BR-100 chain at Wi = 3 with a negligibly low h* = 1e-5 must follow the
same curve of R_end-end (and N_1, inset) against strain as the run without HI.  Every h* gets the SAME start
configurations and the SAME noise stream (Philox keyed by chain id and step), so the two curves
are compared chain by chain as well as in the mean.  A run with h* = 0.5 (the paper's HI setting) shows how far HI
moves the curve.  The strain rate is Wi / lambda: by default with the Rouse stand-in lambda of workloads.py for every
h* (reading A12: the paper's own lambda values are only in Fig. 8, an image), so that all runs share one rate and "Wi"
is nominal for the HI run; with `--lam measured` every h* >= 1e-3 first measures its own lambda from an equilibrium
ensemble (relaxation.py) and runs at rate Wi / lambda(h*), the paper's definition of Wi.

All time stepping is `bd_step` (many steps per launch), observables by `bd_observables`; torch only carries the
buffers.  N_1 = tau_11 - tau_22 (Eq. 29) with tau = N delta + sum_k <T_k Q_k> as printed in Eq. 28
(PAPER.md:290), i.e. N_1 = <S_xx - S_yy> with S = sum_k T_k (x) Q_k from `bd_observables`.
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import relaxation
from .binding import BD, OBS_NAMES
from .workloads import rouse_lambda


def run(n_rods: int, n_chains: int, hstar: float, rate: float, dt: float, steps: int, samples: int, noise_kind: int,
        flow: str = "extension"):
    if flow == "shear":
        kappa = np.zeros((3, 3)); kappa[0, 1] = rate                 # kappa_xy = shear rate
    else:
        kappa = np.diag([rate, -0.5 * rate, -0.5 * rate])
    bd = BD(n_rods=n_rods, n_chains=n_chains, dt=dt, hstar=hstar, kappa=kappa, seed=7, noise_kind=noise_kind)
    bd.set_workspace()
    r = bd.init_random_walk(2024)
    i = {n: k for k, n in enumerate(OBS_NAMES)}
    stride = max(1, steps // samples)
    rows, per_chain = [], []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ms, done = 0.0, 0
    while True:
        per, ens = bd.observables(r)
        torch.cuda.synchronize()
        p = per.cpu().numpy()
        n1 = p[:, i["Sxx"]] - p[:, i["Syy"]]
        rows.append((done * dt * rate, float(np.sqrt(p[:, i["R2"]].mean())), float(n1.mean()),
                     float(n1.std(ddof=1) / np.sqrt(n_chains)), float(p[:, i["rod_dev_max"]].max()),
                     float(np.sqrt(p[:, i["Ry2"]].mean()))))
        per_chain.append(np.sqrt(p[:, i["R2"]]))
        if done >= steps:
            break
        n = min(stride, steps - done)
        e0.record()
        bd.step(r, first_step=done, n_steps=n)
        e1.record()
        torch.cuda.synchronize()
        ms += e0.elapsed_time(e1)
        done += n
    failed = bd.last_info()[0]
    bd.close()
    return rows, np.array(per_chain), ms, failed


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rods", type=int, default=100)
    ap.add_argument("--chains", type=int, default=256)
    ap.add_argument("--Wi", type=float, default=3.0)
    ap.add_argument("--strain", type=float, default=6.0)
    ap.add_argument("--dt", type=float, default=1e-3)
    ap.add_argument("--samples", type=int, default=24)
    ap.add_argument("--hstar", type=float, nargs="+", default=[1e-5, 0.0, 0.5])
    ap.add_argument("--noise-kind", type=int, default=1, help="1 = the paper's uniform law (Eq. 2), 0 = Gaussian")
    ap.add_argument("--lam", choices=("rouse", "measured"), default="rouse")
    ap.add_argument("--lam-value", type=float, default=0.0, help="use this relaxation time for every h* (e.g. the N^1.5 "
                    "extrapolation of profiles/r02_relaxation.md for chains too long to measure)")
    ap.add_argument("--flow", choices=("extension", "shear"), default="extension")
    args = ap.parse_args()
    lam_r = rouse_lambda(args.rods + 1)
    print(f"BR-{args.rods}, {args.chains} chains, start-up of {args.flow} Wi = {args.Wi}, dt = {args.dt}, K* = {1 / args.dt:g}, "
          f"noise kind {args.noise_kind}, to strain {args.strain}; lambda: {args.lam} (Rouse stand-in {lam_r:.4g})")
    res = {}
    for h in args.hstar:
        lam = args.lam_value if args.lam_value > 0 else lam_r
        if args.lam_value <= 0 and args.lam == "measured" and h >= 1e-3:
            lam = relaxation.measure(args.rods, 2048, h, args.dt, 0.5, 200)["lambda"]
        rate = args.Wi / lam
        steps = int(round(args.strain / (rate * args.dt)))
        rows, pc, ms, failed = run(args.rods, args.chains, h, rate, args.dt, steps, args.samples, args.noise_kind, args.flow)
        res[h] = (rows, pc)
        print(f"h* = {h:g}: lambda {lam:.4g}, rate {rate:.4g}, {steps} steps in {ms / 1e3:.1f} s GPU time = {args.chains * steps / (ms * 1e-3):.4g} chain-steps/s, "
              f"{failed} failed chains, max ||Q|-b| = {max(r[4] for r in rows):.3g}", flush=True)
    hs = list(args.hstar)
    print("\n| strain | " + " | ".join(f"R_ee (h* = {h:g}) | sqrt<R_y^2> | N_1 (h* = {h:g}) +- SE" for h in hs) + " |")
    print("|---|" + "---|---|---|" * len(hs))
    for k in range(len(res[hs[0]][0])):
        cells = []
        for h in hs:
            s, ree, n1, se, _, ry = res[h][0][k]
            cells.append(f"{ree:.4f} | {ry:.4f} | {n1:.4g} +- {se:.2g}")
        print(f"| {res[hs[0]][0][k][0]:.3f} | " + " | ".join(cells) + " |")
    if len(hs) >= 2:
        a, b = res[hs[0]], res[hs[1]]
        ra, rb = np.array([r[1] for r in a[0]]), np.array([r[1] for r in b[0]])
        na, nb = np.array([r[2] for r in a[0]]), np.array([r[2] for r in b[0]])
        print(f"\nh* = {hs[0]:g} against h* = {hs[1]:g}: max relative difference of R_ee(strain) = {np.max(np.abs(ra - rb) / rb):.3g}, "
              f"of N_1 = {np.max(np.abs(na - nb) / np.maximum(np.abs(nb), 1.0)):.3g}, "
              f"largest single-chain difference of |R| = {np.max(np.abs(a[1] - b[1])):.3g} b")


if __name__ == "__main__":
    main()
