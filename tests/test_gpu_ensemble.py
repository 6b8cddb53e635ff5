"""GPU ensemble statistics (``-m gpu``): BASELINE.json asks that ensemble observables agree with the oracle within
3 standard errors.  One-step parity is deterministic (same noise, same state); here the two sides run FREE and with
INDEPENDENT noise (different Philox seeds), so that only the statistics can agree:

  * startup uniaxial extension (kappa = diag(e, -e/2, -e/2), reading A4) from equilibrium random walks:
    ensemble means of R^2, R_x^2, R_g^2 and S_xx after the run, GPU ensemble against oracle ensemble, difference
    within 3 combined standard errors; the fused kernel (all steps inside one launch) and the staged kernels both;
  * equilibrium (no flow): <R^2> = N b^2 with and without HI (oracle pin P8) within 3 standard errors
    plus the O(sqrt(dt)) Fraenkel rod stretch allowance used by the oracle's own pin.
Per-chain observables come from ``bd_observables`` / ``orc_observables``; SE = std over chains / sqrt(chains).
"""
import numpy as np
import pytest
import torch

import oracle as O
from paper_2208_06559_b200 import workloads as W

pytestmark = pytest.mark.gpu

OBS = {"R2": 0, "Rx2": 1, "Rg2": 4, "Sxx": 5}


def _gpu_run(N, C, dt, kappa, seed, steps, path, hstar=0.25, init_seed=77):
    from paper_2208_06559_b200.binding import BD
    bd = BD(n_rods=N, n_chains=C, dt=dt, hstar=hstar, kappa=kappa, seed=seed)
    bd.set_workspace()
    bd.set_path(path)
    r = bd.init_random_walk(init_seed)
    bd.step(r, first_step=0, n_steps=steps)
    per, _ = bd.observables(r)
    torch.cuda.synchronize()
    assert bd.last_info() == (0, -1)
    return per.cpu().numpy()


def _oracle_run(N, C, dt, kappa, seed, steps, hstar=0.25, init_seed=78):
    p = O.Params(n_rods=N, dt=dt, hstar=hstar, kappa=kappa, seed=seed)
    r = O.init_random_walk(N, 1.0, init_seed, range(C))
    r, info = O.step_ensemble(p, r, 0, steps)
    assert not info.any()
    return O.observables(p, r)[0]


def _mean_se(per, k):
    x = per[:, k]
    return x.mean(), x.std(ddof=1) / np.sqrt(len(x))


@pytest.mark.parametrize("path,name", [(2, "fused"), (1, "staged")])
def test_startup_extension_statistics_match_oracle(path, name):
    N, dt, steps, rate = 20, 1e-3, 400, 2.0                      # t = 0.4, strain 0.8: the chains stretch visibly
    kappa = np.diag([rate, -0.5 * rate, -0.5 * rate])
    gpu = _gpu_run(N, 2048 if path == 2 else 512, dt, kappa, seed=11, steps=steps, path=path)
    orc = _oracle_run(N, 512, dt, kappa, seed=12, steps=steps)
    for nm, k in OBS.items():
        mg, sg = _mean_se(gpu, k)
        mo, so = _mean_se(orc, k)
        assert abs(mg - mo) <= 3.0 * np.hypot(sg, so), (name, nm, mg, mo, sg, so)
    # the flow did something: R_x^2 grew well beyond its equilibrium value N b^2 / 3
    assert _mean_se(gpu, OBS["Rx2"])[0] > 1.5 * N / 3.0


@pytest.mark.parametrize("hstar", [0.0, 0.25])
def test_equilibrium_end_to_end_distance(hstar):
    N, C, dt, steps = 20, 4096, 1e-3, 200
    per = _gpu_run(N, C, dt, None, seed=5, steps=steps, path=2, hstar=hstar)
    m, se = _mean_se(per, OBS["R2"])
    # stiff Fraenkel rods sit slightly above b: |Q| - b has mean ~ 2 dt and spread sqrt(dt/2) (oracle pin P7)
    assert abs(m - N) <= 3.0 * se + 0.02 * N, (hstar, m, se)
    # isotropy: the three components share <R^2> equally
    comps = [_mean_se(per, k) for k in (1, 2, 3)]
    for mc, sc in comps:
        assert abs(mc - m / 3.0) <= 3.0 * np.hypot(sc, se / 3.0) + 0.01 * N, (hstar, mc, m)
