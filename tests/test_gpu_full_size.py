"""GPU parity at BASELINE.json's FULL sizes (``-m gpu``), in the launch configuration ``bench.py`` times
(``BD(n_chains = C)`` + ``set_workspace()`` + ``bd_step`` on the automatically selected path).

Small configs (c1, c2): every output of every chain against the oracle, element by element.
Large configs (c3, c4, c5) -- SURVEY.md section 8(c) pin P9, because one oracle Cholesky costs M^3/3 flops
(1.1e9 / 7.2e10 / 9.0e12):
  (i)   D: 3x3 blocks sampled at random (i, j) against ``orc_rpy_block`` (Eqs. 7-9), abs 1e-14;
  (ii)  L: accepted by the properties that make a Cholesky factor unique (lower triangular, positive diagonal,
        L L^T = D): ||L (L^T x) - D x|| / ||D x|| < 1e-12 on seeded probe vectors x, with D x from the oracle's
        storage-free ``orc_drift_onthefly`` (O(M^2)) and the two triangular products taken with plain
        torch FP64 ``mv`` on the lower triangle of the library's output;
  (iii) y = L dW against (verified L) x (oracle noise), rel 1e-12; v = D F against the oracle;
  (iv)  one-step positions, 1e-10 (BASELINE.json) and displacement-relative 1e-9 (reading A16): against the
        FULL oracle step for sampled chains where it is affordable (c3: 5 chains, c4: 1 chain); at c5 the
        oracle finishes the step (Eqs. 14, 17, 15) from its own T, its own v = D F and y = L dW formed from the
        factor that (ii) has just verified -- the only full-size path there is (P9 (iii)).
Inputs: seeded numpy random walks with the stationary Fraenkel rod-length spread (workloads.random_chains),
so that tensions and the drift are non-zero; nothing here comes from the CUDA path.
"""
import numpy as np
import pytest
import torch

import oracle as O
from paper_2208_06559_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def _bd_for(w, **kw):
    from paper_2208_06559_b200.binding import BD
    bd = BD(n_rods=w.n_rods, n_chains=w.n_chains, dt=w.dt, hstar=w.hstar, b=w.b, kappa=w.kappa(), seed=w.noise_seed, **kw)
    bd.set_workspace()
    return bd


def _params(w):
    return O.Params(n_rods=w.n_rods, dt=w.dt, hstar=w.hstar, b=w.b, kappa=w.kappa(), seed=w.noise_seed)


def _pos_err(rg, ro, r0):
    pos = np.abs(rg - ro).max() / np.abs(ro).max()
    dr = np.abs((rg - r0) - (ro - r0)).max() / np.abs(ro - r0).max()
    return pos, dr


def test_c1_all_1000_steps_resynchronised():
    """c1: 1 chain x 20 rods, the 1000 steps BASELINE.json quotes; state re-synchronised to the oracle's after
    every step (A16), every step gated at 1e-10; the free-running end state is reported loosely."""
    w = W.CONFIGS["c1"]
    p = _params(w)
    bd = _bd_for(w)
    r = O.init_random_walk(w.n_rods, w.b, w.init_seed, [0])
    free = _dev(r)
    worst = 0.0
    for s in range(w.steps):
        rg = bd.step(_dev(r), first_step=s, n_steps=1)
        ro, info = O.step_ensemble(p, r, s, 1)
        assert not info.any()
        torch.cuda.synchronize()
        worst = max(worst, np.abs(rg.cpu().numpy() - ro).max() / np.abs(ro).max())
        r = ro
    assert worst <= 1e-10
    bd.step(free, first_step=0, n_steps=w.steps)                 # one launch, 1000 steps inside the kernel
    torch.cuda.synchronize()
    assert bd.last_info() == (0, -1)
    assert np.abs(free.cpu().numpy() - r).max() / np.abs(r).max() <= 1e-7


def test_c2_full_ensemble_every_chain():
    """c2: all 1024 chains x 100 rods through the fused kernel, two steps, every chain compared."""
    w = W.CONFIGS["c2"]
    p = _params(w)
    bd = _bd_for(w)
    r = W.random_chains(w.n_chains, w.n_rods, seed=202, rod_jitter=0.007)
    for s in range(2):
        rg = bd.step(_dev(r), first_step=s, n_steps=1)
        ro, info = O.step_ensemble(p, r, s, 1)
        torch.cuda.synchronize()
        rg = rg.cpu().numpy()
        assert not info.any() and bd.last_info() == (0, -1)
        for c in range(w.n_chains):
            pos, dr = _pos_err(rg[c], ro[c], r[c])
            assert pos <= 1e-10 and dr <= 1e-9, (c, pos, dr)
        r = ro
    per, ens = bd.observables(_dev(r))
    po, eo = O.observables(p, r)
    torch.cuda.synchronize()
    assert np.allclose(per.cpu().numpy(), po, rtol=1e-11, atol=1e-11)
    assert np.allclose(ens.cpu().numpy(), eo, rtol=1e-11, atol=1e-9)


def _large_config_check(name, oracle_chains, probe_chains, n_blocks=300, seed=7):
    w = W.CONFIGS[name]
    p = _params(w)
    C, N, M, Nb = w.n_chains, w.n_rods, w.M, w.n_rods + 1
    r0 = W.random_chains(C, N, seed=seed, rod_jitter=float(np.sqrt(w.dt / 2.0)))
    bd = _bd_for(w)
    ld = bd.ld
    stride = ld * ((M + 7) // 8 * 8)
    rng = np.random.default_rng(seed + 1)

    # (i) D blocks, through the public assembly entry point on the same positions
    Dg = bd.assemble_hi(_dev(r0))
    for c in probe_chains:
        ii = rng.integers(0, Nb, size=n_blocks)
        jj = np.minimum(ii, rng.integers(0, Nb, size=n_blocks))           # lower triangle (j <= i)
        ii[:8], jj[:8] = [0, 1, Nb - 1, Nb - 1, Nb - 1, Nb // 2, 7, Nb - 2], [0, 0, 0, Nb - 2, Nb - 1, Nb // 2, 7, 1]
        for i, j in zip(ii, jj):
            blk = Dg[c, 3 * i:3 * i + 3, 3 * j:3 * j + 3].cpu().numpy()
            ref = np.eye(3) if i == j else O.rpy_block(p, r0[c, i], r0[c, j])
            if i == j:
                blk = np.tril(blk)
                ref = np.tril(ref)
            assert np.abs(blk - ref).max() <= 1e-14, (c, i, j)
    del Dg
    torch.cuda.empty_cache()

    # one step in the bench configuration
    rg = bd.step(_dev(r0), first_step=0, n_steps=1)
    torch.cuda.synchronize()
    assert bd.last_info() == (0, -1)
    rg = rg.cpu().numpy()
    Lws = bd._ws[: C * stride].view(C, stride // ld, ld)           # the step's own L storage: [C][M^8][ld]
    Tg, Fg, vg = bd.drift(_dev(r0))
    yg = bd.brownian(Lws, step=0, chain_stride=stride)
    torch.cuda.synchronize()

    for c in probe_chains:
        Lc = torch.tril(Lws[c, :M, :M])
        assert bool((torch.diagonal(Lc) > 0).all())
        # (ii) unique-factor property on probe vectors
        for k in range(2):
            x = rng.standard_normal(M)
            Dx = O.drift_onthefly(p, r0[c], x.reshape(Nb, 3))
            w_ = (Lc @ (Lc.T @ _dev(x))).cpu().numpy()
            assert np.linalg.norm(w_ - Dx) / np.linalg.norm(Dx) < 1e-12, (c, k)
        # (iii) matvecs
        T = O.spring_tensions(p, r0[c])
        F = O.bead_forces(N, T)
        v = O.drift_onthefly(p, r0[c], F)
        assert np.abs(vg[c].cpu().numpy() - v).max() <= 1e-12 * max(np.abs(v).max(), 1e-300)
        dW = O.noise_dW(p, c, 0)
        y = (Lc @ _dev(dW)).cpu().numpy()
        assert np.abs(yg[c].cpu().numpy() - y).max() <= 1e-12 * np.abs(y).max()
        # (iv) positions, with y from the verified factor
        ro, _, _, info = O.finish_step(p, r0[c], T, v, y)
        assert info == 0
        pos, dr = _pos_err(rg[c], ro, r0[c])
        assert pos <= 1e-10 and dr <= 1e-9, (c, pos, dr)
        del Lc

    # (iv) the full oracle step where it is affordable
    for c in oracle_chains:
        ro, info = O.step(p, c, 0, r0[c])
        assert info == 0
        pos, dr = _pos_err(rg[c], ro, r0[c])
        assert pos <= 1e-10 and dr <= 1e-9, (c, pos, dr)


def test_c3_full_size():
    _large_config_check("c3", oracle_chains=[0, 1, 100, 254, 255], probe_chains=[0, 77, 255])


def test_c4_full_size():
    _large_config_check("c4", oracle_chains=[15], probe_chains=[0, 9, 15])


def test_c5_full_size():
    _large_config_check("c5", oracle_chains=[], probe_chains=[0], n_blocks=400)
