"""GPU parity (``-m gpu``) away from the default parameter corner: every kernel carries b, a, K,
h* and chain_id0, so each is compared with the oracle at b != 1, a != h* b, K != 1/dt and a non-zero global chain
id, on the staged AND the fused path; sharding over contexts must be exact to the bit.
Tolerances as in test_gpu_parity.py."""
import math

import numpy as np
import pytest
import torch

import oracle as O
from paper_2208_06559_b200 import workloads as W

pytestmark = pytest.mark.gpu

PATHS = [(1, "staged"), (2, "fused")]
KAPPA = np.array([[0.3, 1.0, -0.4], [0.2, -0.1, 0.2], [0.5, -0.6, -0.2]])
ODD = dict(b=2.0, a=0.7, K=4000.0, hstar=0.3)          # h* b / a = 0.857 <= 1 (reading A3), K dt = 0.4


def _bd(N, C, dt=1e-4, **kw):
    from paper_2208_06559_b200.binding import BD
    return BD(n_rods=N, n_chains=C, dt=dt, **kw)


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def _host(t):
    torch.cuda.synchronize()
    return t.cpu().numpy()


@pytest.mark.parametrize("path,name", PATHS)
@pytest.mark.parametrize("N,C", [(3, 2), (40, 3), (100, 4)])
def test_one_step_off_default_parameters(path, name, N, C):
    dt = 1e-4
    r0 = W.random_chains(C, N, b=ODD["b"], seed=N, rod_jitter=0.01)
    bd = _bd(N, C, dt, kappa=KAPPA * 0.05, seed=9, **ODD)
    bd.set_path(path)
    p = O.Params(n_rods=N, dt=dt, kappa=KAPPA * 0.05, seed=9, **ODD)
    r = r0.copy()
    for s in range(2):
        rg = _host(bd.step(_dev(r), first_step=s, n_steps=1))
        ro, info = O.step_ensemble(p, r, s, 1)
        assert not info.any() and bd.last_info() == (0, -1)
        for c in range(C):
            assert np.abs(rg[c] - ro[c]).max() / np.abs(ro[c]).max() <= 1e-10
            assert np.abs((rg[c] - r[c]) - (ro[c] - r[c])).max() / np.abs(ro[c] - r[c]).max() <= 1e-9
        r = ro


@pytest.mark.parametrize("N,C", [(2, 2), (42, 3), (170, 2)])
def test_stages_with_b_a_K_off_default(N, C):
    """assemble, drift, Cholesky + L dW, update and observables with b = 1.7, a = 0.6, h* = 0.3, K = 777."""
    par = dict(b=1.7, a=0.6, hstar=0.3, K=777.0)
    dt = 2e-4
    r = W.random_chains(C, N, b=par["b"], seed=50 + N, rod_jitter=0.02)
    bd = _bd(N, C, dt, kappa=KAPPA, seed=4, chain_id0=3, **par)
    p = O.Params(n_rods=N, dt=dt, kappa=KAPPA, seed=4, **par)
    M = bd.M
    D = bd.matrix_storage()
    bd.assemble_hi(_dev(r), D)
    Dh = _host(D)
    T, F, v = [_host(x) for x in bd.drift(_dev(r))]
    bd.cholesky(D)
    Lh = _host(D)
    y = _host(bd.brownian(D, step=6))
    per, ens = [_host(x) for x in bd.observables(_dev(r))]
    po, eo = O.observables(p, r)
    assert np.allclose(per, po, rtol=1e-11, atol=1e-9) and np.allclose(ens, eo, rtol=1e-11, atol=1e-9)
    rng = np.random.default_rng(N)
    vv = rng.standard_normal((C, M)) * 20.0
    yy = rng.standard_normal((C, M)) * math.sqrt(2 * dt)
    rg = _host(bd.update(_dev(r), _dev(vv), _dev(yy)))
    for c in range(C):
        Do = O.assemble(p, r[c])
        assert np.abs(np.tril(Dh[c, :, :M]) - np.tril(Do)).max() <= 1e-14
        To = O.spring_tensions(p, r[c]); Fo = O.bead_forces(N, To); vo = O.drift_onthefly(p, r[c], Fo)
        sc = np.abs(To).max()
        assert np.abs(T[c] - To).max() <= 1e-12 * sc and np.abs(F[c] - Fo).max() <= 1e-12 * sc
        assert np.abs(v[c].reshape(-1) - vo).max() <= 1e-12 * max(np.abs(vo).max(), sc)
        Lo, info = O.cholesky(Do)
        assert info == 0
        assert np.linalg.norm(np.tril(Lh[c, :, :M]) - Lo) <= 1e-12 * np.linalg.norm(Lo)
        yo = O.trmv_lower(Lo, O.noise_dW(p, 3 + c, 6))
        assert np.abs(y[c] - yo).max() <= 1e-12 * np.abs(yo).max()
        ro, u, Y, info = O.finish_step(p, r[c], To, vv[c], yy[c])
        assert info == 0 and np.abs(rg[c] - ro).max() <= 1e-12 * np.abs(ro).max()


@pytest.mark.parametrize("path,name", PATHS)
def test_step_with_nonzero_global_chain_id(path, name):
    N, C, dt, id0 = 60, 5, 1e-4, 12345
    r0 = W.random_chains(C, N, seed=77, rod_jitter=0.007)
    bd = _bd(N, C, dt, kappa=KAPPA * 0.02, seed=21, chain_id0=id0)
    bd.set_path(path)
    p = O.Params(n_rods=N, dt=dt, kappa=KAPPA * 0.02, seed=21)
    rg = _host(bd.step(_dev(r0), first_step=3, n_steps=1))
    ro, info = O.step_ensemble(p, r0, 3, 1, chain0=id0)
    assert not info.any()
    assert np.abs(rg - ro).max() / np.abs(ro).max() <= 1e-10
    r_wrong, _ = O.step_ensemble(p, r0, 3, 1, chain0=0)                 # the id really enters the noise
    assert np.abs(rg - r_wrong).max() > 1e-4


@pytest.mark.parametrize("N,C,path", [(30, 600, 2), (30, 40, 1), (120, 6, 0)])
def test_sharded_contexts_equal_one_context_bit_for_bit(N, C, path):
    """f2 / SURVEY.md 8(e): chains (0 .. C/2-1) and (C/2 .. C-1) in two contexts with chain_id0 = 0 and C/2 give
    exactly the positions and ensemble sums of one context with all C chains (C = 600 > 296 resident CTAs on the
    fused path; N = 120 is past the fused limit, path 0 = automatic = staged)."""
    dt, steps, h = 1e-4, 3, C // 2
    r0 = W.random_chains(C, N, seed=5, rod_jitter=0.007)
    kap = W.CONFIGS["c2"].kappa() * 50
    whole = _bd(N, C, dt, kappa=kap, seed=8)
    whole.set_path(path)
    rw = _host(whole.step(_dev(r0), 0, steps))
    ens_w = _host(whole.observables(_dev(rw))[1])
    parts, ens = [], np.zeros((2, 13))
    for k in range(2):
        bd = _bd(N, h, dt, kappa=kap, seed=8, chain_id0=k * h)
        bd.set_path(path)
        rp = bd.step(_dev(r0[k * h:(k + 1) * h]), 0, steps)
        parts.append(_host(rp))
        ens += _host(bd.observables(rp)[1])
    assert np.array_equal(np.concatenate(parts), rw)
    assert np.allclose(ens, ens_w, rtol=1e-13, atol=0)                  # sums over chains in a different order
    ro, info = O.step_ensemble(O.Params(n_rods=N, dt=dt, kappa=kap, seed=8), r0[h - 1:h + 1], 0, 1, chain0=h - 1)
    first = _bd(N, 2, dt, kappa=kap, seed=8, chain_id0=h - 1)
    first.set_path(path)
    assert np.abs(_host(first.step(_dev(r0[h - 1:h + 1]), 0, 1)) - ro).max() / np.abs(ro).max() <= 1e-10


@pytest.mark.parametrize("path,name", PATHS)
def test_failed_chain_is_retried_every_step_and_first_failure_is_kept(path, name):
    """over a multi-step call a failing chain keeps its state and its FIRST failure code while the
    other chains move on, identically on both paths and in the oracle (orc_step_ensemble)."""
    N, steps = 20, 3
    r = W.random_chains(4, N, seed=9, rod_jitter=0.007)
    r[2, 5] = r[2, 1]                                                  # coincident beads: singular D (reading A10)
    p = O.Params(n_rods=N, dt=1e-4, seed=2)
    ro, info = O.step_ensemble(p, r, 0, steps)
    assert info[2] > 0 and not info[[0, 1, 3]].any() and np.array_equal(ro[2], r[2])
    bd = _bd(N, 4, seed=2)
    bd.set_path(path)
    rg = _host(bd.step(_dev(r), 0, steps))
    assert bd.last_info() == (1, 2)
    assert np.array_equal(rg[2], r[2])
    for c in (0, 1, 3):
        assert np.abs(rg[c] - ro[c]).max() / np.abs(ro[c]).max() <= 1e-9      # 3 free-running steps
    torch.cuda.synchronize()


def test_hundred_thousand_chains():
    """n_chains is not limited by a grid dimension: C = 100000 chains of 5 rods, fused bd_step and
    the staged stage entry points, sampled chains against the oracle."""
    N, C, dt = 5, 100_000, 1e-4
    bd = _bd(N, C, dt, seed=6)
    r0 = bd.init_random_walk(77)
    r0h = _host(r0).copy()
    p = O.Params(n_rods=N, dt=dt, seed=6)
    idx = [0, 1, 65534, 65535, 65536, 77777, C - 1]
    want0 = O.init_random_walk(N, 1.0, 77, idx)
    assert np.abs(r0h[idx] - want0).max() <= 1e-12
    rg = _host(bd.step(r0.clone(), 0, 1))
    assert bd.last_info()[0] == 0
    for c in idx:
        ro, info = O.step_ensemble(p, r0h[c:c + 1], 0, 1, chain0=c)
        assert info[0] == 0 and np.abs(rg[c] - ro[0]).max() / np.abs(ro[0]).max() <= 1e-10
    # staged entry points with the chain index beyond 65535
    D = bd.assemble_hi(r0)
    T, F, v = bd.drift(r0)
    bd.cholesky(D)
    y = bd.brownian(D, step=0)
    Lh, yh, vh = _host(D[idx]), _host(y[idx]), _host(v[idx])
    M = bd.M
    for k, c in enumerate(idx):
        Lo, info = O.cholesky(O.assemble(p, r0h[c]))
        assert info == 0 and np.linalg.norm(np.tril(Lh[k, :, :M]) - Lo) <= 1e-12 * np.linalg.norm(Lo)
        yo = O.trmv_lower(Lo, O.noise_dW(p, c, 0))
        assert np.abs(yh[k] - yo).max() <= 1e-12 * np.abs(yo).max()
        Fo = O.bead_forces(N, O.spring_tensions(p, r0h[c]))
        vo = O.drift_onthefly(p, r0h[c], Fo)
        assert np.abs(vh[k].reshape(-1) - vo).max() <= 1e-11        # unit rods: forces are rounding noise (~1e-12), absolute check
    bd1 = _bd(N, C, dt, seed=6)
    bd1.set_path(1)
    rs = _host(bd1.step(_dev(r0h), 0, 1))
    assert np.abs(rs - rg).max() <= 1e-11 * np.abs(rg).max()
