"""GPU parity (``-m gpu``) of the Cohen-Pade bead-spring option (SURVEY.md 8(f) f4; PAPER.md:78-82 Eq. 4, :305-307):
spring law and semi-implicit cubic in every kernel that carries them (forces, update, observables, the fused per-chain
kernel) against the oracle; assemble / Cholesky / L dW are shared with the bead-rod chain.  The paper's BS-20-25 pairing
h* = 0.105, a* = 1.539 is used."""
import math

import numpy as np
import pytest
import torch
from scipy import integrate

import oracle as O
from paper_2208_06559_b200 import workloads as W

pytestmark = pytest.mark.gpu

BS = dict(hstar=0.105, a=1.539, spring_kind=1, nu=25.0)
KAPPA = np.array([[0.3, 1.0, 0.0], [0.0, -0.1, 0.2], [0.5, 0.0, -0.2]]) * 0.1


def _bd(N, C, dt, **kw):
    from paper_2208_06559_b200.binding import BD
    return BD(n_rods=N, n_chains=C, dt=dt, **kw)


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def _host(t):
    torch.cuda.synchronize()
    return t.cpu().numpy()


@pytest.mark.parametrize("path", [1, 2])
@pytest.mark.parametrize("N,C", [(1, 3), (20, 4), (100, 2)])
def test_one_step_positions_match_oracle(path, N, C):
    dt = 1e-3
    r0 = W.random_spring_chains(C, N, BS["nu"], seed=N)
    bd = _bd(N, C, dt, kappa=KAPPA, seed=3, **BS)
    bd.set_path(path)
    p = O.Params(n_rods=N, dt=dt, kappa=KAPPA, seed=3, **BS)
    r = r0.copy()
    for s in range(2):
        rg = _host(bd.step(_dev(r), first_step=s, n_steps=1))
        ro, info = O.step_ensemble(p, r, s, 1)
        assert not info.any() and bd.last_info() == (0, -1)
        for c in range(C):
            assert np.abs(rg[c] - ro[c]).max() / np.abs(ro[c]).max() <= 1e-10
            assert np.abs((rg[c] - r[c]) - (ro[c] - r[c])).max() / np.abs(ro[c] - r[c]).max() <= 1e-9
        r = ro


def test_forces_update_and_observables_match_oracle():
    N, C, dt = 20, 5, 1e-3
    par = dict(BS, b=1.5, nu=12.0)
    r = W.random_spring_chains(C, N, par["nu"], b=par["b"], seed=8, max_extension=0.97)
    bd = _bd(N, C, dt, kappa=KAPPA, **par)
    p = O.Params(n_rods=N, dt=dt, kappa=KAPPA, **par)
    T, F, v = [_host(x) for x in bd.drift(_dev(r))]
    per, ens = [_host(x) for x in bd.observables(_dev(r))]
    po, eo = O.observables(p, r)
    assert np.allclose(per, po, rtol=1e-11, atol=1e-9) and np.allclose(ens, eo, rtol=1e-11, atol=1e-9)
    rng = np.random.default_rng(1)
    M = 3 * (N + 1)
    vv = rng.standard_normal((C, M)) * 5.0
    yy = rng.standard_normal((C, M)) * math.sqrt(2 * dt) * 40.0
    yy[:, 3 * 7:3 * 7 + 3] += 40.0                                       # one bead kicked far: |Y| beyond full extension
    rg = _host(bd.update(_dev(r), _dev(vv), _dev(yy)))
    Lfull = par["nu"] * par["b"]
    beyond = 0
    for c in range(C):
        To = O.spring_tensions(p, r[c]); Fo = O.bead_forces(N, To)
        sc = np.abs(To).max()
        assert np.abs(T[c] - To).max() <= 1e-12 * sc and np.abs(F[c] - Fo).max() <= 1e-12 * sc
        ro, u, Y, info = O.finish_step(p, r[c], To, vv[c], yy[c])
        assert info == 0 and np.abs(rg[c] - ro).max() <= 1e-11 * np.abs(ro).max()
        assert np.linalg.norm(np.diff(rg[c], axis=0), axis=1).max() < Lfull          # finite extensibility
        beyond += (np.linalg.norm(Y, axis=1) > Lfull).sum()
    assert beyond > 0


def test_rejects_bad_spring_parameters():
    from paper_2208_06559_b200.binding import BDError
    with pytest.raises(BDError):
        _bd(5, 1, 1e-3, spring_kind=1, nu=0.0)
    with pytest.raises(BDError):
        _bd(5, 1, 1e-3, spring_kind=2, nu=1.0)


def test_dumbbell_equilibrium_on_the_gpu():
    """free-draining Cohen-Pade dumbbells on the fused path: <Q^2> against the quadrature of
    P(x) ~ x^2 exp(-nu x^2/2) (1 - x^2)^nu (the pin of the oracle, here with 65536 chains)."""
    nu, C = 10.0, 65536
    w = lambda x: x * x * math.exp(-nu * x * x / 2) * (1 - x * x) ** nu
    m2 = integrate.quad(lambda x: x * x * w(x), 0, 1)[0] / integrate.quad(w, 0, 1)[0] * nu * nu
    bd = _bd(1, C, 2e-3, hstar=0.0, spring_kind=1, nu=nu, seed=4)
    r = bd.init_random_walk(9)
    bd.step(r, 0, 4000)
    per = _host(bd.observables(r)[0])
    assert bd.last_info() == (0, -1)
    Q2 = per[:, 0]
    assert abs(Q2.mean() - m2) < 4 * Q2.std() / math.sqrt(C) + 0.01 * m2
    assert Q2.max() < nu * nu
