"""GPU parity (``-m gpu``) of the two Cholesky implementations behind bd_cholesky (bd_set_cholesky): 1 = blocked
right-looking, one launch per block operation (potrf.cu); 2 = the persistent left-looking tile kernel (potrf_tiles.cu:
TMA-fed DMMA tiles, ticket counter, ready flags).  Both against the oracle's row-by-row Cholesky (Eq. 10,
PAPER.md:116-118) at sizes that cover one tile, ragged last tiles of every width class, several tile columns and
several chains; tolerances as in test_gpu_parity.py."""
import numpy as np
import pytest
import torch

import oracle as O
from paper_2208_06559_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _bd(N, C, **kw):
    from paper_2208_06559_b200.binding import BD
    return BD(n_rods=N, n_chains=C, dt=1e-4, **kw)


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def _host(t):
    torch.cuda.synchronize()
    return t.cpu().numpy()


# M = 6, 63, 129 (one full tile + 1 row), 192, 258, 387 (3 tiles + 3), 513, 1026, 1365
@pytest.mark.parametrize("algo", [1, 2])
@pytest.mark.parametrize("N,C", [(1, 2), (20, 3), (42, 2), (63, 1), (85, 3), (128, 2), (170, 2), (341, 2), (454, 1)])
def test_cholesky_both_algorithms_match_oracle(algo, N, C):
    r = W.random_chains(C, N, seed=700 + N, rod_jitter=0.01)
    bd = _bd(N, C)
    bd.set_cholesky(algo)
    M = bd.M
    p = O.Params(n_rods=N, dt=1e-4)
    DL = bd.matrix_storage(); DL.fill_(-7.0)
    bd.assemble_hi(_dev(r), DL)
    info = torch.full((C,), 99, dtype=torch.int32, device="cuda")
    bd.cholesky(DL, info)
    Lh = _host(DL)
    assert not _host(info).any()
    for c in range(C):
        D = O.assemble(p, r[c])
        Lo, io = O.cholesky(D)
        assert io == 0
        L = np.tril(Lh[c, :, :M])
        assert np.linalg.norm(L - Lo) <= 1e-12 * np.linalg.norm(Lo)
        assert np.linalg.norm(L @ L.T - D) < 1e-12 * np.linalg.norm(D)
        assert np.all(np.diag(L) > 0)
        assert np.all(Lh[c, :, :M][np.triu_indices(M, 1)] == -7.0)      # strict upper never written
        assert np.all(Lh[c, :, M:] == -7.0)                              # padding columns never written


def test_tile_kernel_repeated_calls_and_storage_change():
    """flags are reused through an epoch counter and tickets through a running base: repeated factorisations, with
    a second storage (new tensor map) in between, give the same factor bit for bit."""
    N, C = 200, 3
    r = W.random_chains(C, N, seed=3, rod_jitter=0.01)
    bd = _bd(N, C)
    bd.set_cholesky(2)
    outs = []
    for k in range(4):
        DL = bd.matrix_storage(ld=bd.ld + (16 if k == 2 else 0))
        bd.assemble_hi(_dev(r), DL)
        bd.cholesky(DL)
        outs.append(np.tril(_host(DL)[:, :, :bd.M]))
    for o in outs[1:]:
        assert np.array_equal(o, outs[0])


@pytest.mark.parametrize("row", [5, 70, 130, 200, 300])
def test_tile_kernel_reports_failing_pivot_row(row):
    """a matrix that stops being positive definite at a given row: info = that 1-based row, on every chain alike."""
    M, N = 303, 100
    rng = np.random.default_rng(row)
    B = rng.standard_normal((M, M))
    A = B @ B.T + M * np.eye(M)
    Lref = np.linalg.cholesky(A)
    A[row, row] = (Lref[row, :row] ** 2).sum() - 1.0                     # pivot `row` becomes -1
    bd = _bd(N, 2)
    bd.set_cholesky(2)
    DL = bd.matrix_storage()
    DL[:, :, :M] = _dev(np.tril(A))
    info = torch.zeros(2, dtype=torch.int32, device="cuda")
    bd.cholesky(DL, info)
    assert _host(info).tolist() == [row + 1, row + 1]
    Lo, io = O.cholesky(A)
    assert io == row + 1


@pytest.mark.parametrize("algo", [1, 2])
def test_staged_step_with_either_cholesky(algo):
    N, C, dt = 150, 3, 1e-4
    r0 = W.random_chains(C, N, seed=12, rod_jitter=0.007)
    kap = W.CONFIGS["c3"].kappa() * 30
    bd = _bd(N, C, kappa=kap, seed=4)
    bd.set_path(1)
    bd.set_cholesky(algo)
    rg = _host(bd.step(_dev(r0), 0, 1))
    ro, info = O.step_ensemble(O.Params(n_rods=N, dt=dt, kappa=kap, seed=4), r0, 0, 1)
    assert not info.any() and bd.last_info() == (0, -1)
    assert np.abs(rg - ro).max() / np.abs(ro).max() <= 1e-10


def test_two_contexts_on_two_streams_factor_concurrently():
    """every context owns its flags, ticket counter and inverse blocks, and a tile only waits for tiles with smaller
    tickets of its OWN launch: two persistent tile kernels in flight on two streams finish and agree with the oracle."""
    from paper_2208_06559_b200.binding import BD
    N, C = 300, 2
    r = W.random_chains(2 * C, N, seed=77, rod_jitter=0.01)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    bds, Ds = [], []
    for k, st in enumerate(streams):
        with torch.cuda.stream(st):
            bd = BD(n_rods=N, n_chains=C, dt=1e-4, stream=st)
            bd.set_cholesky(2)
            D = bd.matrix_storage()
            bd.assemble_hi(_dev(r[k * C:(k + 1) * C]), D)
            bds.append(bd); Ds.append(D)
    torch.cuda.synchronize()
    for rep in range(3):                                  # launches interleave on the two streams
        for bd, D, st in zip(bds, Ds, streams):
            with torch.cuda.stream(st):
                if rep:
                    bd.assemble_hi(_dev(r[bds.index(bd) * C:(bds.index(bd) + 1) * C]), D)
                bd.cholesky(D)
    torch.cuda.synchronize()
    p = O.Params(n_rods=N, dt=1e-4)
    for k, (bd, D) in enumerate(zip(bds, Ds)):
        assert bd.last_info() == (0, -1)
        Lh = _host(D)
        for c in range(C):
            Lo, io = O.cholesky(O.assemble(p, r[k * C + c]))
            assert io == 0 and np.linalg.norm(np.tril(Lh[c, :, :bd.M]) - Lo) <= 1e-12 * np.linalg.norm(Lo)
