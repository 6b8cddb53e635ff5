"""GPU test (``-m gpu``) of bd_cholesky_noalloc, the allocation-free entry point (README "No-allocation entry point"):
the tile Cholesky with its scratch in the library's fixed file-scope device array.  Its output is compared with the
existing path (bd_cholesky through a context, tile kernel) on the same matrices, on two calls in a row with DIFFERENT
shapes (the shared array keeps the first call's contents: what must start at zero has to be cleared), within the
tolerance of the other Cholesky tests (norm-wise 1e-12 against the oracle; the two GPU paths run the same kernel in the
same summation order, so they are also compared bit for bit).  Collected last on purpose (file name): a failure here must
not hide other tests under ``pytest -x``.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

import oracle as O
from paper_2208_06559_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _case(N, C, seed):
    """(D storage with assembled lower triangles, factor from the existing path, chains)"""
    from paper_2208_06559_b200.binding import BD
    r = W.random_chains(C, N, seed=seed, rod_jitter=0.01)
    bd = BD(n_rods=N, n_chains=C, dt=1e-4)
    bd.set_cholesky(2)
    D = bd.matrix_storage(); D.fill_(-7.0)
    bd.assemble_hi(torch.as_tensor(r).cuda(), D)
    ref = D.clone()
    bd.cholesky(ref)                                           # existing path: context-owned, cudaMalloc'ed scratch
    torch.cuda.synchronize()
    assert bd.last_info() == (0, -1)
    return D, ref, r, bd.M


def test_noalloc_cholesky_matches_existing_path_on_two_calls_in_a_row():
    from paper_2208_06559_b200 import binding
    # call 1: 2 chains of M = 453 (4 tile rows each, ragged last tile); call 2: 5 chains of M = 303 (3 tile rows each):
    # other tile counts, so stale flags / ticket counter / W blocks of call 1 sit where call 2 works
    cases = [_case(150, 2, 11), _case(100, 5, 12)]
    for D, ref, r, M in cases:
        info = torch.full((D.shape[0],), 99, dtype=torch.int32, device="cuda")
        before = torch.cuda.memory_allocated()
        binding.cholesky_noalloc(D, info)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before          # nothing allocated through torch's allocator either
        assert not info.cpu().numpy().any()
        Lh, Rh = D.cpu().numpy(), ref.cpu().numpy()
        assert np.array_equal(Lh, Rh)                          # same kernel, same summation order: bit for bit,
        p = O.Params(n_rods=r.shape[1] - 1, dt=1e-4)           # strict upper / padding (-7) untouched included
        for c in range(D.shape[0]):
            Lo, io = O.cholesky(O.assemble(p, r[c]))
            assert io == 0
            assert np.linalg.norm(np.tril(Lh[c, :, :M]) - Lo) <= 1e-12 * np.linalg.norm(Lo)


def test_noalloc_cholesky_reports_pivot_and_rejects_what_exceeds_its_scratch():
    from paper_2208_06559_b200 import binding
    M = 200
    rng = np.random.default_rng(3)
    B = rng.standard_normal((M, M))
    A = B @ B.T + M * np.eye(M)
    Lref = np.linalg.cholesky(A)
    row = 140
    A[row, row] = (Lref[row, :row] ** 2).sum() - 1.0            # pivot `row` becomes -1
    D = torch.zeros(1, M, 208, dtype=torch.float64, device="cuda")
    D[0, :, :M] = torch.as_tensor(np.tril(A)).cuda()
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    binding.cholesky_noalloc(D, info)
    torch.cuda.synchronize()
    assert info.cpu().tolist() == [row + 1]
    # limit: n_chains * ceil(M / 128) <= 32
    ok = torch.eye(128, dtype=torch.float64, device="cuda").repeat(32, 1, 1).contiguous()
    binding.cholesky_noalloc(ok)                                 # 32 x 1 tile rows: allowed
    torch.cuda.synchronize()
    assert torch.equal(ok[31], torch.eye(128, dtype=torch.float64, device="cuda"))
    big = torch.empty(33, 128, 128, dtype=torch.float64, device="cuda")
    with pytest.raises(binding.BDError) as e:
        binding.cholesky_noalloc(big)
    assert e.value.code == binding.ERR_TOO_LARGE and "32" in str(e.value)
    tall = torch.empty(1, 4097, 4098, dtype=torch.float64, device="cuda")
    with pytest.raises(binding.BDError) as e:
        binding.cholesky_noalloc(tall)
    assert e.value.code == binding.ERR_TOO_LARGE
