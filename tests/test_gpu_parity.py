"""GPU parity (``-m gpu``): every stage of libbd, called through the C ABI binding, against the CPU
oracle on the same seeded inputs, element by element.  Tolerances:
  D entries          abs 1e-14 (entries are O(1); the kernel uses rsqrt, the oracle sqrt + divisions)
  L                  norm-wise 1e-12, residual |LL^T - D|/|D| < 1e-12 (BASELINE.json)
  noise / y / v      relative 1e-12 (libm differences <= 2 ulp, summation order)
  one-step positions max_i|r_gpu - r_orc|_inf / max_i|r_orc|_inf <= 1e-10 (BASELINE.json, reading A16)
"""
import math

import numpy as np
import pytest
import torch

import oracle as O
from paper_2208_06559_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _bd(N, C, dt=1e-4, **kw):
    from paper_2208_06559_b200.binding import BD
    return BD(n_rods=N, n_chains=C, dt=dt, **kw)


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def _host(t):
    torch.cuda.synchronize()
    return t.cpu().numpy()


def _lower(Dg, M):
    """[C][M][ld] device storage -> [C][M][M] lower triangles."""
    return np.tril(_host(Dg)[:, :, :M])


KAPPA = np.array([[0.3, 1.0, 0.0], [0.0, -0.1, 0.2], [0.5, 0.0, -0.2]])
SIZES = [(1, 1), (2, 3), (20, 2), (21, 1), (42, 3), (100, 5), (170, 2), (300, 2)]


# ------------------------------------------------------------------------------------------ a0
@pytest.mark.parametrize("kind", [0, 1])
def test_noise_matches_oracle(kind):
    N, C, dt = 100, 4, 1e-4
    bd = _bd(N, C, dt, seed=0xDEADBEEF12345, chain_id0=7, noise_kind=kind)
    p = O.Params(n_rods=N, dt=dt, seed=0xDEADBEEF12345, noise_kind=kind)
    for step in (0, 5, (3 << 32) + 11):
        dW = _host(bd.noise(step))
        want = np.stack([O.noise_dW(p, 7 + c, step) for c in range(C)])
        assert np.allclose(dW, want, rtol=1e-13, atol=1e-17)


def test_init_random_walk_matches_oracle():
    for N, C in ((1, 2), (20, 3), (100, 4), (1000, 2)):
        bd = _bd(N, C, chain_id0=5)
        r = _host(bd.init_random_walk(1234))
        want = O.init_random_walk(N, 1.0, 1234, range(5, 5 + C))
        assert np.abs(r - want).max() <= 1e-12 * max(1.0, np.abs(want).max())


# ------------------------------------------------------------------------------------------ a1, a4
@pytest.mark.parametrize("N,C", SIZES)
def test_forces_and_drift_match_oracle(N, C):
    r = W.random_chains(C, N, seed=N, rod_jitter=0.01)
    bd = _bd(N, C, hstar=0.25)
    p = O.Params(n_rods=N, dt=1e-4)
    T, F, v = [_host(x) for x in bd.drift(_dev(r))]
    for c in range(C):
        To = O.spring_tensions(p, r[c]); Fo = O.bead_forces(N, To); vo = O.drift_onthefly(p, r[c], Fo)
        scale = np.abs(To).max()
        assert np.abs(T[c] - To).max() <= 1e-12 * scale
        assert np.abs(F[c] - Fo).max() <= 1e-12 * scale
        assert np.abs(v[c].reshape(-1) - vo).max() <= 1e-12 * max(np.abs(vo).max(), scale)


# ------------------------------------------------------------------------------------------ a2
@pytest.mark.parametrize("N,C", SIZES)
def test_assemble_matches_oracle(N, C):
    r = W.random_chains(C, N, seed=100 + N, rod_jitter=0.01)
    bd = _bd(N, C)
    M = bd.M
    p = O.Params(n_rods=N, dt=1e-4)
    D = bd.matrix_storage(); D.fill_(-7.0)
    bd.assemble_hi(_dev(r), D)
    Dh = _host(D)
    for c in range(C):
        want = O.assemble(p, r[c])
        assert np.abs(np.tril(Dh[c, :, :M]) - np.tril(want)).max() <= 1e-14
        assert np.all(Dh[c, :, :M][np.triu_indices(M, 1)] == -7.0)   # strict upper never written
        assert np.all(Dh[c, :, M:] == -7.0)                      # padding columns never written
    Df = bd.matrix_storage(ld=M + 1 + (M + 1) % 2); Df.fill_(-7.0)
    bd.assemble_hi(_dev(r), Df, full=True)
    Dfh = _host(Df)
    for c in range(C):
        assert np.abs(Dfh[c, :, :M] - O.assemble(p, r[c])).max() <= 1e-14
        assert np.all(Dfh[c, :, M:] == -7.0)


def test_assemble_exercises_both_rpy_branches_and_free_draining():
    N = 100
    r = W.random_chains(2, N, seed=5)
    p = O.Params(n_rods=N, dt=1e-4)
    d = np.linalg.norm(r[0][:, None] - r[0][None], axis=-1) + np.eye(N + 1)
    assert (d < 0.5).sum() > 0 and (d >= 0.5).sum() > 0          # Eq. 9 and Eq. 8 both occur
    bd0 = _bd(N, 2, hstar=0.0)
    D0 = _lower(bd0.assemble_hi(_dev(r)), 3 * (N + 1))
    assert np.array_equal(D0[0], np.eye(3 * (N + 1)))            # h* = 0 -> D = I exactly


# ------------------------------------------------------------------------------------------ a3
@pytest.mark.parametrize("N,C", SIZES)
def test_cholesky_matches_oracle(N, C):
    r = W.random_chains(C, N, seed=200 + N, rod_jitter=0.01)
    bd = _bd(N, C)
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
        Lg = np.tril(Lh[c, :, :M])
        assert np.all(np.diag(Lg) > 0)
        assert np.linalg.norm(Lg - Lo) / np.linalg.norm(Lo) <= 1e-12
        assert np.linalg.norm(Lg @ Lg.T - D) / np.linalg.norm(D) < 1e-12
        assert np.all(Lh[c, :, :M][np.triu_indices(M, 1)] == -7.0)   # strict upper untouched (LAPACK style)


def test_cholesky_on_general_spd_and_unpadded_ld():
    """not only RPY matrices: random SPD input, ld = M (+1 if odd) instead of the padded default."""
    rng = np.random.default_rng(3)
    for N in (20, 85, 127):
        M = 3 * (N + 1)
        ld = M + (M % 2)
        bd = _bd(N, 2)
        A = rng.standard_normal((2, M, M)); A = A @ A.transpose(0, 2, 1) + M * np.eye(M)
        buf = np.zeros((2, M, ld)); buf[:, :, :M] = A
        DL = _dev(buf)
        bd.cholesky(DL)
        Lg = np.tril(_host(DL)[:, :, :M])
        for c in range(2):
            assert np.linalg.norm(Lg[c] - np.linalg.cholesky(A[c])) / np.linalg.norm(Lg[c]) < 1e-13


@pytest.mark.parametrize("N", [341, 455, 699])
def test_cholesky_recursive_panels_and_trailing_update_against_oracle(N):
    """M = 1026, 1368, 2100: just past / well past the outer panel width (1024) -> trailing update + second panel, ragged
    recursion halves (M not a multiple of 64), general SPD input; expected factor from the oracle's row-by-row Cholesky."""
    M = 3 * (N + 1)
    rng = np.random.default_rng(N)
    G = rng.standard_normal((M, M)) / np.sqrt(M)
    A = G @ G.T + 0.5 * np.eye(M)
    bd = _bd(N, 1)
    buf = np.zeros((1, M, bd.ld)); buf[0, :, :M] = A
    DL = _dev(buf)
    bd.cholesky(DL)
    Lg = np.tril(_host(DL)[0, :, :M])
    Lo, info = O.cholesky(A)
    assert info == 0
    assert np.linalg.norm(Lg - Lo) / np.linalg.norm(Lo) <= 1e-12
    assert np.linalg.norm(Lg @ Lg.T - A) / np.linalg.norm(A) < 1e-12


@pytest.mark.parametrize("row", [5, 40, 70, 100, 190])
def test_cholesky_failing_pivot_row_in_every_part_of_a_block(row):
    """a non-positive pivot in the first / second half of the first 64-block, in the second block, further down:
    info must be the oracle's 1-based failing row (reading A10)."""
    N = 66                                                         # M = 201
    M = 3 * (N + 1)
    rng = np.random.default_rng(row)
    G = rng.standard_normal((M, M)) / np.sqrt(M)
    A = G @ G.T + 0.5 * np.eye(M)
    A[row, row] = -1.0                                             # leading minor of order row + 1 is not positive definite
    bd = _bd(N, 1)
    buf = np.zeros((1, M, bd.ld)); buf[0, :, :M] = A
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    bd.cholesky(_dev(buf), info)
    want = O.cholesky(A)[1]
    assert want == row + 1 and int(_host(info)[0]) == want


def test_cholesky_reports_non_positive_pivot():
    """reading A10: bead 2 sits on bead 0 -> D singular at row 7 (exact zero pivot); other chains unaffected."""
    N = 20
    r = W.random_chains(3, N, seed=9)
    r[1, 2] = r[1, 0]
    bd = _bd(N, 3)
    DL = bd.assemble_hi(_dev(r))
    info = torch.zeros(3, dtype=torch.int32, device="cuda")
    bd.cholesky(DL, info)
    ih = _host(info)
    p = O.Params(n_rods=N, dt=1e-4)
    want = O.cholesky(O.assemble(p, r[1]))[1]
    assert want > 0 and ih[1] == want and ih[0] == 0 and ih[2] == 0
    bd.cholesky(bd.assemble_hi(_dev(r)))                         # info_dev = NULL -> context array
    assert bd.last_info() == (1, 1)


# ------------------------------------------------------------------------------------------ a5
@pytest.mark.parametrize("N,C", SIZES + [(345, 1), (400, 2)])     # M = 1038, 1203: the shared-memory-staged kernel
def test_brownian_matches_oracle(N, C):
    r = W.random_chains(C, N, seed=300 + N)
    dt = 1e-4
    bd = _bd(N, C, dt, seed=42, chain_id0=3)
    M = bd.M
    p = O.Params(n_rods=N, dt=dt, seed=42)
    Ls = np.zeros((C, M, bd.ld))
    ys, dWs = [], []
    for c in range(C):
        Lo, info = O.cholesky(O.assemble(p, r[c]))
        Ls[c, :, :M] = Lo + np.triu(np.full((M, M), 1e300), 1)   # poison: strict upper must never be read
        dW = O.noise_dW(p, 3 + c, 17)
        dWs.append(dW); ys.append(O.trmv_lower(Lo, dW))
    Lg = _dev(Ls)
    y_internal = _host(bd.brownian(Lg, step=17))                 # in-kernel Philox
    y_given = _host(bd.brownian(Lg, step=0, dW=_dev(np.stack(dWs))))
    for c in range(C):
        scale = np.abs(ys[c]).max()
        assert np.abs(y_internal[c] - ys[c]).max() <= 1e-12 * scale
        assert np.abs(y_given[c] - ys[c]).max() <= 1e-13 * scale


# ------------------------------------------------------------------------------------------ a6-a8
@pytest.mark.parametrize("N,C", SIZES)
def test_update_matches_oracle(N, C):
    r = W.random_chains(C, N, seed=400 + N, rod_jitter=0.01)
    dt = 1e-4
    rng = np.random.default_rng(N)
    v = rng.standard_normal((C, 3 * (N + 1))) * 50.0
    y = rng.standard_normal((C, 3 * (N + 1))) * math.sqrt(2 * dt)
    bd = _bd(N, C, dt, kappa=KAPPA)
    p = O.Params(n_rods=N, dt=dt, kappa=KAPPA)
    rg = _host(bd.update(_dev(r), _dev(v), _dev(y)))
    for c in range(C):
        ro, u, Y, info = O.finish_step(p, r[c], O.spring_tensions(p, r[c]), v[c], y[c])
        assert info == 0
        assert np.abs(rg[c] - ro).max() <= 1e-12 * np.abs(ro).max()
    rin = _dev(r)
    bd.update(rin, _dev(v), _dev(y), r_out=rin)                  # in place
    assert np.array_equal(_host(rin), rg)


# ------------------------------------------------------------------------------------------ whole step
def _step_parity(N, C, dt, hstar, kappa, steps, noise_kind=0, seed=0, jitter=0.007, rseed=0, path=0):
    r0 = W.random_chains(C, N, seed=rseed, rod_jitter=jitter)
    bd = _bd(N, C, dt, hstar=hstar, kappa=kappa, seed=seed, noise_kind=noise_kind)
    bd.set_path(path)
    p = O.Params(n_rods=N, dt=dt, hstar=hstar, kappa=kappa if kappa is not None else np.zeros((3, 3)), seed=seed,
                 noise_kind=noise_kind)
    r = r0.copy()
    worst_pos, worst_dr = 0.0, 0.0
    for s in range(steps):
        rg = _host(bd.step(_dev(r), first_step=s, n_steps=1))
        ro, info = O.step_ensemble(p, r, s, 1)
        assert not info.any() and bd.last_info() == (0, -1)
        for c in range(C):
            worst_pos = max(worst_pos, np.abs(rg[c] - ro[c]).max() / np.abs(ro[c]).max())
            worst_dr = max(worst_dr, np.abs((rg[c] - r[c]) - (ro[c] - r[c])).max() / np.abs(ro[c] - r[c]).max())
        r = ro                                                   # re-synchronise each checked step (A16)
    return worst_pos, worst_dr


PATHS = [(1, "staged"), (2, "fused")]       # bd_set_path: staged kernels / fused per-chain kernel (M <= 320)
FUSED_SIZES = [(1, 1), (2, 3), (7, 2), (8, 2), (15, 3), (20, 2), (21, 1), (42, 3), (100, 5), (105, 300)]


@pytest.mark.parametrize("N,C", SIZES)
def test_one_step_positions_match_oracle_staged(N, C):
    pos, dr = _step_parity(N, C, 1e-4, 0.25, KAPPA * 0.05, steps=2, rseed=N, path=1)
    assert pos <= 1e-10                                          # BASELINE.json gate
    assert dr <= 1e-9                                            # the stricter displacement-relative figure (A16)


@pytest.mark.parametrize("N,C", FUSED_SIZES)
def test_one_step_positions_match_oracle_fused(N, C):
    """the fused per-chain kernel: ragged last panels (M % 24 != 0), one panel only (M <= 24), more chains
    than resident CTAs (C = 300 > 2 x 148)."""
    pos, dr = _step_parity(N, C, 1e-4, 0.25, KAPPA * 0.05, steps=2 if C < 100 else 1, rseed=N, path=2)
    assert pos <= 1e-10
    assert dr <= 1e-9


@pytest.mark.parametrize("path,name", PATHS)
def test_step_variants_uniform_noise_free_draining_shear(path, name):
    assert _step_parity(30, 3, 1e-3, 0.5, None, steps=2, noise_kind=1, seed=77, path=path)[0] <= 1e-10   # paper's law, h* = a* = 0.5
    assert _step_parity(30, 3, 1e-4, 0.0, W.CONFIGS["c3"].kappa() * 100, steps=2, path=path)[0] <= 1e-10  # h* = 0, shear
    assert _step_parity(64, 2, 5e-5, 0.25, W.CONFIGS["c2"].kappa(), steps=2, path=path)[0] <= 1e-10


def test_fused_and_staged_paths_agree():
    N, C = 100, 16
    r0 = W.random_chains(C, N, seed=31, rod_jitter=0.007)
    outs = []
    for path in (1, 2):
        bd = _bd(N, C, 1e-4, kappa=W.CONFIGS["c2"].kappa(), seed=5)
        bd.set_path(path)
        outs.append(_host(bd.step(_dev(r0), 0, 3)))
    assert np.abs(outs[0] - outs[1]).max() / np.abs(outs[0]).max() <= 1e-11


@pytest.mark.parametrize("path,name", PATHS)
def test_negligible_hstar_follows_the_free_draining_run(path, name):
    """PAPER.md:262 / Fig. 6 (:419): with h* = 1e-5 the run with HI must agree with the run without HI (same start,
    same noise).  D = I + O(h*), so L = I + O(h*): after 200 steps of the paper's variant (uniform noise, dt = 1e-3,
    K* = 1e3, extension) the two differ by O(h* x displacement), and each tracks the oracle at its own h*."""
    N, C, dt, steps = 100, 4, 1e-3, 200
    kappa = np.diag([0.01, -0.005, -0.005])
    r0 = W.random_chains(C, N, seed=61, rod_jitter=0.0)
    out = {}
    for h in (1e-5, 0.0):
        bd = _bd(N, C, dt, hstar=h, kappa=kappa, seed=3, noise_kind=1)
        bd.set_path(path)
        out[h] = _host(bd.step(_dev(r0), 0, steps))
        assert bd.last_info() == (0, -1)
        assert _step_parity(N, 2, dt, h, kappa, steps=1, noise_kind=1, seed=3, jitter=0.0, rseed=61, path=path)[0] <= 1e-10
    moved = np.abs(out[0.0] - r0).max()
    diff = np.abs(out[1e-5] - out[0.0]).max()
    assert moved > 0.5                                           # the chains did move (200 steps of sqrt(2 dt) kicks)
    assert 0.0 < diff <= 1e-3 * moved                            # HI is ON (diff > 0) but negligible


def test_fused_path_rejected_for_long_chains():
    from paper_2208_06559_b200.binding import BDError
    bd = _bd(200, 1)
    with pytest.raises(BDError):
        bd.set_path(2)


@pytest.mark.parametrize("path,name", PATHS)
def test_multi_step_call_equals_repeated_single_steps_and_tracks_oracle(path, name):
    N, C, dt = 40, 4, 1e-4
    r0 = W.random_chains(C, N, seed=2)
    bd = _bd(N, C, dt, seed=11)
    bd.set_path(path)
    a = _host(bd.step(_dev(r0), first_step=0, n_steps=6))
    rb = _dev(r0)
    for s in range(6):
        bd.step(rb, first_step=s, n_steps=1)
    assert np.array_equal(a, _host(rb))                          # deterministic, counter-based noise
    ro, info = O.step_ensemble(O.Params(n_rods=N, dt=dt, seed=11), r0, 0, 6)
    assert np.abs(a - ro).max() / np.abs(ro).max() <= 1e-9       # free-running 6 steps: reported, loose


@pytest.mark.parametrize("path,name", PATHS)
def test_failed_chain_keeps_its_state(path, name):
    N = 20
    r = W.random_chains(3, N, seed=9)
    r[1, 2] = r[1, 0]
    bd = _bd(N, 3)
    bd.set_path(path)
    rg = _host(bd.step(_dev(r), 0, 1))
    assert np.array_equal(rg[1], r[1])                           # A10: reported, unchanged
    assert bd.last_info() == (1, 1)
    assert not np.array_equal(rg[0], r[0])


# ------------------------------------------------------------------------------------------ a9
@pytest.mark.parametrize("N,C", [(1, 1), (20, 7), (100, 40), (300, 3)])
def test_observables_match_oracle(N, C):
    r = W.random_chains(C, N, seed=500 + N, rod_jitter=0.02)
    bd = _bd(N, C, 1e-4)
    per, ens = [_host(x) for x in bd.observables(_dev(r))]
    po, eo = O.observables(O.Params(n_rods=N, dt=1e-4), r)
    assert np.allclose(per, po, rtol=1e-11, atol=1e-9)
    assert np.allclose(ens, eo, rtol=1e-11, atol=1e-9)


def test_step_host_roundtrip_equals_device_path():
    N, C = 20, 8
    r0 = W.random_chains(C, N, seed=4)
    bd = _bd(N, C, seed=3)
    dev = _host(bd.step(_dev(r0), 0, 3))
    rh = torch.from_numpy(r0.copy()).pin_memory()
    ens = torch.zeros(2, 13, dtype=torch.float64).pin_memory()
    bd.step_host(rh, 0, 3, ens)
    assert np.array_equal(rh.numpy(), dev)
    assert np.allclose(ens.numpy(), O.observables(O.Params(n_rods=N, dt=1e-4), dev)[1], rtol=1e-11, atol=1e-9)


def test_bad_arguments_are_rejected_without_launching():
    from paper_2208_06559_b200.binding import BD, BDError
    with pytest.raises(BDError):
        BD(n_rods=0, n_chains=1, dt=1e-4)
    with pytest.raises(BDError):
        BD(n_rods=5, n_chains=1, dt=1e-4, hstar=0.5, a=0.25)      # h*/a > 1 (reading A3)
    bd = _bd(5, 1)
    n0 = bd.launch_count()
    with pytest.raises(BDError) as e:
        bd.assemble_hi(torch.zeros(1, 6, 3, dtype=torch.float64, device="cuda"),
                       torch.zeros(1, 18, 17, dtype=torch.float64, device="cuda"))      # ld odd and < M
    assert e.value.code == -4 and bd.launch_count() == n0


# ------------------------------------------------------------------------------------------ f1: relaxation-time observable
@pytest.mark.parametrize("N,C", [(1, 3), (20, 300), (100, 1000)])
def test_end_to_end_and_autocorrelation_match_oracle(N, C):
    """bd_end_to_end / bd_autocorr against orc_end_to_end / orc_autocorr on moved chains."""
    r0 = W.random_chains(C, N, seed=900 + N, rod_jitter=0.01)
    r1 = W.random_chains(C, N, seed=901 + N, rod_jitter=0.01) * 0.3 + r0           # correlated with r0, not equal
    bd = _bd(N, C)
    R0 = bd.end_to_end(_dev(r0))
    assert np.array_equal(_host(R0), O.end_to_end(N, r0))
    out = _host(bd.autocorr(_dev(r1), R0))
    want = O.autocorr(N, r1, O.end_to_end(N, r0))
    assert np.allclose(out, want, rtol=1e-12, atol=0)
    assert np.allclose(_host(bd.autocorr(_dev(r0), R0)), O.autocorr(N, r0, O.end_to_end(N, r0)), rtol=1e-12)


def test_relaxation_time_pipeline_free_draining():
    """relaxation.measure on the GPU path (bd_step + bd_autocorr): without HI a 10-rod chain relaxes on the Rouse
    scale (the paper's Fig. 8 check); round 1 measured lambda = 1.27 lambda_Rouse for bead-rod chains."""
    from paper_2208_06559_b200 import relaxation
    row = relaxation.measure(10, 2048, 0.0, 1e-3, 2.0, 50)
    assert 0.9 < row["lambda"] / row["lambda_rouse"] < 1.7
    assert abs(row["Ree"] ** 2 / 10.0 - 1.0) < 0.1                                # <R^2> = N b^2 at equilibrium


def test_relaxation_run_resumed_from_a_checkpoint_is_the_uninterrupted_run(tmp_path):
    """relaxation.measure with a time budget of zero stops after one sample and writes its state; resumed, it returns
    exactly the row of the uninterrupted run (counter-based noise, deterministic kernels)."""
    from paper_2208_06559_b200 import relaxation
    full = relaxation.measure(10, 256, 0.25, 1e-3, 1.0, 20)
    ck = str(tmp_path / "ck.npz")
    assert relaxation.measure(10, 256, 0.25, 1e-3, 1.0, 20, save=ck, budget_s=0.0) is None
    cont = relaxation.measure(10, 256, 0.25, 1e-3, 1.0, 20, resume=ck)
    assert cont == full
