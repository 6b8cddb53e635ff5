"""Pins for the CPU oracle (``-m "not gpu"``): the oracle is checked against what the paper and the
mathematics fix -- hand-computed values (tests/golden/), closed forms, invariants, special cases that
reduce to a LAPACK/numpy routine, and the paper's own formula written the paper's way (difference
tensors, Eq. 14/21) -- never against itself.  Pin numbers P1..P11 refer to DESIGN.md.
"""
import math
import os

import numpy as np
import pytest
from scipy import stats

import oracle as O
from paper_2208_06559_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _params(N, dt=1e-4, **kw):
    return O.Params(n_rods=N, dt=dt, **kw)


# ------------------------------------------------------------------------------------------ P5
def test_philox_known_answers():
    """Random123 KAT vectors (tests/golden/philox4x32_10_kat.txt)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if not l.startswith("#")]
    assert len(rows) == 3
    for row in rows:
        w = [int(x, 16) for x in row]
        assert O.philox4x32_10(w[0:4], w[4:6]) == w[6:10]


def test_u01_exact_open_interval():
    assert O.u01(0) == 2.0 ** -53
    assert O.u01(2 ** 64 - 1) == 1.0 - 2.0 ** -53
    assert O.u01(1 << 12) == 3.0 * 2.0 ** -53
    assert O.u01((1 << 12) - 1) == 2.0 ** -53          # low 12 bits are discarded
    assert O.u01(1 << 63) == 0.5 + 2.0 ** -53


def test_normals_follow_counter_layout_and_box_muller():
    """g_{2p}, g_{2p+1} recomputed in the test from the KAT-pinned block function and the stated
    counter layout (p, chain, step_lo, step_hi28 | purpose<<28), key = (seed_lo, seed_hi)."""
    seed, chain, step = 0x1234567_89ABCDEF, 77, (5 << 32) | 9
    g = O.normals(seed, chain, step, 7)
    for p in range(4):
        w = O.philox4x32_10([p, chain, step & 0xFFFFFFFF, (step >> 32) & 0x0FFFFFFF],
                            [seed & 0xFFFFFFFF, seed >> 32])
        x1, x2 = (w[1] << 32) | w[0], (w[3] << 32) | w[2]
        u1 = (2 * (x1 >> 12) + 1) / 2.0 ** 53
        u2 = (2 * (x2 >> 12) + 1) / 2.0 ** 53
        rho, th = math.sqrt(-2.0 * math.log(u1)), 6.283185307179586 * u2
        assert g[2 * p] == pytest.approx(rho * math.cos(th), rel=1e-14, abs=1e-15)
        if 2 * p + 1 < 7:
            assert g[2 * p + 1] == pytest.approx(rho * math.sin(th), rel=1e-14, abs=1e-15)
    # streams differ by chain, step and seed; a prefix of a longer draw is the shorter draw
    assert not np.array_equal(O.normals(seed, chain + 1, step, 7), g)
    assert not np.array_equal(O.normals(seed, chain, step + 1, 7), g)
    assert not np.array_equal(O.normals(seed, chain, step + (1 << 32), 7), g)
    assert not np.array_equal(O.normals(seed + 1, chain, step, 7), g)
    assert np.array_equal(O.normals(seed, chain, step, 63)[:7], g)


def test_normals_distribution():
    g = O.normals(0, 3, 11, 2_000_000)
    n = g.size
    assert abs(g.mean()) < 4.0 / math.sqrt(n)
    assert abs(g.var() - 1.0) < 4.0 * math.sqrt(2.0 / n)
    assert abs((g ** 4).mean() - 3.0) < 4.0 * math.sqrt(96.0 / n)
    assert abs((g[0::2] * g[1::2]).mean()) < 4.0 / math.sqrt(n / 2)      # cos/sin partners uncorrelated
    assert stats.kstest(g[:200_000], "norm").pvalue > 1e-3


def test_uniform_noise_law_eq2():
    """Eq. 2: n uniform in [-1,1]; dW = sqrt(6 dt) n has variance 2 dt."""
    n = O.uniforms_pm1(5, 1, 2, 1_000_001)
    assert n.min() > -1.0 and n.max() < 1.0
    assert abs(n.mean()) < 4.0 / math.sqrt(3 * n.size)
    assert stats.kstest(n[:200_000], "uniform", args=(-1.0, 2.0)).pvalue > 1e-3
    p = _params(200_000, dt=1e-3, noise_kind=1)
    dW = O.noise_dW(p, 0, 0)
    assert abs(dW.var() / (2 * 1e-3) - 1.0) < 0.01
    pg = _params(200_000, dt=1e-3, noise_kind=0)
    dWg = O.noise_dW(pg, 0, 0)
    assert abs(dWg.var() / (2 * 1e-3) - 1.0) < 0.01
    assert np.allclose(dWg, math.sqrt(2e-3) * O.normals(0, 0, 0, pg.M), rtol=1e-15)


# ------------------------------------------------------------------------------------------ P1
def test_rpy_hand_values():
    for line in open(os.path.join(GOLD, "rpy_spot_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        h, a, R, dpar, dperp = [float(x) for x in line.split()]
        p = _params(1, hstar=h, a=a)
        B = O.rpy_block(p, [R, 0, 0], [0, 0, 0])
        assert np.allclose(B, np.diag([dpar, dperp, dperp]), rtol=1e-15, atol=1e-16)
        # rotated separation: block = dperp I + (dpar - dperp) n n^T
        n = np.array([1.0, 2.0, -2.0]) / 3.0
        Bn = O.rpy_block(p, R * n + 0.3, np.full(3, 0.3))
        assert np.allclose(Bn, dperp * np.eye(3) + (dpar - dperp) * np.outer(n, n), rtol=1e-13, atol=1e-15)


def test_rpy_continuity_trace_symmetry_limits():
    p = _params(1, hstar=0.25, a=0.25)
    n = np.array([2.0, -1.0, 2.0]) / 3.0
    lo = O.rpy_block(p, (0.5 - 1e-12) * n, np.zeros(3))
    hi = O.rpy_block(p, (0.5 + 1e-12) * n, np.zeros(3))
    assert np.allclose(lo, hi, atol=1e-11)                      # Eq. 8 = Eq. 9 at R = 2a
    for R in (0.5, 0.7, 1.0, 3.3, 40.0):                        # far branch: trace = (3h/4R) * 4 exactly
        B = O.rpy_block(p, R * n, np.zeros(3))
        assert np.trace(B) == pytest.approx(3 * 0.25 / (4 * R) * 4.0, rel=1e-14)
        assert np.allclose(B, B.T, rtol=1e-15, atol=1e-18)
        assert np.allclose(B, O.rpy_block(p, np.zeros(3), R * n), rtol=1e-15)    # D_ij = D_ji
    assert np.allclose(O.rpy_block(p, 1e-9 * n, np.zeros(3)), np.eye(3), atol=1e-8)   # R -> 0: (h/a) I
    assert np.array_equal(O.rpy_block(p, np.zeros(3), np.zeros(3)), np.eye(3))
    # b != 1: lengths scale with b
    p2 = _params(1, hstar=0.25, a=0.5, b=2.0)
    assert np.allclose(O.rpy_block(p2, 2.0 * 0.8 * n, np.zeros(3)), O.rpy_block(p, 0.8 * n, np.zeros(3)), rtol=1e-14)


def test_assemble_layout_and_free_draining():
    r = W.random_chains(1, 7, seed=3)[0]
    p = _params(7, hstar=0.25)
    D = O.assemble(p, r)
    assert D.shape == (24, 24)
    for i in range(8):
        for j in range(8):
            blk = D[3 * i:3 * i + 3, 3 * j:3 * j + 3]            # Eqs. 18-19: row 3i+k, col 3j+l
            if i == j:
                assert np.array_equal(blk, np.eye(3))            # Eq. 7
            else:
                assert np.array_equal(blk, O.rpy_block(p, r[i], r[j]))
    assert np.allclose(D, D.T, rtol=1e-15, atol=1e-17)
    assert np.array_equal(O.assemble(_params(7, hstar=0.0), r), np.eye(24))     # h* = 0 -> D = I


# ------------------------------------------------------------------------------------------ P2
def test_two_bead_eigenvalues_closed_form():
    """D = [[I,B],[B,I]], B = alpha I + beta nn^T -> eigenvalues 1 +- (alpha+beta), 1 +- alpha (x2)."""
    h = a = 0.25
    for R in (0.3, 0.5, 1.0, 2.5):
        n = np.array([0.6, 0.0, 0.8])
        r = np.array([np.zeros(3), R * n])
        D = O.assemble(_params(1, hstar=h, a=a), r)
        if R >= 2 * a:
            alpha = 3 * h / (4 * R) * (1 + 2 * a * a / (3 * R * R))
            beta = 3 * h / (4 * R) * (1 - 2 * a * a / (R * R))
        else:
            alpha = 3 * h / (8 * a) * (8 / 3 - 3 * R / (4 * a))
            beta = 3 * h / (8 * a) * R / (4 * a)
        want = sorted([1 + alpha + beta, 1 - alpha - beta] + [1 + alpha] * 2 + [1 - alpha] * 2)
        assert np.allclose(np.linalg.eigvalsh(D), want, rtol=1e-13)
        assert min(want) > 0


def test_positive_definite_on_workload_chains():
    for N, seed in ((20, 1), (100, 2), (300, 3)):
        r = W.random_chains(2, N, seed=seed, rod_jitter=0.007)
        for c in range(2):
            D = O.assemble(_params(N), r[c])
            assert np.linalg.eigvalsh(D)[0] > 0
            L, info = O.cholesky(D)
            assert info == 0 and np.all(np.diag(L) > 0)


def test_hstar_over_a_above_one_is_not_pd():
    """reading A3: h*/a = 2 is not guaranteed PD -- the oracle must REPORT it (A10), not hide it."""
    r = W.random_chains(1, 100, seed=5)[0]
    D = O.assemble(_params(100, hstar=0.5, a=0.25), r)
    assert np.linalg.eigvalsh(D)[0] < 0
    L, info = O.cholesky(D)
    assert info > 0
    # the reported row is the first non-positive pivot: leading (info-1) block is PD, leading info block is not
    assert np.linalg.eigvalsh(D[:info - 1, :info - 1])[0] > 0
    assert np.linalg.eigvalsh(D[:info, :info])[0] <= 1e-12


# ------------------------------------------------------------------------------------------ P3
def test_cholesky_residual_and_lapack():
    rng = np.random.default_rng(0)
    for M in (1, 2, 5, 63, 200):
        A = rng.standard_normal((M, M))
        A = A @ A.T + M * np.eye(M)
        L, info = O.cholesky(A)
        assert info == 0
        assert np.array_equal(np.triu(L, 1), np.zeros((M, M)))
        assert np.linalg.norm(L @ L.T - A) / np.linalg.norm(A) < 1e-14
        assert np.allclose(L, np.linalg.cholesky(A), rtol=1e-12, atol=1e-13)
    r = W.random_chains(1, 100, seed=11)[0]
    D = O.assemble(_params(100), r)
    L, info = O.cholesky(D)
    assert info == 0
    assert np.linalg.norm(L @ L.T - D) / np.linalg.norm(D) < 1e-12           # BASELINE.json gate
    assert np.allclose(L, np.linalg.cholesky(D), rtol=0, atol=1e-13)


def test_cholesky_reads_lower_triangle_only():
    rng = np.random.default_rng(1)
    A = rng.standard_normal((9, 9)); A = A @ A.T + 9 * np.eye(9)
    Aj = np.tril(A) + np.triu(rng.standard_normal((9, 9)), 1)      # garbage in the strict upper
    assert np.array_equal(O.cholesky(Aj)[0], O.cholesky(A)[0])


def test_cholesky_two_bead_closed_form():
    """L = [[I,0],[B, chol(I - B^2)]] for D = [[I,B],[B,I]]."""
    r = np.array([[0.0, 0.0, 0.0], [0.3, 0.4, 1.2]])
    D = O.assemble(_params(1, hstar=0.25), r)
    B = D[3:, :3]
    L, info = O.cholesky(D)
    assert info == 0
    assert np.allclose(L[:3, :3], np.eye(3)) and np.allclose(L[3:, :3], B, rtol=1e-15)
    assert np.allclose(L[3:, 3:], np.linalg.cholesky(np.eye(3) - B @ B), rtol=1e-13, atol=1e-15)


def test_cholesky_brute_force_left_looking_column_algorithm():
    """independent second algorithm (column Cholesky-Crout, written here) on M <= 63."""
    r = W.random_chains(1, 20, seed=4, rod_jitter=0.007)[0]
    D = O.assemble(_params(20), r)
    M = 63
    Lc = np.zeros((M, M))
    for j in range(M):
        col = D[j:, j] - Lc[j:, :j] @ Lc[j, :j]
        Lc[j, j] = math.sqrt(col[0])
        Lc[j + 1:, j] = col[1:] / Lc[j, j]
    L, info = O.cholesky(D)
    assert info == 0 and np.allclose(L, Lc, rtol=1e-13, atol=1e-15)


def test_cholesky_reports_failing_pivot():
    A = np.eye(5); A[3, 3] = -1.0
    assert O.cholesky(A)[1] == 4
    A = np.eye(5); A[2, 2] = float("nan")
    assert O.cholesky(A)[1] == 3
    A = np.array([[1.0, 1.0], [1.0, 1.0]])            # singular: pivot exactly 0
    assert O.cholesky(A)[1] == 2


# ------------------------------------------------------------------------------------------ P4
def test_matvecs_against_numpy():
    rng = np.random.default_rng(2)
    M = 57
    A = rng.standard_normal((M, M)); x = rng.standard_normal(M)
    assert np.allclose(O.symv(A, x), A @ x, rtol=1e-13, atol=1e-13)
    assert np.allclose(O.trmv_lower(A, x), np.tril(A) @ x, rtol=1e-13, atol=1e-13)   # ignores strict upper
    L = np.tril(A)
    for j in (0, 5, M - 1):
        e = np.zeros(M); e[j] = 1.0
        assert np.array_equal(O.trmv_lower(L, e), L[:, j])


def test_drift_onthefly_equals_stored_symv():
    r = W.random_chains(1, 40, seed=8, rod_jitter=0.01)[0]
    p = _params(40)
    F = O.bead_forces(40, O.spring_tensions(p, r))
    assert np.array_equal(O.drift_onthefly(p, r, F), O.symv(O.assemble(p, r), F.reshape(-1)))


def test_cov_L_dW_is_2_D_dt():
    """BASELINE.json pin: cov(L dW) -> 2 D dt (Eq. 10 + Ermak-McCammon), over 2e5 draws, N = 3."""
    N, dt = 3, 1e-3
    p = _params(N, dt=dt)
    r = np.array([[0, 0, 0], [0.9, 0.1, 0.0], [1.2, 0.9, 0.3], [1.0, 0.5, 0.35]], dtype=float)   # one overlap pair
    D = O.assemble(p, r)
    L, info = O.cholesky(D)
    assert info == 0
    n = 200_000
    dW = np.stack([O.noise_dW(p, 0, s) for s in range(n // 100)] +
                  [O.noise_dW(p, c, 0) for c in range(1, n - n // 100 + 1)])
    y = dW @ L.T                                      # y_s = L dW_s (numpy route for the matvec)
    assert np.allclose(y[7], O.trmv_lower(L, dW[7]), rtol=1e-13, atol=1e-18)
    cov = y.T @ y / n
    target = 2 * dt * D
    se = np.sqrt((np.outer(np.diag(target), np.diag(target)) + target ** 2) / n)
    assert np.all(np.abs(cov - target) < 4.5 * se)
    assert abs(y.mean()) < 1e-4


# ------------------------------------------------------------------------------------------ forces
def test_spring_and_bead_forces_closed_form():
    p = _params(2, dt=1e-4, K=1e4)
    r = np.array([[0, 0, 0], [1.1, 0, 0], [1.1, 0.9, 0]], dtype=float)
    T = O.spring_tensions(p, r)
    assert np.allclose(T, [[1e4 * 0.1, 0, 0], [0, 1e4 * (-0.1), 0]], rtol=1e-12)     # Eq. 3
    F = O.bead_forces(2, T)
    assert np.allclose(F, [T[0], T[1] - T[0], -T[1]])                                 # Eq. 1 / Eq. 22
    assert np.allclose(F.sum(0), 0, atol=1e-9)
    pb = _params(1, K=50.0, b=2.0)
    assert np.allclose(O.spring_tensions(pb, [[0, 0, 0], [0, 0, 3.0]]), [[0, 0, 50.0 * (3 - 2) / 3 * 3]])


# ------------------------------------------------------------------------------------------ P6
def test_semi_implicit_identity_eq15():
    """Q'[1 + 2 dt K (|Q'|-b)/|Q'|] = Y (Eq. 15) for the Q' the oracle returns from its own Y."""
    N = 30
    p = _params(N, dt=1e-4, kappa=W.CONFIGS["c3"].kappa() * 50)
    r = W.random_chains(1, N, seed=9, rod_jitter=0.02)[0]
    rn, info, tr = O.step(p, 0, 3, r, trace=True)
    assert info == 0
    Qn = np.diff(rn, axis=0)
    qn = np.linalg.norm(Qn, axis=1, keepdims=True)
    K, dt = 1e4, 1e-4
    assert np.allclose(Qn * (1 + 2 * dt * K * (qn - 1) / qn), tr["Y"], rtol=1e-13, atol=1e-15)
    assert np.allclose(rn.mean(0), 0, atol=1e-13)                      # A8: centre of mass pinned


def test_semi_implicit_unit_Y_gives_unit_rod():
    p = _params(1, dt=1e-4)
    r = np.array([[0, 0, 0], [0.6, 0.0, 0.8]])
    T = O.spring_tensions(p, r)
    assert np.allclose(T, 0)
    rn, u, Y, info = O.finish_step(p, r, T, np.zeros(6), np.zeros(6))
    assert info == 0 and np.allclose(np.linalg.norm(rn[1] - rn[0]), 1.0, rtol=1e-15)


def test_single_rod_geometric_relaxation():
    """N = 1, no HI, no noise, no flow: Y = Q exactly (the -2T explicit part cancels +2T, A7) and
    |Q_n| - b = (|Q_0| - b)/(1 + 2 dt K)^n  (from Eqs. 14, 17)."""
    dt, K = 1e-3, 300.0
    p = _params(1, dt=dt, K=K, hstar=0.0)
    r = np.array([[0, 0, 0], [0.0, 1.3, 0.0]])
    for n in range(1, 6):
        T = O.spring_tensions(p, r)
        F = O.bead_forces(1, T)
        v = O.symv(O.assemble(p, r), F.reshape(-1))
        r, u, Y, info = O.finish_step(p, r, T, v, np.zeros(6))
        assert info == 0
        assert np.linalg.norm(r[1] - r[0]) - 1.0 == pytest.approx(0.3 / (1 + 2 * dt * K) ** n, rel=1e-12)


def test_single_rod_shear_closed_form():
    """no noise, rod at rest length: Y = (I + dt kappa) Q."""
    dt = 1e-3
    kap = np.zeros((3, 3)); kap[0, 1] = 2.5
    p = _params(1, dt=dt, K=1e3, hstar=0.0, kappa=kap)
    Q = np.array([0.0, 1.0, 0.0])
    r = np.array([-Q / 2, Q / 2])
    T = O.spring_tensions(p, r)
    rn, u, Y, info = O.finish_step(p, r, T, np.zeros(6), np.zeros(6))
    assert np.allclose(Y[0], (np.eye(3) + dt * kap) @ Q, rtol=1e-15)
    assert np.allclose(u.reshape(2, 3), dt * (r @ kap.T), rtol=1e-15, atol=1e-18)
    Yn = np.linalg.norm(Y[0])
    assert np.allclose(rn[1] - rn[0], Y[0] * ((2 * dt * 1e3 + Yn) / (2 * dt * 1e3 + 1)) / Yn, rtol=1e-14)


def test_eq14_written_with_difference_tensors():
    """The paper's own form (Eqs. 14, 21, 23-24): difference tensors
    Diff = D_{k+1,.} - D_{k,.} and sigma-Diff, multiplied by F and sqrt(6/dt) n ... here with the
    Gaussian dW.  Reading A7 says the oracle's bead-space form is the same number."""
    N = 12
    kap = W.Workload("x", 1, N, 1e-4, "extension", 10.0, 1).kappa() * 200
    p = _params(N, dt=1e-4, kappa=kap)
    r = W.random_chains(1, N, seed=21, rod_jitter=0.02)[0]
    rn, info, tr = O.step(p, 4, 17, r, trace=True)
    assert info == 0
    D = O.assemble(p, r)
    sig = np.linalg.cholesky(D)                       # LAPACK, not the oracle's
    Fs = tr["F"].reshape(-1)
    dW = O.noise_dW(p, 4, 17)
    Q = np.diff(r, axis=0)
    for k in range(N):
        Diff = D[3 * (k + 1):3 * (k + 1) + 3, :] - D[3 * k:3 * k + 3, :]
        sDiff = sig[3 * (k + 1):3 * (k + 1) + 3, :] - sig[3 * k:3 * k + 3, :]
        Yk = Q[k] + 1e-4 * (kap @ Q[k] + Diff @ Fs + 2 * tr["T"][k]) + sDiff @ dW
        assert np.allclose(tr["Y"][k], Yk, rtol=1e-11, atol=1e-14)


# ------------------------------------------------------------------------------------------ P11
def _numpy_step(p, r, dW):
    """Independent vectorised restatement (numpy + LAPACK) for brute force on tiny N."""
    cp = p.c()
    N = p.n_rods
    Q = np.diff(r, axis=0)
    q = np.linalg.norm(Q, axis=1, keepdims=True)
    T = cp.K * (q - cp.b) / q * Q
    F = np.zeros((N + 1, 3)); F[:-1] += T; F[1:] -= T
    M = 3 * (N + 1)
    D = np.eye(M)
    for i in range(N + 1):
        for j in range(N + 1):
            if i == j:
                continue
            Rv = (r[i] - r[j]) / cp.b; R = np.linalg.norm(Rv); a = cp.a / cp.b; n = Rv / R
            if R >= 2 * a:
                blk = 3 * cp.hstar / (4 * R) * ((1 + 2 * a * a / (3 * R * R)) * np.eye(3) + (1 - 2 * a * a / (R * R)) * np.outer(n, n))
            else:
                blk = 3 * cp.hstar / (4 * R) * (R / (2 * a)) * ((8 / 3 - 3 * R / (4 * a)) * np.eye(3) + R / (4 * a) * np.outer(n, n))
            D[3 * i:3 * i + 3, 3 * j:3 * j + 3] = blk
    L = np.linalg.cholesky(D)
    kap = np.array(list(cp.kappa)).reshape(3, 3)
    u = cp.dt * (r @ kap.T + (D @ F.reshape(-1)).reshape(-1, 3)) + (L @ dW).reshape(-1, 3)
    Y = Q + np.diff(u, axis=0) + 2 * cp.dt * T
    Yn = np.linalg.norm(Y, axis=1, keepdims=True)
    Qn = Y * ((2 * cp.dt * cp.K * cp.b + Yn) / (2 * cp.dt * cp.K + 1)) / Yn
    rn = np.zeros_like(r); rn[1:] = np.cumsum(Qn, axis=0)
    return rn - rn.mean(0)


@pytest.mark.parametrize("N", [1, 2, 3, 9])
def test_brute_force_tiny_chains(N):
    kap = np.array([[0.3, 1.0, 0.0], [0.0, -0.1, 0.2], [0.5, 0.0, -0.2]])
    for nk in (0, 1):
        p = _params(N, dt=2e-4, hstar=0.3, a=0.35, b=1.0, K=4000.0, kappa=kap, seed=99, noise_kind=nk)
        r = W.random_chains(1, N, seed=N, rod_jitter=0.03)[0]
        rn, info = O.step(p, 6, 41, r)
        assert info == 0
        want = _numpy_step(p, r, O.noise_dW(p, 6, 41))
        assert np.allclose(rn, want, rtol=1e-12, atol=1e-13)


# ------------------------------------------------------------------------------------------ P7 / P8 / P10
def test_initial_walk_is_equilibrium_freely_jointed_chain():
    N, C = 50, 4096
    r = O.init_random_walk(N, 1.0, 1234, range(C))
    Q = np.diff(r, axis=1)
    assert np.allclose(np.linalg.norm(Q, axis=2), 1.0, rtol=1e-14)
    assert np.allclose(r.mean(axis=1), 0, atol=1e-12)
    R2 = ((r[:, -1] - r[:, 0]) ** 2).sum(1)
    assert abs(R2.mean() - N) < 3.5 * math.sqrt(2.0 / 3.0) * N / math.sqrt(C)      # <R^2> = N b^2
    assert np.all(np.abs(Q.mean(axis=(0, 1))) < 4 / math.sqrt(3 * N * C))           # isotropic
    assert np.all(np.abs((Q ** 2).mean(axis=(0, 1)) - 1 / 3) < 4 * math.sqrt(4 / 45) / math.sqrt(N * C))
    assert abs((Q[:, :-1] * Q[:, 1:]).sum(2).mean()) < 4 / math.sqrt(3 * (N - 1) * C)   # freely jointed
    r2 = O.init_random_walk(N, 2.5, 1234, [7])
    assert np.allclose(r2[0], 2.5 * r[7], rtol=1e-14)
    assert not np.allclose(O.init_random_walk(N, 1.0, 1235, [0])[0], r[0])


def test_rod_lengths_and_equilibrium_R2_with_and_without_HI():
    """P7: Fraenkel rods are stiff, not rigid: std(|Q|-b) ~ sqrt(dt/2), max < 0.1 b.
    P8: <R^2> = N b^2 within 3 SE, HI does not change the equilibrium distribution."""
    N, C, dt, steps = 20, 256, 1e-4, 150
    r0 = O.init_random_walk(N, 1.0, 77, range(C))
    for h in (0.0, 0.25):
        p = _params(N, dt=dt, hstar=h, seed=5)
        r, info = O.step_ensemble(p, r0, 0, steps)
        assert not info.any()
        q = np.linalg.norm(np.diff(r, axis=1), axis=2)
        assert np.abs(q - 1).max() < 0.1
        assert abs((q - 1).std() / math.sqrt(dt / 2) - 1.0) < 0.15
        per, ens = O.observables(p, r)
        mean = ens[0, 0] / C
        se = math.sqrt(max(ens[1, 0] / C - mean ** 2, 0) / C)
        assert abs(mean - N) < 3.5 * se + 0.02 * N
        assert per[:, 12].max() == pytest.approx(np.abs(q - 1).max(), rel=1e-12)


def test_low_hstar_tracks_free_draining():
    """the paper's own validation: h* = 1e-5 reproduces the no-HI run."""
    N = 30
    kap = W.Workload("x", 1, N + 0, 1e-4, "extension", 3.0, 1).kappa()
    r0 = O.init_random_walk(N, 1.0, 3, range(4))
    outs = []
    for h in (0.0, 1e-5):
        p = _params(N, dt=1e-4, hstar=h, a=0.25, kappa=kap, seed=8)
        r, info = O.step_ensemble(p, r0, 0, 50)
        assert not info.any()
        outs.append(r)
    diff = np.abs(outs[0] - outs[1]).max()
    assert 0 < diff < 1e-3            # O(h*) coupling, not zero, not large


# ------------------------------------------------------------------------------------------ observables
def test_observables_closed_forms():
    N = 10
    p = _params(N, dt=1e-4, K=1e4)
    r = np.zeros((1, N + 1, 3)); r[0, :, 0] = 1.1 * np.arange(N + 1)       # straight, stretched 10 %
    per, ens = O.observables(p, r)
    o = dict(zip(O.OBS_NAMES, per[0]))
    assert o["R2"] == pytest.approx((1.1 * N) ** 2) and o["Rx2"] == pytest.approx((1.1 * N) ** 2)
    assert o["Ry2"] == 0 and o["Rz2"] == 0
    assert o["Rg2"] == pytest.approx(1.1 ** 2 * ((N + 1) ** 2 - 1) / 12.0)    # equally spaced points
    assert o["Sxx"] == pytest.approx(N * 1e4 * 0.1 * 1.1, rel=1e-11)          # sum_k T_k Q_k (Eq. 28)
    assert o["Syy"] == 0 and o["Sxy"] == 0
    assert o["rod_dev_ms"] == pytest.approx(0.01, rel=1e-11) and o["rod_dev_max"] == pytest.approx(0.1, rel=1e-11)
    # ensemble sums
    r2 = np.concatenate([r, 2 * r])
    per2, ens2 = O.observables(p, r2)
    assert np.allclose(ens2[0], per2.sum(0)) and np.allclose(ens2[1], (per2 ** 2).sum(0))
    # off-diagonal stress: rod along (1,1,0)/sqrt2 stretched
    rr = np.zeros((1, 2, 3)); rr[0, 1] = np.array([1, 1, 0]) / math.sqrt(2) * 1.2
    o = dict(zip(O.OBS_NAMES, O.observables(_params(1, K=100.0), rr)[0][0]))
    assert o["Sxy"] == pytest.approx(100.0 * 0.2 * 1.2 * 0.5, rel=1e-12)
    assert o["Sxx"] == pytest.approx(o["Syy"]) and o["Sxz"] == 0


def test_observables_generic_position_every_component_distinct():
    """Eqs. 25-28 written out by hand for a 2-rod chain in GENERAL position, so that every one of the
    13 outputs is a distinct non-zero number (a y<->z swap, or a swapped pair of stress indices, fails here):
        r_0 = (0,0,0), Q_0 = (0.3, 0.4, 1.2) (|Q_0| = 1.3), Q_1 = (-0.6, 0.2, 0.3) (|Q_1| = 0.7), b = 1, K = 100.
    End to end R = Q_0 + Q_1 = (-0.3, 0.6, 1.5); centre of mass (0, 1/3, 0.9);
    T_k = K (|Q_k| - b)/|Q_k| Q_k: c_0 = 100 * 0.3/1.3 = 300/13, c_1 = 100 * (-0.3)/0.7 = -300/7 (Eq. 3);
    S = c_0 Q_0 Q_0^T + c_1 Q_1 Q_1^T (Eq. 28 without N delta)."""
    from fractions import Fraction as Fr
    r = np.array([[[0, 0, 0], [0.3, 0.4, 1.2], [-0.3, 0.6, 1.5]]], dtype=float)
    o = dict(zip(O.OBS_NAMES, O.observables(_params(2, K=100.0), r)[0][0]))
    c0, c1 = Fr(300, 13), Fr(-300, 7)
    want = {
        "Rx2": Fr(9, 100), "Ry2": Fr(36, 100), "Rz2": Fr(225, 100), "R2": Fr(270, 100),
        # sum_i |r_i - cm|^2 = (0 + 1/9 + 81/100) + (9/100 + 1/225 + 9/100) + (9/100 + 16/225 + 36/100) = 122/75
        "Rg2": Fr(122, 225),
        "Sxx": c0 * Fr(9, 100) + c1 * Fr(36, 100),
        "Syy": c0 * Fr(16, 100) + c1 * Fr(4, 100),
        "Szz": c0 * Fr(144, 100) + c1 * Fr(9, 100),
        "Sxy": c0 * Fr(12, 100) + c1 * Fr(-12, 100),
        "Sxz": c0 * Fr(36, 100) + c1 * Fr(-18, 100),
        "Syz": c0 * Fr(48, 100) + c1 * Fr(6, 100),
        "rod_dev_ms": Fr(9, 100), "rod_dev_max": Fr(3, 10),
    }
    vals = [float(v) for k, v in want.items() if not k.startswith("rod_dev")]
    assert len({round(abs(v), 9) for v in vals}) == len(vals)          # the 11 R / Rg / S entries are pairwise distinct
    for k, v in want.items():
        assert o[k] == pytest.approx(float(v), rel=1e-12), k


def test_initial_walk_follows_the_purpose_one_counter_layout():
    """Reading A13 / DESIGN.md section 3: link k of chain c comes from the KAT-pinned Philox block function with counter
    (k, c, step 0, purpose 1 << 28), key = (init_seed lo, hi): z = 2 u1 - 1, phi = 2 pi u2,
    Q_k = b (sqrt(1 - z^2) cos phi, sqrt(1 - z^2) sin phi, z).  Recomputed here, link by link."""
    N, b, seed, chain = 9, 1.7, 0xABCDEF01_23456789, 41
    r = O.init_random_walk(N, b, seed, [chain])[0]
    assert np.allclose(r.mean(0), 0.0, atol=1e-14)
    Q = np.diff(r, axis=0)
    for k in range(N):
        w = O.philox4x32_10([k, chain, 0, 1 << 28], [seed & 0xFFFFFFFF, seed >> 32])
        x1, x2 = (w[1] << 32) | w[0], (w[3] << 32) | w[2]
        u1, u2 = (2 * (x1 >> 12) + 1) / 2.0 ** 53, (2 * (x2 >> 12) + 1) / 2.0 ** 53
        z, phi = 2.0 * u1 - 1.0, 6.283185307179586 * u2
        s = math.sqrt(1.0 - z * z)
        assert Q[k] == pytest.approx([b * s * math.cos(phi), b * s * math.sin(phi), b * z], rel=1e-13, abs=1e-14)
    # purpose 0 (the noise stream) with the same key / chain / pair gives different words
    assert O.philox4x32_10([0, chain, 0, 0], [seed & 0xFFFFFFFF, seed >> 32]) != \
        O.philox4x32_10([0, chain, 0, 1 << 28], [seed & 0xFFFFFFFF, seed >> 32])


def test_end_to_end_autocorrelation_closed_forms():
    """PAPER.md:283 (relaxation time from the autocorrelation of the end-to-end vector; reading B3: ensemble at lag t).
    (i) two chains written out by hand; (ii) every chain rigidly rotated by theta about its own axis perpendicular
    to R0: sum R.R0 = cos(theta) sum |R0|^2; (iii) translation of the chains changes nothing; (iv) t = 0 gives 1."""
    N = 2
    r = np.array([[[0, 0, 0], [1, 0, 0], [1, 2, 2]], [[1, 1, 1], [0, 0, 0], [-1, 1, 4]]], dtype=float)
    R = O.end_to_end(N, r)
    assert np.array_equal(R, [[1, 2, 2], [-2, 0, 3]])
    R0 = np.array([[2, -1, 0.5], [1, 1, 1]])
    out = O.autocorr(N, r, R0)
    # chain 0: (1,2,2).(2,-1,0.5) = 1; chain 1: (-2,0,3).(1,1,1) = 1;  |R0|^2 = 5.25 and 3
    assert out == pytest.approx([2.0, 2.0, 8.25], rel=1e-15)
    rng = np.random.default_rng(11)
    C, N = 50, 7
    r = W.random_chains(C, N, seed=4)
    R0 = O.end_to_end(N, r)
    assert O.autocorr(N, r, R0) == pytest.approx([(R0 ** 2).sum(), ((R0 ** 2).sum(1) ** 2).sum(), (R0 ** 2).sum()], rel=1e-14)
    theta = 0.7
    rot = np.empty_like(r)
    for c in range(C):
        axis = np.cross(R0[c], rng.standard_normal(3)); axis /= np.linalg.norm(axis)       # perpendicular to R0
        K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
        Rm = np.eye(3) + math.sin(theta) * K + (1 - math.cos(theta)) * K @ K                # Rodrigues
        rot[c] = r[c] @ Rm.T + rng.standard_normal(3)                                       # rotated and shifted
    out = O.autocorr(N, rot, R0)
    assert out[0] == pytest.approx(math.cos(theta) * (R0 ** 2).sum(), rel=1e-12)
    assert out[2] == pytest.approx((R0 ** 2).sum(), rel=1e-14)


def test_failure_leaves_state_unchanged():
    """A10: coincident beads with h* = a make D singular -> reported, state untouched."""
    r = np.array([[0, 0, 0], [1.0, 0, 0], [0, 0, 0]], dtype=float)     # bead 2 on top of bead 0
    p = _params(2, dt=1e-4, hstar=0.25)
    rn, info = O.step(p, 0, 0, r)
    assert info > 0 and np.array_equal(rn, r)
