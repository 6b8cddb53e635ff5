"""Pins for the Cohen-Pade bead-spring option of the oracle (Eq. 4 with
alpha = 3, beta = 1; :305-307 the BS-20-25 comparison model).  The paper states the semi-implicit scheme for the Fraenkel
rod only (Eqs. 13-17); for the spring law of Eq. 4 the same Eq. 13 gives a cubic for the fractional extension (DESIGN.md
reading B4).  Pinned by: hand values and limits of the force law, an independent cubic solver (numpy.roots), the
Eq. 13 identity, finite extensibility, a numpy/LAPACK restatement of the whole step, and the equilibrium distribution
of a dumbbell, P(x) ~ x^2 exp(-nu x^2 / 2) (1 - x^2)^nu, integrated by quadrature."""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle as O
from paper_2208_06559_b200 import workloads as W


def _p(N, **kw):
    kw.setdefault("dt", 1e-3)
    kw.setdefault("spring_kind", 1)
    kw.setdefault("nu", 25.0)
    return O.Params(n_rods=N, **kw)


def test_force_law_hand_values_and_limits():
    p = _p(1)                                                 # b = 1, nu = 25: full extension 25
    # r^ = 0.5: (3 * 0.5 - 0.125) / 0.75 = 11/6
    assert O.spring_coeff(p, 12.5) * 12.5 == pytest.approx(11.0 / 6.0, rel=1e-14)
    # r^ = 0.8: (2.4 - 0.512) / 0.36 = 1.888 / 0.36
    assert O.spring_coeff(p, 20.0) * 20.0 == pytest.approx(1.888 / 0.36, rel=1e-13)
    # Hookean limit |F| -> 3 r^  (inverse Langevin function at small extension)
    for x in (1e-3, 1e-5):
        assert O.spring_coeff(p, 25.0 * x) * 25.0 * x / x == pytest.approx(3.0, rel=3 * x * x)
    # finite extensibility: |F| (1 - r^) -> 1 as r^ -> 1   ((3 - 1) / (1 + 1))
    for eps in (1e-4, 1e-7):
        assert O.spring_coeff(p, 25.0 * (1 - eps)) * 25.0 * (1 - eps) * eps == pytest.approx(1.0, rel=5 * eps)
    # length unit b: force in kT / b, extension relative to nu b
    p2 = _p(1, b=2.0, nu=10.0)
    assert O.spring_coeff(p2, 10.0) * 10.0 == pytest.approx((11.0 / 6.0) / 2.0, rel=1e-14)
    # T is along Q
    r = np.array([[0.0, 0, 0], [3.0, 4.0, 12.0]])             # |Q| = 13, r^ = 0.52
    T = O.spring_tensions(p, r)[0]
    F = (3 * 0.52 - 0.52 ** 3) / (1 - 0.52 ** 2)
    assert T == pytest.approx(F * np.array([3.0, 4.0, 12.0]) / 13.0, rel=1e-13)


def test_implicit_length_is_the_root_of_the_cubic_and_of_eq13():
    rng = np.random.default_rng(3)
    for b, nu, dt in ((1.0, 25.0, 1e-3), (2.0, 10.0, 1e-2), (1.0, 3.0, 0.2)):
        p = _p(1, b=b, nu=nu, dt=dt)
        L, c = nu * b, 2 * dt / (nu * b * b)
        for Yn in np.concatenate([rng.uniform(0, 2 * L, 40), [1e-9, 0.999 * L, L, 50 * L]]):
            q = O.implicit_length(p, Yn)
            assert 0.0 <= q < L                                # finite extensibility, however large |Y|
            # Eq. 13 with D_ii = I and T parallel to Q':  |Y| = |Q'| + 2 dt |T(|Q'|)|
            # (near full extension d|Y|/d|Q'| ~ dt / (1 - x)^2: one ulp of |Q'| is a relative 1e-10 of |Y| there)
            assert q + 2 * dt * O.spring_coeff(p, q) * q == pytest.approx(Yn, rel=1e-11 if Yn < 0.9 * L else 1e-8, abs=1e-13)
            # the same root from a general polynomial solver
            y = Yn / L
            roots = np.roots([1 + c, -y, -(1 + 3 * c), y])
            inside = [z.real for z in roots if abs(z.imag) < 1e-12 and -1e-14 <= z.real < 1]
            assert len(inside) == 1 and q / L == pytest.approx(inside[0], rel=1e-9, abs=1e-12)
    # dt -> 0: the explicit value
    assert O.implicit_length(_p(1, dt=1e-12), 7.0) == pytest.approx(7.0, rel=1e-10)


def _numpy_step_cp(p, r, dW):
    """independent restatement of one step with the Cohen-Pade spring (numpy + LAPACK + numpy.roots)."""
    cp = p.c()
    N = p.n_rods
    L = cp.nu * cp.b
    Q = np.diff(r, axis=0)
    q = np.linalg.norm(Q, axis=1, keepdims=True)
    x = q / L
    T = (3 * x - x ** 3) / (1 - x ** 2) / cp.b * Q / q
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
    Lc = np.linalg.cholesky(D)
    kap = np.array(list(cp.kappa)).reshape(3, 3)
    u = cp.dt * (r @ kap.T + (D @ F.reshape(-1)).reshape(-1, 3)) + (Lc @ dW).reshape(-1, 3)
    Y = Q + np.diff(u, axis=0) + 2 * cp.dt * T
    Qn = np.empty_like(Y)
    c = 2 * cp.dt / (cp.nu * cp.b ** 2)
    for k in range(N):
        Yn = np.linalg.norm(Y[k]); y = Yn / L
        roots = np.roots([1 + c, -y, -(1 + 3 * c), y])
        xr = [z.real for z in roots if abs(z.imag) < 1e-12 and 0 <= z.real < 1][0]
        Qn[k] = Y[k] / Yn * xr * L
    rn = np.zeros_like(r); rn[1:] = np.cumsum(Qn, axis=0)
    return rn - rn.mean(0)


@pytest.mark.parametrize("N", [1, 2, 5, 20])
def test_whole_step_against_numpy_restatement(N):
    kap = np.array([[0.3, 1.0, 0.0], [0.0, -0.1, 0.2], [0.5, 0.0, -0.2]]) * 0.1
    nu = 25.0
    rng = np.random.default_rng(N)
    Qs = rng.standard_normal((N, 3)) * math.sqrt(nu / 3.0)            # Gaussian springs: <Q^2> = nu b^2
    Qs *= np.minimum(1.0, 0.9 * nu / np.linalg.norm(Qs, axis=1, keepdims=True))
    r = np.zeros((N + 1, 3)); r[1:] = np.cumsum(Qs, axis=0); r -= r.mean(0)
    for nk in (0, 1):
        p = _p(N, dt=1e-3, hstar=0.105, a=1.539, nu=nu, kappa=kap, seed=5, noise_kind=nk)   # the paper's BS-20-25 pairing (:307)
        rn, info = O.step(p, 2, 9, r)
        assert info == 0
        want = _numpy_step_cp(p, r, O.noise_dW(p, 2, 9))
        assert np.allclose(rn, want, rtol=1e-9, atol=1e-10)
    # the Fraenkel path is untouched by the new fields
    pf = O.Params(n_rods=N, dt=1e-4, seed=5, nu=25.0)
    pf0 = O.Params(n_rods=N, dt=1e-4, seed=5)
    rr = W.random_chains(1, N, seed=1, rod_jitter=0.01)[0]
    assert np.array_equal(O.step(pf, 0, 0, rr)[0], O.step(pf0, 0, 0, rr)[0])


def test_dumbbell_equilibrium_distribution():
    """free-draining Cohen-Pade dumbbells relax to P(x) ~ x^2 exp(-nu x^2/2) (1-x^2)^nu, x = |Q|/(nu b)
    (U/kT = nu [x^2/2 - ln(1-x^2)] is the integral of Eq. 4): <Q^2> from quadrature against the ensemble."""
    nu, C = 10.0, 4000
    w = lambda x: x * x * math.exp(-nu * x * x / 2) * (1 - x * x) ** nu
    m2 = integrate.quad(lambda x: x * x * w(x), 0, 1)[0] / integrate.quad(w, 0, 1)[0] * nu * nu
    p = _p(1, dt=2e-3, hstar=0.0, nu=nu, seed=17)
    r = O.init_random_walk(1, 1.0, 5, range(C))
    r, info = O.step_ensemble(p, r, 0, 3000)                  # 6 time units, dumbbell relaxation time nu/12 = 0.83
    assert not info.any()
    acc = []
    for k in range(8):                                        # 8 samples one relaxation time apart
        r, info = O.step_ensemble(p, r, 3000 + 500 * k, 500)
        acc.append((np.diff(r, axis=1)[:, 0] ** 2).sum(1))
    Q2 = np.concatenate(acc)
    se = Q2.std() / math.sqrt(Q2.size / 2)                    # samples one relaxation time apart: ~ half independent
    assert abs(Q2.mean() - m2) < 4 * se + 0.01 * m2           # O(dt) bias of the first-order scheme inside 1 %
    assert Q2.max() < (nu * 1.0) ** 2                         # never beyond full extension
