"""Host logic of the Levenberg-Marquardt iteration with delayed Jacobian updates (Appendix C, 751-818; lm.cu) on problems
with known answers -- no GPU involved: the callback is Python, the algebra (thin SVD, (C.5), rules 1-4) is the library's."""
from __future__ import annotations

import numpy as np
import pytest


@pytest.fixture(scope="module")
def sww():
    import paper_1210_5672_b200 as pkg
    assert pkg.lib_path().exists()
    return pkg


def test_linear_least_squares_in_one_jacobian(sww):
    """r = A c - b: the first full step is the least-squares solution (lambda = 0 inside the trust region); one Jacobian suffices"""
    rng = np.random.default_rng(1)
    A, b = rng.standard_normal((20, 5)), rng.standard_normal(20)
    fun = lambda c, wj: (A @ c - b, A if wj else None)
    c, rep = sww.lm_minimize(fun, np.zeros(5), 20, delta0=100.0, f_tol=0.0, g_tol=1e-13)
    want = np.linalg.lstsq(A, b, rcond=None)[0]
    assert np.abs(c - want).max() < 1e-13
    assert rep["jacobian_evals"] <= 2
    assert abs(rep["f"] - 0.5 * np.sum((A @ want - b) ** 2)) < 1e-14


def test_trust_region_step_has_the_prescribed_length(sww):
    """(C.4)-(C.5): with a radius shorter than the Gauss-Newton step the first accepted step has |p| = Delta and points along
    -(J^T J + lambda I)^-1 J^T r"""
    rng = np.random.default_rng(2)
    A, b = rng.standard_normal((12, 4)), rng.standard_normal(12)
    seen = []
    def fun(c, wj):
        seen.append(c.copy())
        return A @ c - b, (A if wj else None)
    sww.lm_minimize(fun, np.zeros(4), 12, delta0=0.05, max_iter=1)
    p = seen[1] - seen[0]
    assert abs(np.linalg.norm(p) - 0.05) < 1e-12
    # the multiplier that gives this length
    g = A.T @ (-b)
    lo, hi = 0.0, 1e6
    for _ in range(200):
        lam = 0.5 * (lo + hi)
        q = np.linalg.solve(A.T @ A + lam * np.eye(4), -g)
        lo, hi = (lam, hi) if np.linalg.norm(q) > 0.05 else (lo, lam)
    assert np.abs(p - q).max() < 1e-9


def test_rosenbrock_residuals(sww):
    """small-residual nonlinear least squares: r = (10 (y - x^2), 1 - x) from (-1.2, 1) -> (1, 1), f -> 0, with re-used Jacobians"""
    def fun(c, wj):
        x, y = c
        r = np.array([10 * (y - x * x), 1 - x])
        J = np.array([[-20 * x, 10.0], [-1.0, 0.0]]) if wj else None
        return r, J
    c, rep = sww.lm_minimize(fun, np.array([-1.2, 1.0]), 2, delta0=1.0, f_tol=1e-28, max_iter=200)
    assert np.abs(c - 1).max() < 1e-10
    assert rep["f"] < 1e-20
    assert rep["residual_evals"] > rep["jacobian_evals"]      # J is re-used between evaluations (rule 4)


def test_fixed_unknowns_stay_fixed(sww):
    """exponential fit y = a exp(-b t) + d with d held constant ("holding c_1 constant")"""
    t = np.linspace(0, 2, 30)
    y = 2.0 * np.exp(-1.5 * t) + 0.25
    def fun(c, wj):
        a, b, d = c
        e = np.exp(-b * t)
        J = np.stack([e, -a * t * e, np.ones_like(t)], axis=1) if wj else None
        return a * e + d - y, J
    c, rep = sww.lm_minimize(fun, np.array([1.0, 1.0, 0.25]), 30, fixed=[0, 0, 1], delta0=1.0, f_tol=1e-28, max_iter=100)
    assert c[2] == 0.25
    assert abs(c[0] - 2.0) < 1e-9 and abs(c[1] - 1.5) < 1e-9


def test_rank_deficient_jacobian_is_survived(sww):
    """two identical columns: sigma_min = 0; the step lives in the range of V with sigma > 0 and the residual still goes to zero"""
    rng = np.random.default_rng(3)
    a = rng.standard_normal(10)
    A = np.stack([a, a, rng.standard_normal(10)], axis=1)
    b = A @ np.array([1.0, 2.0, -1.0])
    fun = lambda c, wj: (A @ c - b, A if wj else None)
    c, rep = sww.lm_minimize(fun, np.zeros(3), 10, delta0=10.0)
    assert np.abs(A @ c - b).max() < 1e-12
    assert abs(c[0] - c[1]) < 1e-12          # minimum-norm direction: the null vector (1, -1, 0) is not excited
