"""Pins of the oracle's mesh refinement (2.10)-(2.11), against what the paper and the mathematics fix
(no GPU, no CUDA code involved): the printed properties of E, a closed-form harmonic function sampled at the refined points,
and the fact that the right-hand sides, the time stepping and the respacing are statements about functions of x, so their
values cannot depend on the mesh they are sampled on (beyond spectrally small interpolation errors)."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from test_oracle_pins import LD, PI, ld, split_ld


@pytest.fixture()
def orc(orc_ld):
    yield orc_ld
    orc_ld.set_mesh()   # back to the uniform mesh whatever the test did


def xi_points(orc, N):
    """x_j = xi(alpha_j) of the oracle's current mesh, long double"""
    xp, E, E1 = orc.mesh_tables(N)
    return 2 * PI * np.arange(N, dtype=LD) / N + ld(xp), ld(E), ld(E1)


@pytest.mark.parametrize("rho", [1.0, 0.6, 0.25, 0.08])
def test_mesh_function_properties(orc, rho):
    """(2.11): min/max of E at 0 and pi, their ratio rho; E has mean one (P in (2.10)), so xi(2 pi) = 2 pi;
    xi' = E and xi'' = E1 (spectral differentiation is exact on these trigonometric polynomials); the two variants mirror."""
    N = 64
    orc.set_mesh(rho, 0)
    x0, E0, E10 = xi_points(orc, N)
    lo_, hi_ = 8 * LD(rho) / (5 + 3 * LD(rho)), 8 / (5 + 3 * LD(rho))
    assert abs(E0[N // 2] - lo_) < 1e-18 and abs(E0[0] - hi_) < 1e-18          # refined (small spacing) at x = pi
    assert abs(E0.min() / E0.max() - rho) < 1e-18
    assert abs(E0.mean() - 1) < 1e-18
    assert np.all(np.diff(x0) > 0) and x0[0] == 0 and x0[-1] < 2 * PI
    assert abs(x0[N // 2] - PI) < 1e-18                                         # xi(pi) = pi: the crests stay on mesh points
    xp = x0 - 2 * PI * np.arange(N, dtype=LD) / N
    assert np.abs(ld(orc.multiplier(oracle.MUL_D, split_ld(xp))) - (E0 - 1)).max() < 2e-17
    assert np.abs(ld(orc.multiplier(oracle.MUL_D, split_ld(E0))) - E10).max() < 2e-17
    orc.set_mesh(rho, 1)
    x1, E1_, E11 = xi_points(orc, N)
    assert np.abs(E1_ - np.roll(E0, N // 2)).max() < 1e-18                      # cos^4 variant = sin^4 variant shifted by pi
    assert abs(E1_[0] - lo_) < 1e-18
    assert np.abs(E11 - np.roll(E10, N // 2)).max() < 1e-18


def harmonic(x, h, k, coef):
    """phi = cosh(k y) cos(k x) on y = h + eta(x), eta a cosine polynomial: samples at the points x and the exact G phi, phi_x, phi_y"""
    m = np.arange(len(coef), dtype=LD)
    eta = sum(LD(c) * np.cos(mm * x) for mm, c in zip(m, coef))
    ex = sum(-LD(c) * mm * np.sin(mm * x) for mm, c in zip(m, coef))
    Y = LD(h) + eta
    phi = np.cosh(k * Y) * np.cos(k * x)
    px = -k * np.cosh(k * Y) * np.sin(k * x)
    py = k * np.sinh(k * Y) * np.cos(k * x)
    return eta, phi, py - ex * px, px, py


@pytest.mark.parametrize("rho,where,h", [(0.4, 0, 1.0), (0.4, 1, 1.0), (0.15, 0, 0.5), (0.5, 1, float("inf"))])
def test_harmonic_function_on_refined_mesh(orc, rho, where, h):
    """(2.5)-(2.9) with x = xi(alpha): G phi, phi_x, phi_y of a harmonic function at the refined points, closed form.  A wrong
    zeta', zeta'', x-difference, diagonal limit or 1/|xi'| factor fails this at O(1)."""
    coef = [0.0, 0.07, -0.03, 0.015, 0.0, 0.004]
    errs = []
    for N in (32, 64, 128, 256):
        orc.set_mesh(rho, where)
        x, _, _ = xi_points(orc, N)
        if np.isinf(h):   # deep water: phi = e^{k y} cos(k x) about y = eta
            m = np.arange(len(coef), dtype=LD)
            eta = sum(LD(c) * np.cos(mm * x) for mm, c in zip(m, coef))
            ex = sum(-LD(c) * mm * np.sin(mm * x) for mm, c in zip(m, coef))
            phi, px, py = np.exp(2 * eta) * np.cos(2 * x), -2 * np.exp(2 * eta) * np.sin(2 * x), 2 * np.exp(2 * eta) * np.cos(2 * x)
            w = py - ex * px
        else:
            eta, phi, w, px, py = harmonic(x, h, 2, coef)
        z = np.zeros((1, N))
        out, base = orc.dtn_linearized(split_ld(eta), h, split_ld(phi), z, z, want_base=True)
        got = ld(orc.dtn_apply(split_ld(eta), h, split_ld(phi)))[0]
        errs.append(float(np.abs(got - w).max() / np.abs(w).max()))
    assert errs[1] < 0.05 * errs[0] and errs[2] < 0.05 * errs[1] + 1e-17, errs     # spectral convergence
    assert errs[3] < 3e-16 / rho ** 2, errs                                         # roundoff grows as the spacing shrinks
    assert np.abs(ld(base["u"]) - px).max() < 3e-15 / rho ** 2
    assert np.abs(ld(base["v"]) - py).max() < 3e-15 / rho ** 2
    assert np.abs(ld(base["W0"]) - w).max() < 3e-15 / rho ** 2


def test_respacing_reproduces_functions_of_x(orc):
    """from the uniform mesh the stored samples are a trigonometric polynomial in alpha, so the respaced values
    are the polynomial itself at the new points (exact up to rounding); between two refined meshes the error is spectrally small."""
    f = lambda x: np.cos(3 * x) + LD(0.5) * np.sin(5 * x) - LD(0.25) * np.cos(11 * x)
    Mo, Mn = 48, 80   # neither a power of two
    a = 2 * PI * np.arange(Mo, dtype=LD) / Mo
    orc.set_mesh(0.3, 0)
    xn, _, _ = xi_points(orc, Mn)
    got = ld(orc.respace(split_ld(f(a)), (Mo, 1.0, 0), (Mn, 0.3, 0)))
    assert np.abs(got - f(xn)).max() < 2e-17
    orc.set_mesh(0.5, 1)
    xo, _, _ = xi_points(orc, 128)
    got = ld(orc.respace(split_ld(np.stack([f(xo), np.cos(xo)])), (128, 0.5, 1), (Mn, 0.3, 0)))
    assert np.abs(got[0] - f(xn)).max() < 1e-15 and np.abs(got[1] - np.cos(xn)).max() < 1e-15
    same = ld(orc.respace(split_ld(f(xo)), (128, 0.5, 1), (128, 0.5, 1)))     # onto itself: beta_j = alpha_j
    assert np.abs(same - f(xo)).max() < 1e-17


def smooth_state(x):
    """a smooth wave state and two variational columns as functions of x (cosine/sine polynomials with decaying coefficients)"""
    eta = sum(LD(0.08) * LD(0.45) ** k * np.cos(k * x) for k in range(1, 9))
    phi = sum(LD(0.11) * LD(0.4) ** k * np.cos(k * x + LD(0.3) * k) for k in range(1, 9))
    de = np.stack([np.cos(2 * x) + LD(0.2) * np.sin(x), LD(0.5) * np.sin(3 * x)])
    dp = np.stack([np.sin(x) - LD(0.3) * np.cos(4 * x), np.cos(x) + LD(0.1) * np.cos(2 * x)])
    return eta, phi, de, dp


@pytest.mark.parametrize("rho,where,sigma,h", [(0.5, 0, 0.0, 1.0), (0.35, 1, 0.3, 0.7), (0.6, 0, 0.2, float("inf"))])
def test_right_hand_sides_do_not_depend_on_the_mesh(orc, rho, where, sigma, h):
    """(2.1), (B.1)-(B.4) are equations between functions of x: evaluated on the refined mesh they must equal the uniform-mesh
    values interpolated to the refined points (both resolved to roundoff here).  Pins d/dx = (1/xi') d/dalpha in every term,
    the mean over x removed by P, and the weight of the energy integral."""
    N = 128
    a = 2 * PI * np.arange(N, dtype=LD) / N
    orc.set_mesh()
    eta, phi, de, dp = smooth_state(a)
    ref = orc.rhs(split_ld(eta), split_ld(phi), h, 1.0, split_ld(de), split_ld(dp), filter=False, sigma=sigma)
    orc.set_mesh(rho, where)
    x, E, _ = xi_points(orc, N)
    eta, phi, de, dp = smooth_state(x)
    got = orc.rhs(split_ld(eta), split_ld(phi), h, 1.0, split_ld(de), split_ld(dp), filter=False, sigma=sigma)
    for key in ("eta_t", "phi_t", "deta_t", "dphi_t"):
        want = ld(orc.respace(ref[key], (N, 1.0, 0), (N, rho, where)))
        scale = np.abs(want).max()
        assert np.abs(ld(got[key]) - want).max() < 2e-15 * scale, key
    assert abs(ld(got["energy"]) - ld(ref["energy"])) < 1e-17
    assert abs((ld(got["phi_t"]) * E).mean()) < 1e-18          # zero mean over x, not over alpha
    assert abs((ld(got["eta_t"]) * E).mean()) < 1e-17          # mass conservation: int eta_t dx = 0


def test_time_stepping_across_a_respacing(orc):
    """Section 2.2: a uniform segment followed by a finer, refined one gives the solution that the uniform
    mesh alone gives, sampled at the refined points; the energy is the same number on both meshes."""
    h, g, dt, N, M2, rho = 1.0, 1.0, 0.05, 128, 160, 0.5
    a = 2 * PI * np.arange(N, dtype=LD) / N
    eta0, phi0, de0, dp0 = smooth_state(a)
    orc.set_mesh()
    ref = orc.rk_advance(split_ld(eta0), split_ld(phi0), h, g, dt, 8, split_ld(de0[:1]), split_ld(dp0[:1]), filter=False, want_energy=True)
    mid = orc.rk_advance(split_ld(eta0), split_ld(phi0), h, g, dt, 4, split_ld(de0[:1]), split_ld(dp0[:1]), filter=False)
    old, new = (N, 1.0, 0), (M2, rho, 0)
    st = {k: orc.respace(mid[k], old, new) for k in ("eta", "phi", "deta", "dphi")}
    orc.set_mesh(rho, 0)
    fin = orc.rk_advance(st["eta"], st["phi"], h, g, dt, 4, st["deta"], st["dphi"], filter=False, want_energy=True)
    for k in ("eta", "phi", "deta", "dphi"):
        want = ld(orc.respace(ref[k], old, new))
        assert np.abs(ld(fin[k]) - want).max() < 1e-13 * max(1.0, float(np.abs(want).max())), k
    assert abs(ld(fin["energies"])[-1] - ld(ref["energies"])[-1]) < 1e-15


def test_shooting_with_segments_is_mesh_independent(orc):
    """(3.17): f = r.r / 2 approximates (1/4pi) int phi(x, T/4)^2 dx and (J^T r)_k = (1/2pi) int phidot_k phi dx by the
    trapezoidal rule with dx = E dalpha -- numbers that cannot depend on the mesh strategy.  A one-segment uniform shot and a three-
    segment refined shot (both ends, growing M) of the same c agree in f, in the gradient J^T r and in the Gauss-Newton matrix J^T J;
    the residual itself is the uniform one interpolated to the last mesh times sqrt(E/M).  A missing or misplaced weight fails this."""
    from oracle import shooting
    h, g = 1.0, 1.0
    c = np.array([7.1, 0.02, 0.004, -0.001, 0.0005])
    one = shooting.shoot(orc, c, 64, h, g, 24, filter=False)
    segs = [(64, 0.4, 1.0, 0, 10), (80, 0.3, 0.6, 0, 8), (96, 0.3, 0.45, 1, 8)]
    seg = shooting.shoot_segments(orc, c, segs, h, g, filter=False)
    assert seg["r"].shape == (96,) and seg["J"].shape == (96, 5)
    f1, f2 = 0.5 * one["r"] @ one["r"], 0.5 * seg["r"] @ seg["r"]
    assert abs(f1 - f2) < 1e-12 * f1
    g1, g2 = one["J"].T @ one["r"], seg["J"].T @ seg["r"]
    assert np.abs(g1 - g2).max() < 1e-11 * np.abs(g1).max()
    H1, H2 = one["J"].T @ one["J"], seg["J"].T @ seg["J"]
    assert np.abs(H1 - H2).max() < 1e-11 * np.abs(H1).max()
    orc.set_mesh(0.45, 1)
    _, E, _ = xi_points(orc, 96)
    orc.set_mesh()
    want = ld(orc.respace(split_ld(one["phi"]), (64, 1.0, 0), (96, 0.45, 1))) * np.sqrt(E / 96)
    assert np.abs(seg["r"] - want).max() < 1e-11 * np.abs(want).max()
    # one segment on the uniform mesh through shoot_segments is shoot itself
    same = shooting.shoot_segments(orc, c, [(64, 1.0, 1.0, 0, 24)], h, g, filter=False)
    assert np.abs(same["r"] - one["r"]).max() == 0 and np.abs(same["J"] - one["J"]).max() == 0


def test_shooting_segments_quad_matches_long_double(orc, orc_q):
    """the __float128 build of the segmented map against the long-double one (same c, same segments)"""
    from oracle import shooting
    c = np.array([7.0, -0.01, 0.003, 0.001])
    segs = [(32, 0.5, 1.0, 0, 3), (64, 0.5, 0.5, 1, 3)]
    try:
        a = shooting.shoot_segments(orc, c, segs, 1.0, 1.0)
        b = shooting.shoot_segments_quad(orc_q, c, segs, 1.0, 1.0)
    finally:
        orc_q.set_mesh()
    assert np.abs(ld(b["r"]) - a["r"]).max() < 5e-18
    assert np.abs(ld(b["J"]) - a["J"]).max() < 5e-17


@pytest.mark.parametrize("rho,where,sigma", [(0.5, 0, 0.0), (0.4, 1, 0.5)])
def test_adjoint_identity_on_refined_mesh(orc_q, rho, where, sigma):
    """(B.4)-(B.6), PAPER.md:716-747 on the mesh (2.10): <DF(q) qdot, q~> = <qdot, DF(q)^* q~> with the inner product
    (1/2pi) int (.) dx = (1/M) sum_j (.)_j E_j.  The stored samples are smooth functions of alpha (hence of x); the gap between the
    two sides closes spectrally with M, as on the uniform mesh."""
    import sww_inputs as si
    h, gaps = 1.0, []
    try:
        for N in (32, 64, 128):
            rng = np.random.default_rng(11)
            def smooth(amp):
                c, s_ = np.zeros(7), np.zeros(7)
                c[1:] = amp * rng.standard_normal(6) * np.exp(-0.6 * np.arange(1, 7))
                s_[1:] = amp * rng.standard_normal(6) * np.exp(-0.6 * np.arange(1, 7))
                return si.synth(N, c, s_)[0].astype(LD)
            eta, phi = smooth(0.05), smooth(0.1)
            qd = (np.stack([smooth(1.0), smooth(1.0)]), np.stack([smooth(1.0), smooth(1.0)]))
            qt = (np.stack([smooth(1.0), smooth(1.0)]), np.stack([smooth(1.0), smooth(1.0)]))
            sp = lambda a: split_ld(a) if a.ndim == 1 else tuple(np.stack(t) for t in zip(*[split_ld(r) for r in a]))
            orc_q.set_mesh(rho, where)
            E = ld(orc_q.mesh_tables(N)[1])
            lin = orc_q.rhs(sp(eta), sp(phi), h, 1.0, sp(qd[0]), sp(qd[1]), filter=False, sigma=sigma)
            adj = orc_q.adjoint_rhs(sp(eta), sp(phi), h, 1.0, sp(qt[0]), sp(qt[1]), sigma=sigma)
            gap = 0.0
            for a in range(2):
                for b in range(2):
                    lhs = ((ld(lin["deta_t"])[a] * qt[0][b] + ld(lin["dphi_t"])[a] * qt[1][b]) * E).mean()
                    rhs = ((qd[0][a] * ld(adj["eta_s"])[b] + qd[1][a] * ld(adj["phi_s"])[b]) * E).mean()
                    assert abs(lhs) > 1e-3
                    gap = max(gap, float(abs(lhs - rhs)))
            gaps.append(gap)
    finally:
        orc_q.set_mesh()
    assert gaps[0] < 1e-3 and gaps[1] < 1e-4 * gaps[0] and gaps[2] < 1e-15, gaps
