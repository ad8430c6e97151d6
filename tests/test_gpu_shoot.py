"""GPU parity tests of the shooting map (sww_shooter_create / sww_shoot): residual (3.17) and Jacobian (3.31) of the overdetermined
shooting method against the oracle (oracle/shooting.py), per column as in DESIGN.md section 6, and the
small-amplitude branch the paper prints (T = 7.19976) recovered through the device path."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from parity_util import ld

pytestmark = pytest.mark.gpu
LD = np.longdouble


@pytest.fixture(scope="module")
def sww():
    import paper_1210_5672_b200 as pkg
    assert pkg.lib_path().exists() and torch.cuda.is_available()
    return pkg


def unknowns(n, T=7.0, amp=-0.02, seed=3):
    """c_0 = T off the linear period, c_1 the carrier, the other modes decaying like the paper's small-amplitude waves"""
    rng = np.random.default_rng(seed)
    c = np.zeros(n + 1)
    c[0] = T
    c[1] = amp
    for k in range(2, n + 1):
        c[k] = 0.2 * abs(amp) * rng.standard_normal() * np.exp(-0.7 * k)
    return c


def col_err(gpu, ref):
    """per column: max |gpu - ref| / max |ref| (columns along axis 0 of both arrays)"""
    return np.abs(gpu.astype(LD) - ref).max(axis=1) / np.abs(ref).max(axis=1)


@pytest.mark.parametrize("N,n,nsteps", [(64, 6, 6), (128, 9, 5), (256, 12, 8)])   # dt inside the stability interval of the RK8 scheme (|omega_max| dt < 3)
def test_residual_and_jacobian_fp64(sww, orc_ld, N, n, nsteps):
    from oracle import shooting
    c = unknowns(n)
    S = sww.Shooter(N, n, 1.0, 1.0)
    r, J, eta, phi = S.shoot(c, nsteps, want_state=True)
    o = shooting.shoot(orc_ld, c, N, 1.0, 1.0, nsteps)
    assert float(np.abs(r.cpu().numpy().astype(LD) - o["r"]).max() / np.abs(o["r"]).max()) <= 1e-11
    e = col_err(J.cpu().numpy(), o["J"].T)
    assert float(e.max()) <= 1e-11, e
    assert float(np.abs(eta.cpu().numpy().astype(LD) - o["eta"]).max() / np.abs(o["eta"]).max()) <= 1e-11
    assert float(np.abs(phi.cpu().numpy().astype(LD) - o["phi"]).max() / np.abs(o["phi"]).max()) <= 1e-11
    # a second shot through the same handle (what a Levenberg-Marquardt iteration does): same bits for the same c, and a
    # changed period changes the result
    r2, J2 = S.shoot(c, nsteps)
    assert torch.equal(r, r2) and torch.equal(J, J2)
    c2 = c.copy()
    c2[0] += 0.1
    r3, _ = S.shoot(c2, nsteps)
    assert not torch.equal(r, r3)
    S.close()


def test_residual_and_jacobian_dd(sww, orc_q):
    from oracle import shooting
    N, n, nsteps = 64, 5, 3
    c = unknowns(n)
    S = sww.Shooter(N, n, 1.0, 1.0, prec=sww.DD)
    r, J = S.shoot(c, nsteps)
    o = shooting.shoot_quad(orc_q, c, N, 1.0, 1.0, nsteps)
    rg = r.cpu().numpy()
    dr = (rg[0].astype(LD) - o["r"][0].astype(LD)) + (rg[1].astype(LD) - o["r"][1].astype(LD))
    assert float(np.abs(dr).max() / np.abs(o["r"][0]).max()) <= 1e-25
    Jg = J.cpu().numpy()                                     # (2, n + 1, N)
    dJ = (Jg[0].astype(LD) - o["J"][0].T.astype(LD)) + (Jg[1].astype(LD) - o["J"][1].T.astype(LD))
    e = np.abs(dJ).max(axis=1) / np.abs(o["J"][0].T).max(axis=1)
    assert float(e.max()) <= 1e-25, e
    S.close()


def test_residual_and_jacobian_dd_with_sdc15(sww, orc_q):
    """the paper's quadruple-precision shooting: double-double state advanced by SDC15, two large steps to T/4"""
    from oracle import shooting
    N, n, nsteps = 64, 4, 2
    c = unknowns(n)
    S = sww.Shooter(N, n, 1.0, 1.0, prec=sww.DD)
    S.set_method("sdc15")
    r, J = S.shoot(c, nsteps)
    o = shooting.shoot_quad(orc_q, c, N, 1.0, 1.0, nsteps, method="sdc15")
    rg = r.cpu().numpy()
    dr = (rg[0].astype(LD) - o["r"][0].astype(LD)) + (rg[1].astype(LD) - o["r"][1].astype(LD))
    assert float(np.abs(dr).max() / np.abs(o["r"][0]).max()) <= 1e-25
    Jg = J.cpu().numpy()
    dJ = (Jg[0].astype(LD) - o["J"][0].T.astype(LD)) + (Jg[1].astype(LD) - o["J"][1].T.astype(LD))
    e = np.abs(dJ).max(axis=1) / np.abs(o["J"][0].T).max(axis=1)
    assert float(e.max()) <= 1e-25, e
    S.close()


@pytest.mark.parametrize("h,key,T0,nsteps", [(1.0, "T_linear_h1", 7.0, 16), (0.05, "T_linear_h0.05", 27.0, 64), (float("inf"), "T_linear_hinf", 6.0, 16)])
def test_gauss_newton_on_the_period_finds_the_linear_period(sww, h, key, T0, nsteps):
    """the small-amplitude branch: Gauss-Newton on c_0 = T alone with the device residual and Jacobian column 0 converges to the
    printed linear periods: T = 2 pi / sqrt(tanh 1) = 7.19976, 28.1110 at h = 0.05, 2 pi in deep water;
    f = r.r / 2 falls to roundoff"""
    golden = {}
    from pathlib import Path
    for line in (Path(__file__).parent / "golden" / "paper_values.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            k, v, tol = line.split()[:3]
            golden[k] = (float(v), float(tol))
    n = 1
    N = 64 if h > 0.5 else 512           # shallow water: the image surface is 2h = 0.1 away, the mesh must resolve that distance
    eps = 1e-6 if h > 0.5 else 1e-9      # and the Ursell number A lambda^2 / h^3 must be small too
    S = sww.Shooter(N, n, h, 1.0)
    T = T0
    for _ in range(6):
        r, J = S.shoot([T, eps], nsteps)
        J0 = J[0]
        T -= float((J0 @ r) / (J0 @ J0))
    want, tol = golden[key]
    assert abs(T - want) < tol
    assert float(0.5 * (r @ r)) < 1e-22
    S.close()


def test_argument_checks(sww):
    with pytest.raises(sww.SwwError):
        sww.Shooter(64, 32, 1.0)          # 2 n < N
    S = sww.Shooter(64, 2, 1.0)
    with pytest.raises(sww.SwwError):
        S.shoot([0.0, 0.1, 0.0], 4)       # the period must be positive
    with pytest.raises(sww.SwwError):
        S.shoot([7.0, 0.1, 0.0], 0)
    S.close()


def test_levenberg_marquardt_finds_a_standing_wave(sww, orc_ld):
    """Section 4.1: from the linearized solution with c_1 held fixed, Levenberg-Marquardt with delayed Jacobian
    updates (Appendix C) on the device shooting map reaches f at the roundoff floor; the ORACLE's shooting map confirms that the
    c found is time-periodic, the period sits O(c_1^2) from the linear one, and the Jacobian was re-used"""
    from oracle import shooting
    N, n, nsteps, c1 = 64, 10, 24, -0.01
    c0 = np.zeros(n + 1)
    c0[0] = 7.19976
    c0[1] = c1
    fixed = [0] * (n + 1)
    fixed[1] = 1
    S = sww.Shooter(N, n, 1.0, 1.0)
    r0 = S.residual(c0, nsteps)
    f0 = float(0.5 * (r0 @ r0))
    c, rep = S.solve(c0, nsteps, fixed=fixed, delta0=0.1, f_tol=1e-26, max_iter=60)
    S.close()
    assert c[1] == c1
    assert rep["f"] < 1e-24 and rep["f"] < 1e-12 * f0, (rep, f0)
    assert rep["residual_evals"] >= rep["jacobian_evals"]
    assert 1e-8 < abs(c[0] - 7.19976) < 0.01          # a nonlinear correction of order c_1^2 to the period
    assert abs(c[2]) > 1e-6 and abs(c[3]) > 1e-9     # second and third harmonics were found
    o = shooting.shoot(orc_ld, np.array(c), N, 1.0, 1.0, nsteps)
    assert float(0.5 * (o["r"] @ o["r"])) < 1e-24


def test_period_correction_changes_sign_with_depth(sww):
    """(4.36): the period of small standing waves first decreases with amplitude for h < 1.0581 and increases
    from the start for h > 1.0581.  Standing waves are computed by Levenberg-Marquardt on the device shooting map at two small
    amplitudes per depth; omega_2 = lim 2 (omega - omega_0) / eps^2 with eps = A = 2 |c_1| omega_0 ((4.35): phi(x, 0) = 2 c_1 cos x,
    A/B = sqrt(tanh h)) is extrapolated to zero amplitude, compared with the printed formula, and its root in h with the printed 1.0581."""
    import math
    golden = {}
    from pathlib import Path
    for line in (Path(__file__).parent / "golden" / "paper_values.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            k, v, tol = line.split()[:3]
            golden[k] = (float(v), float(tol))
    N, n, nsteps = 64, 8, 24

    def omega2_measured(h):
        w0 = math.sqrt(math.tanh(h))
        S = sww.Shooter(N, n, h, 1.0)
        vals = []
        for c1 in (-0.004, -0.008):
            c0 = np.zeros(n + 1)
            c0[0], c0[1] = 2 * math.pi / w0, c1
            fixed = [0] * (n + 1)
            fixed[1] = 1
            c, rep = S.solve(c0, nsteps, fixed=fixed, delta0=0.1, f_tol=1e-28, max_iter=60)
            assert rep["f"] < 1e-24, rep
            eps = 2 * abs(c1) * w0
            vals.append(2 * (2 * math.pi / c[0] - w0) / eps ** 2)
        S.close()
        return (4 * vals[0] - vals[1]) / 3          # the O(eps^2) term of the measured ratio removed

    def omega2_formula(h):
        w = math.sqrt(math.tanh(h))
        return (9 * w ** -7 - 12 * w ** -3 - 3 * w - 2 * w ** 5) / 32

    hs = [1.0, 1.05, 1.066]
    m = [omega2_measured(h) for h in hs]
    for h, v in zip(hs, m):
        assert abs(v - omega2_formula(h)) < 2e-3 * max(abs(omega2_formula(1.0)), abs(v)), (h, v, omega2_formula(h))
    assert m[0] > 0 and m[1] > 0 and m[2] < 0         # positive below 1.0581, negative above
    h_root = hs[1] + (hs[2] - hs[1]) * m[1] / (m[1] - m[2])      # secant between the bracketing depths (omega_2 is nearly linear in h there)
    want, tol = golden["h_omega2_sign"]
    assert abs(h_root - want) < 3e-4, (h_root, want)


@pytest.mark.parametrize("N,n,nsteps,h,sigma,filt", [(64, 6, 10, 1.0, 0.0, True), (128, 9, 12, float("inf"), 0.0, True), (32, 5, 32, 1.0, 0.3, False)])
def test_adjoint_gradient_equals_jacobian_transpose_times_residual(sww, orc_ld, N, n, nsteps, h, sigma, filt):
    """Section 3.2, (3.25)-(3.30): the gradient of f from ONE backward solve of the adjoint system equals
    df/dc_k = <(0, phi), (0, phidot_k)> = (J^T r)_k from the n variational solutions -- against the oracle's J^T r (its J is pinned by
    finite differences) and against the device's own J^T r; f itself against r.r / 2"""
    from oracle import shooting
    c = unknowns(n, T=7.1, amp=-0.03)
    S = sww.Shooter(N, n, h, 1.0, filter=filt)
    S.set_sigma(sigma)
    f, grad = S.gradient(c, nsteps)
    r, J = S.shoot(c, nsteps)
    S.close()
    own = (J @ r).cpu().numpy()
    o = shooting.shoot(orc_ld, c, N, h, 1.0, nsteps, filter=filt, sigma=sigma)
    want = np.asarray(o["J"].T @ o["r"], dtype=np.float64)
    scale = float(np.abs(want).max())
    assert abs(f - float(0.5 * (o["r"] @ o["r"]))) <= 1e-11 * f
    assert float(np.abs(grad - want).max()) <= 1e-11 * scale, (grad, want)      # the parity bar against the oracle
    assert float(np.abs(grad - own).max()) <= 1e-12 * scale                      # measured: 1e-15 (the two device paths share the forward solve)
    assert scale > 1e-6
