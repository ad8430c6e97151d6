"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA code involved).

Every test names the passage (PAPER.md:<line>) or the textbook identity it checks, and is chosen so that a
plausible mistake in oracle/sww_oracle.c (a dropped term, a wrong sign or index, a transposed operand) fails it.
"""
from __future__ import annotations

import math
from pathlib import Path

import mpmath
import numpy as np
import pytest

import oracle
import sww_inputs as si

GOLDEN = Path(__file__).resolve().parent / "golden"
LD = np.longdouble
PI = 4 * np.arctan(LD(1))   # long-double pi (np.pi is only a double)


def ld(x):
    """(hi, lo) -> numpy long double"""
    if isinstance(x, tuple):
        return np.asarray(x[0], dtype=LD) + np.asarray(x[1], dtype=LD)
    return np.asarray(x, dtype=LD)


def golden():
    out = {}
    for line in (GOLDEN / "paper_values.txt").read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            k, v, t = line.split()
            out[k] = (float(v), float(t))
    return out


def pure_modes(N, ks, kind="cos"):
    """exact (hi, lo) samples of cos(k alpha_j) / sin(k alpha_j)"""
    K = max(ks) + 1
    cc = np.zeros((len(ks), K))
    for i, k in enumerate(ks):
        cc[i, k] = 1.0
    return si.synth_dd(N, cc) if kind == "cos" else si.synth_dd(N, np.zeros_like(cc), cc)


# ----------------------------------------------------------------------------------------------------------
# T1: flat-surface symbol G[e^{ikx}] = k tanh(kh) e^{ikx}   ((4.34)) -- pins the image-kernel sign (R1),
# the 1/N scaling, the diagonal limits and the D/H conventions at once.
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec,tol", [("ld", 2e-16), ("q", 5e-30)])
@pytest.mark.parametrize("h", [1.0, float("inf")])
def test_flat_symbol_all_modes(prec, tol, h):
    N = 64
    orc = oracle.Oracle(prec)
    ks = list(range(1, N // 2))
    for kind in ("cos", "sin"):
        f = pure_modes(N, ks, kind)
        whi, wlo = orc.dtn_apply(np.zeros(N), h, f)
        with mpmath.workdps(40):
            for i, k in enumerate(ks):
                s = mpmath.mpf(k) * mpmath.tanh(mpmath.mpf(k) * h) if math.isfinite(h) else mpmath.mpf(k)
                for j in range(0, N, 5):
                    got = mpmath.mpf(float(whi[i, j])) + mpmath.mpf(float(wlo[i, j]))
                    want = s * (mpmath.mpf(float(f[0][i, j])) + mpmath.mpf(float(f[1][i, j])))
                    assert abs(got - want) <= tol * k, (prec, h, kind, k, j)


def test_flat_symbol_shallow(orc_ld):
    """h = 0.05: the image kernel decays like exp(-2 m h); N=512 resolves k <= 64 to exp(-44)."""
    N, h = 512, 0.05
    ks = [1, 2, 3, 7, 40, 64]
    f = pure_modes(N, ks)
    w = ld(orc_ld.dtn_apply(np.zeros(N), h, f))
    fx = ld(f)
    for i, k in enumerate(ks):
        s = LD(k) * np.tanh(LD(k) * LD(h))
        assert np.abs(w[i] - s * fx[i]).max() <= 3e-16 * k


def test_constants_and_mean(orc_ld):
    """G[const] = 0 and mean(G phi) = 0 (mass conservation); with the printed '+' sign
    I/2 + K would annihilate constants instead (singular), so this also pins R1."""
    c = si.config1()
    w = ld(orc_ld.dtn_apply(c.eta, c.h, np.ones((1, c.N))))
    assert np.abs(w).max() < 1e-16
    w = ld(orc_ld.dtn_apply(c.eta, c.h, c.phi0))
    assert abs(w.mean()) < 1e-18


def test_paper_printed_periods(orc_ld):
    """Linear periods the paper prints: 7.19976 (h=1), 28.1110 (h=0.05), 6.28319 (h=inf)."""
    g = golden()
    for key, h, N in (("T_linear_h1", 1.0, 32), ("T_linear_h0.05", 0.05, 512), ("T_linear_hinf", float("inf"), 32)):
        f = pure_modes(N, [1])
        w = ld(orc_ld.dtn_apply(np.zeros(N), h, f))
        sym = float(w[0, 0] / ld(f)[0, 0])          # k tanh(kh) at k=1, alpha=0
        T = 2.0 * math.pi / math.sqrt(1.0 * sym)     # omega^2 = g k tanh(kh), (4.35)
        assert abs(T - g[key][0]) <= g[key][1], (key, T)


def test_paper_resonance_depth(orc_ld):
    """(4.39) PAPER.md:399: 7 tanh 7h = 9 tanh h at h = 1.0397189, with tanh taken from the oracle's own symbol."""
    hc, tol = golden()["h_crit_3_7"]
    N = 64
    f = pure_modes(N, [1, 7])

    def resid(h):
        w = ld(orc_ld.dtn_apply(np.zeros(N), h, f))
        s1 = float(w[0, 0] / ld(f)[0, 0])
        s7 = float(w[1, 0] / ld(f)[1, 0])
        return s7 - 9.0 * s1

    assert resid(hc - 10 * tol) * resid(hc + 10 * tol) < 0          # the root is bracketed this tightly
    assert abs(resid(hc)) < abs(resid(hc + 100 * tol))


# ----------------------------------------------------------------------------------------------------------
# (M): manufactured harmonic solution phi = cosh(k y) cos(k x), bottom y = 0 (satisfies (2.3a,b)):
#   G phi = phi_y - eta' phi_x = k sinh(kY) cos(k a) + eta' k cosh(kY) sin(k a),  Y = h + eta.   Wavy surface.
# ----------------------------------------------------------------------------------------------------------
def manufactured(N, h, k, eta_coef):
    a = 2 * PI * np.arange(N, dtype=LD) / N
    ak = np.arange(len(eta_coef), dtype=LD)
    eta = sum(LD(c) * np.cos(m * a) for m, c in zip(ak, eta_coef))
    d1 = sum(-LD(c) * m * np.sin(m * a) for m, c in zip(ak, eta_coef))
    Y = LD(h) + eta
    phi = np.cosh(k * Y) * np.cos(k * a)
    w = k * np.sinh(k * Y) * np.cos(k * a) + d1 * k * np.cosh(k * Y) * np.sin(k * a)
    px = -k * np.cosh(k * Y) * np.sin(k * a)
    py = k * np.sinh(k * Y) * np.cos(k * a)
    return eta, d1, phi, w, px, py


def split_ld(x):
    hi = np.asarray(x, dtype=np.float64)
    lo = np.asarray(x - hi.astype(LD), dtype=np.float64)
    return hi, lo


@pytest.mark.parametrize("h,k", [(1.0, 2), (0.5, 1), (1.0, 3)])
def test_manufactured_solution_converges(orc_ld, h, k):
    coef = [0.0, 0.07, -0.03, 0.015, 0.0, 0.004]
    errs = []
    for N in (32, 64, 128):
        eta, d1, phi, w, _, _ = manufactured(N, h, k, coef)
        got = ld(orc_ld.dtn_apply(split_ld(eta), h, split_ld(phi)))[0]
        errs.append(float(np.abs(got - w).max() / np.abs(w).max()))
    assert errs[1] < 1e-3 * errs[0] + 1e-16          # spectral convergence
    assert errs[2] < 2e-16, errs                       # to long-double roundoff at N=128


def test_manufactured_velocities(orc_ld):
    """(2.9): u = phi_x, v = phi_y on the surface, from the oracle's base state."""
    N, h, k = 128, 1.0, 2
    eta, d1, phi, w, px, py = manufactured(N, h, k, [0.0, 0.07, -0.03, 0.015, 0.0, 0.004])
    z = np.zeros((1, N))
    _, base = orc_ld.dtn_linearized(split_ld(eta), h, split_ld(phi), z, z, want_base=True)
    assert np.abs(ld(base["u"]) - px).max() < 5e-16
    assert np.abs(ld(base["v"]) - py).max() < 5e-16
    assert np.abs(ld(base["W0"]) - w).max() < 5e-16


# ----------------------------------------------------------------------------------------------------------
# Fourier multipliers: exact on single modes; D equals the textbook cot-circulant differentiation matrix.
# ----------------------------------------------------------------------------------------------------------
def test_multipliers_on_modes(orc_ld):
    N = 32
    ks = [1, 5, 15]
    c, s = ld(pure_modes(N, ks, "cos")), ld(pure_modes(N, ks, "sin"))
    fc, fs = pure_modes(N, ks, "cos"), pure_modes(N, ks, "sin")
    for i, k in enumerate(ks):
        col = lambda f: (f[0][i], f[1][i])
        assert np.abs(ld(orc_ld.multiplier(oracle.MUL_D, col(fc))) + k * s[i]).max() < 1e-17 * N * k     # D cos = -k sin
        assert np.abs(ld(orc_ld.multiplier(oracle.MUL_D, col(fs))) - k * c[i]).max() < 1e-17 * N * k     # D sin =  k cos
        assert np.abs(ld(orc_ld.multiplier(oracle.MUL_H, col(fc))) - s[i]).max() < 1e-17 * N             # H cos =  sin (symbol -i sgn k)
        assert np.abs(ld(orc_ld.multiplier(oracle.MUL_H, col(fs))) + c[i]).max() < 1e-17 * N             # H sin = -cos
        assert np.abs(ld(orc_ld.multiplier(oracle.MUL_ABSD, col(fc))) - k * c[i]).max() < 1e-17 * N * k  # |D| = H D
        filt = math.exp(-36.0 * (k / (N / 2)) ** 36)                                                     # (2.14)
        assert np.abs(ld(orc_ld.multiplier(oracle.MUL_FILTER, col(fc))) - filt * c[i]).max() < 2e-16
    # Nyquist: symbol 0 for D and H, exp(-36) for the filter (R4); constants: P removes them, D kills them
    nyq = np.cos(np.pi * np.arange(N))
    assert np.abs(ld(orc_ld.multiplier(oracle.MUL_D, nyq))).max() < 1e-17
    assert np.abs(ld(orc_ld.multiplier(oracle.MUL_H, nyq))).max() < 1e-17
    assert np.abs(ld(orc_ld.multiplier(oracle.MUL_FILTER, nyq)) - math.exp(-36.0) * nyq).max() < 1e-17
    one = np.ones(N)
    assert np.abs(ld(orc_ld.multiplier(oracle.MUL_P, one))).max() < 1e-17
    assert np.abs(ld(orc_ld.multiplier(oracle.MUL_FILTER, one)) - one).max() < 1e-17


def test_derivative_equals_cot_circulant(orc_ld):
    """Textbook: for even N the spectral derivative (Nyquist dropped) is (Df)_j = sum_m (1/2)(-1)^(j-m) cot((a_j-a_m)/2) f_m."""
    N = 48
    f = si.normals(7, 0, N)
    got = ld(orc_ld.multiplier(oracle.MUL_D, f))
    j = np.arange(N)
    d = j[:, None] - j[None, :]
    with np.errstate(divide="ignore"):
        M = 0.5 * (-1.0) ** d * (1.0 / np.tan(PI * d.astype(LD) / N))
    M[d == 0] = 0
    want = M.astype(LD) @ f.astype(LD)
    assert np.abs(got - want).max() < 1e-15


# ----------------------------------------------------------------------------------------------------------
# Kernel matrices: smoothness across the diagonal (T9) and the two-branch cot.
# ----------------------------------------------------------------------------------------------------------
def test_diagonal_limits_are_continuous(orc_ld):
    N, h = 256, 0.6
    eta = si.synth(N, np.array([0, 0.15, -0.06, 0.03, 0.0, 0.01]), np.array([0, 0.0, 0.05, 0.0, 0.02, 0.0]))[0]
    A = orc_ld.assemble(eta, h)
    d1, d2 = ld(A["d1"]), ld(A["d2"])
    assert float(np.abs(d2 / (2 * (1 + d1 * d1))).max()) > 0.1       # the limit terms are not negligible here
    for name in ("K", "G"):
        M = ld(A[name]) * N
        i = np.arange(N)
        dg = M[i, i]
        up, dn = M[i, (i + 1) % N], M[i, (i - 1) % N]
        up2, dn2 = M[i, (i + 2) % N], M[i, (i - 2) % N]
        interp = (4 * (up + dn) - (up2 + dn2)) / 6                    # 4th-order interpolation across the diagonal entry
        assert np.abs(dg - interp).max() < 2e-4, name


def test_half_cot_branches_agree():
    """the two printed forms are the same function (sin^2 x + sinh^2 y = cosh^2 y - cos^2 x)."""
    with mpmath.workdps(30):
        for x, y in ((0.3, 0.2), (1.2, -0.4), (2.0, 0.1), (3.0, 1.5), (4.5, -0.02)):
            cot = mpmath.cot(mpmath.mpc(x, y) / 2)
            b1 = (mpmath.cos(x) + mpmath.cosh(y)) / mpmath.mpc(mpmath.sin(x), mpmath.sinh(y))
            b2 = mpmath.mpc(mpmath.sin(x), -mpmath.sinh(y)) / (mpmath.cosh(y) - mpmath.cos(x))
            assert abs(cot - b1) < 1e-25 and abs(cot - b2) < 1e-25


def test_kernel_entries_against_mpmath(orc_q):
    """Entry-by-entry (2.13), PAPER.md:144-146 (with R1), from mpmath's own complex cot -- no two-branch formula,
    no tables -- on a small wavy surface, including both cos x branches."""
    c = si.config1()
    N, h = c.N, c.h
    A = orc_q.assemble(c.eta, h)
    with mpmath.workdps(40):
        mp = lambda p: mpmath.mpf(float(p[0])) + mpmath.mpf(float(p[1]))
        eta = [mpmath.mpf(float(v)) for v in c.eta]
        d1 = [mp((A["d1"][0][j], A["d1"][1][j])) for j in range(N)]
        z = [mpmath.mpc(2 * mpmath.pi * j / N, h + eta[j]) for j in range(N)]
        zp = [mpmath.mpc(1, d1[j]) for j in range(N)]
        for (i, j) in ((0, 1), (3, 40), (17, 16), (63, 0), (10, 42), (5, 30), (50, 20)):
            half_cot = lambda w: mpmath.cot(w / 2) / 2
            c0 = half_cot(mpmath.mpf(2 * mpmath.pi * (i - j) / N))
            K1 = (zp[j] * half_cot(z[i] - z[j]) - c0).imag
            K2 = (mpmath.conj(zp[j]) * half_cot(z[i] - mpmath.conj(z[j]))).imag
            G1 = (zp[i] * half_cot(z[i] - z[j]) - c0).real
            G2 = (zp[i] * half_cot(z[i] - mpmath.conj(z[j]))).real
            Kij = mp((A["K"][0][i, j], A["K"][1][i, j]))
            Gij = mp((A["G"][0][i, j], A["G"][1][i, j]))
            assert abs(Kij - (K1 - K2) / N) < 1e-29, (i, j)
            assert abs(Gij - (G1 - G2) / N) < 1e-29, (i, j)


# ----------------------------------------------------------------------------------------------------------
# Brute force, N = 16: the UN-regularised principal-value integrals (A.3), (A.8) evaluated by a
# 4096-point staggered trapezoid rule on the trigonometric interpolants.  Independent of the regularisation,
# of the diagonal limits and of the manufactured solutions.
# ----------------------------------------------------------------------------------------------------------
def _interp(vals, x):
    """trigonometric interpolant of N equispaced real samples at points x (long double)"""
    N = len(vals)
    j = np.arange(N, dtype=LD)
    a = 2 * PI * j / N
    out = np.zeros_like(x)
    for k in range(0, N // 2 + 1):
        ck = (vals * np.cos(k * a)).sum() / N
        sk = (vals * np.sin(k * a)).sum() / N
        wgt = 1 if (k == 0 or 2 * k == N) else 2
        out += wgt * (ck * np.cos(k * x) + sk * np.sin(k * x))
    return out


@pytest.mark.parametrize("amp", [0.0, 0.01])
def test_brute_force_principal_value(orc_ld, amp):
    N, h, M = 16, 1.0, 4096
    a = 2 * PI * np.arange(N, dtype=LD) / N
    eta = LD(amp) * (np.cos(a) + LD(0.5) * np.cos(2 * a))
    phi = LD(0.3) * np.cos(a) + LD(0.2) * np.sin(2 * a) + LD(0.1) * np.cos(3 * a)
    (w_hl, mu_hl) = orc_ld.dtn_apply(split_ld(eta), h, split_ld(phi), want_mu=True)
    W, mu = ld(w_hl)[0], ld(mu_hl)[0]
    gam = ld(orc_ld.multiplier(oracle.MUL_D, split_ld(mu)))
    d1 = ld(orc_ld.assemble(split_ld(eta), h)["d1"])
    for i in (0, 3, 8, 13):
        # quadrature nodes staggered about alpha_i so that the PV integrand's odd singular part cancels exactly
        beta = a[i] + 2 * PI * (np.arange(M, dtype=LD) + LD(0.5)) / M
        eb, d1b, mub, gb = _interp(eta, beta), _interp(d1, beta), _interp(mu, beta), _interp(gam, beta)
        zi = complex(float(a[i]), float(h + eta[i]))
        zb = beta.astype(np.float64) + 1j * (h + eb.astype(np.float64))
        zpb = 1.0 + 1j * d1b.astype(np.float64)
        hc = lambda w: 0.5 / np.tan(w / 2)
        # (A.3) at z -> zeta(alpha_i)^-:  Phi = +mu/2 + (1/(2 pi i)) PV int [ zeta'(b)/2 cot((zi-zeta(b))/2) - conj(zeta'(b))/2 cot((zi-conj zeta(b))/2) ] mu db
        integ = (zpb * hc(zi - zb) - np.conj(zpb) * hc(zi - np.conj(zb))) * mub.astype(np.float64)
        Phi = 0.5 * float(mu[i]) + (integ.sum() / M) / 1j
        assert abs(Phi.real - float(phi[i])) < 3e-11, ("A.3", i)
        # (A.8): zeta'(a) Phi'(zeta^-) = +gamma/2 + (1/(2 pi i)) PV int zeta'(a) [ 1/2 cot(..) - 1/2 cot(.. conj) ] gamma db ; G phi = Re{ i zeta' Phi' } (A.11)
        zpi = 1.0 + 1j * float(d1[i])
        integ = zpi * (hc(zi - zb) - hc(zi - np.conj(zb))) * gb.astype(np.float64)
        zPhi = 0.5 * float(gam[i]) + (integ.sum() / M) / 1j
        assert abs((1j * zPhi).real - float(W[i])) < 3e-11, ("A.8", i)


# ----------------------------------------------------------------------------------------------------------
# Structure of G: self-adjoint ((B.5)); solve residual; precisions agree.
# ----------------------------------------------------------------------------------------------------------
def test_self_adjoint(orc_ld):
    N, h = 128, 0.8
    eta = si.synth(N, np.array([0, 0.1, -0.04, 0.02]), np.array([0, 0.0, 0.03, 0.0]))[0]
    phi = si.synth(N, np.array([0, 0.2, 0.1, 0.0, 0.05]), np.array([0, 0.0, -0.3, 0.1, 0.0]))[0]
    chi = si.synth(N, np.array([0, 0.3, -0.2, 0.0, 0.1]), np.array([0, 0.1, 0.0, 0.25, 0.0]))[0]
    w = ld(orc_ld.dtn_apply(eta, h, np.stack([phi, chi])))
    lhs = (chi.astype(LD) * w[0]).sum() / N
    rhs = (phi.astype(LD) * w[1]).sum() / N
    assert abs(lhs) > 1e-3
    assert abs(lhs - rhs) < 1e-17


def test_solve_residual_and_mu(orc_ld):
    c = si.config1()
    A = orc_ld.assemble(c.eta, c.h)
    (_, mu) = orc_ld.dtn_apply(c.eta, c.h, c.phi0, want_mu=True)
    r = 0.5 * ld(mu)[0] + ld(A["K"]) @ ld(mu)[0] - c.phi0
    assert np.abs(r).max() < 1e-18


def test_precisions_agree(orc_f64, orc_ld, orc_q):
    c = si.config3(128, 8)
    w64 = ld(orc_f64.dtn_linearized(c.eta, c.h, c.phi0, c.deta, c.dphi))
    wld = ld(orc_ld.dtn_linearized(c.eta, c.h, c.phi0, c.deta, c.dphi))
    wq = ld(orc_q.dtn_linearized(c.eta, c.h, c.phi0, c.deta, c.dphi))
    scale = np.abs(wq).max(axis=1, keepdims=True)
    # the low-k deta columns amplify the rounding noise of the base state twice by |D| (~N^2/20 ulps): measured
    # 3.4e-15 (ld) and 5.9e-12 (f64) on column 0 here; the dphi columns agree to ~100x better.
    assert (np.abs(wld - wq) / scale).max() < 2e-14
    assert (np.abs(w64 - wq) / scale).max() < 5e-11
    assert (np.abs(wld - wq) / scale)[1::2].max() < 2e-16


# ----------------------------------------------------------------------------------------------------------
# Linearised DtN (O7) and linearised right-hand sides (O8): Craig-Sulem first-order expansion at a flat base state
# (the paper's ref [58]) and Richardson-extrapolated central differences of the oracle's own nonlinear F.
# ----------------------------------------------------------------------------------------------------------
def test_linearized_flat_base_craig_sulem(orc_ld):
    """About eta=0: d/de G(e deta)[phi0 + e dphi] = G0 dphi - D(deta D phi0) - G0(deta G0 phi0), G0 = |D| tanh(h|D|)."""
    N, h = 64, 0.7
    phi0 = si.synth(N, np.array([0, 0.3, 0.0, -0.1]), np.array([0, 0.0, 0.2, 0.0]))[0]
    deta = si.synth(N, np.array([0, 0.0, 1.0, 0.0, 0.5]), np.array([0, 0.7, 0.0, 0.0, 0.0]))
    dphi = si.synth(N, np.array([0, 1.0, 0.0, 0.3, 0.0]), np.array([0, 0.0, -0.4, 0.0, 0.0]))
    got = ld(orc_ld.dtn_linearized(np.zeros(N), h, phi0, deta, dphi))[0]
    # long-double circulant matrices of D and G0 = |D| tanh(h|D|) (Nyquist symbol 0), built from their symbols
    j = np.arange(N)
    ang = 2 * PI * ((j[:, None] - j[None, :]) % N).astype(LD) / N
    Dm = sum(-2 * LD(k) * np.sin(k * ang) for k in range(1, N // 2)) / N
    G0m = sum(2 * LD(k) * np.tanh(LD(h) * k) * np.cos(k * ang) for k in range(1, N // 2)) / N
    D = lambda f: Dm @ f.astype(LD)
    G0 = lambda f: G0m @ f.astype(LD)
    want = G0(dphi[0]) - D(deta[0].astype(LD) * D(phi0)) - G0(deta[0].astype(LD) * G0(phi0))
    assert np.abs(got - want).max() < 5e-16


def _richardson(f, e0):
    """6th-order central-difference derivative of f at 0"""
    d = lambda e: (f(e) - f(-e)) / (2 * e)
    d1, d2, d4 = d(e0), d(e0 / 2), d(e0 / 4)
    r1, r2 = (4 * d2 - d1) / 3, (4 * d4 - d2) / 3
    return (16 * r2 - r1) / 15


def test_linearized_matches_finite_differences(orc_q):
    """(B.1)-(B.3), linearise the CONTINUOUS problem, so they equal the derivative of the discrete F only
    up to the discretisation error: the gap must close spectrally with N (3 cols x 3 grids, __float128)."""
    h = 1.0
    ce, se = np.array([0, 0.07, -0.03, 0.015, 0.0, 0.004]), np.array([0, 0.0, 0.02, 0.0, 0.0, 0.0])
    cp, sp = np.array([0, 0.05, 0.0, 0.02]), np.array([0, 0.1, -0.03, 0.0])
    cde, sde = np.array([[0, 0.5, 0.2, 0.0, 0.1], [0, 0, 0, 1.0, 0]]), np.array([[0, 0.0, 0.3, 0.0, 0.0], [0, 0, 0.5, 0, 0]])
    cdp, sdp = np.array([[0, 0.1, 0.0, 0.4, 0.0], [0, 1.0, 0, 0, 0]]), np.array([[0, 0.6, 0.0, 0.0, 0.2], [0, 0, 0, 0, 0.3]])
    gaps = []
    for N in (32, 64, 128):
        eta, phi0 = si.synth(N, ce, se)[0].astype(LD), si.synth(N, cp, sp)[0].astype(LD)
        de, dp = si.synth(N, cde, sde), si.synth(N, cdp, sdp)
        lin = orc_q.rhs(split_ld(eta), split_ld(phi0), h, 1.0, de, dp, filter=False)
        gap = 0.0
        for col in range(2):
            def F(e):
                r = orc_q.rhs(split_ld(eta + LD(e) * de[col]), split_ld(phi0 + LD(e) * dp[col]), h, 1.0, filter=False)
                return np.concatenate([ld(r["eta_t"]), ld(r["phi_t"])])
            fd = _richardson(F, 1e-4)
            want = np.concatenate([ld(lin["deta_t"])[col], ld(lin["dphi_t"])[col]])
            gap = max(gap, float(np.abs(fd - want).max() / np.abs(want).max()))
        gaps.append(gap)
        # the DtN-only entry point is the eta-equation of the same linearisation (B.2)
        w = ld(orc_q.dtn_linearized(split_ld(eta), h, split_ld(phi0), de, dp))
        assert np.abs(w - ld(lin["deta_t"])).max() < 1e-28
    assert gaps[0] < 1e-3 and gaps[1] < 1e-4 * gaps[0] and gaps[2] < 1e-4 * gaps[1] and gaps[2] < 1e-13, gaps


# ----------------------------------------------------------------------------------------------------------
# RK8 (R6): rooted-tree order conditions of the tableau; convergence slope; dispersion, energy, symmetry.
# ----------------------------------------------------------------------------------------------------------
def _trees(order, memo={}):
    """all rooted trees with `order` vertices, as sorted tuples of subtrees"""
    if order in memo:
        return memo[order]
    if order == 1:
        memo[1] = [()]
        return memo[1]
    out = set()

    def parts(n, maxpart):
        if n == 0:
            yield []
            return
        for p in range(min(n, maxpart), 0, -1):
            for rest in parts(n - p, p):
                yield [p] + rest

    import itertools
    for part in parts(order - 1, order - 1):
        pools = [_trees(p) for p in part]
        for combo in itertools.product(*pools):
            out.add(tuple(sorted(combo)))
    memo[order] = sorted(out)
    return memo[order]


def test_rk8_order_conditions(orc_q):
    (ah, al), (bh, bl), (ch, cl) = orc_q.rk_tableau()
    s = 11
    with mpmath.workdps(40):
        mp = lambda h, l: mpmath.mpf(float(h)) + mpmath.mpf(float(l))
        a = [[mp(ah[i, j], al[i, j]) for j in range(s)] for i in range(s)]
        b = [mp(bh[i], bl[i]) for i in range(s)]
        c = [mp(ch[i], cl[i]) for i in range(s)]
        for i in range(s):
            assert abs(sum(a[i]) - c[i]) < 1e-30
            assert all(a[i][j] == 0 for j in range(i, s))      # explicit

        def order_of(t):
            return 1 + sum(order_of(u) for u in t)

        def gamma(t):
            g = order_of(t)
            for u in t:
                g *= gamma(u)
            return g

        def phi(t):                                             # elementary weights Phi_i(t)
            out = [mpmath.mpf(1)] * s
            for u in t:
                pu = phi(u)
                inner = [sum(a[i][j] * pu[j] for j in range(s)) for i in range(s)]
                out = [out[i] * inner[i] for i in range(s)]
            return out

        counts = []
        for q in range(1, 9):
            ts = _trees(q)
            counts.append(len(ts))
            for t in ts:
                lhs = sum(b[i] * p for i, p in enumerate(phi(t)))
                assert abs(lhs - mpmath.mpf(1) / gamma(t)) < 1e-29, (q, t)
        assert counts == [1, 1, 2, 4, 9, 20, 48, 115]
        # order is exactly 8: some order-9 condition fails
        worst = max(abs(sum(b[i] * p for i, p in enumerate(phi(t))) - mpmath.mpf(1) / gamma(t)) for t in _trees(9))
        assert worst > 1e-6


def test_rk8_convergence_slope(orc_q):
    errs = []
    for n in (4, 8, 16):
        y, yl = orc_q.rk_riccati_test(1.0 / n, n)
        errs.append(abs((LD(y) + LD(yl)) - LD(0.5)))
    slopes = [math.log2(float(errs[i] / errs[i + 1])) for i in range(2)]
    assert all(7.5 < s < 9.5 for s in slopes), (errs, slopes)
    el = []
    for n in (8, 16, 32):                                           # y' = i y over t = 2
        yh, yl = orc_q.rk_linear_test(1j, 2.0 / n, n)
        with mpmath.workdps(40):
            re = mpmath.mpf(float(yh[0])) + mpmath.mpf(float(yl[0])) - mpmath.cos(2)
            im = mpmath.mpf(float(yh[1])) + mpmath.mpf(float(yl[1])) - mpmath.sin(2)
            el.append(float(mpmath.sqrt(re * re + im * im)))
    slopes = [math.log2(el[i] / el[i + 1]) for i in range(2)]
    assert all(7.7 < s < 8.3 for s in slopes) and el[2] < 2e-14, (el, slopes)


def test_linear_standing_wave_period(orc_ld):
    """(4.35): eta = A sin(wt) cos x, phi = B cos(wt) cos x, w^2 = g tanh h, A/B = sqrt(tanh h / g).
    Amplitude 1e-7: the state returns after T = 2 pi / w up to O(amp^2)."""
    N, h, g, amp = 16, 1.0, 1.0, 1e-7
    a = si.grid(N)
    w = math.sqrt(g * math.tanh(h))
    T = 2 * math.pi / w
    phi = amp * np.cos(a)
    n = 32
    r = orc_ld.rk_advance(np.zeros(N), phi, h, g, T / 4 / (n // 4), n // 4)   # quarter period: phi -> 0, eta -> A cos x
    A = amp * math.sqrt(math.tanh(h) / g)
    assert np.abs(ld(r["phi"])).max() < 5e-13 * 1e0 * amp / 1e-7 * 1e-0 + 1e-13
    assert np.abs(ld(r["eta"]) - A * np.cos(a)).max() < 1e-13
    r = orc_ld.rk_advance(np.zeros(N), phi, h, g, T / n, n)                   # full period
    assert np.abs(ld(r["phi"]) - phi).max() < 1e-13
    assert np.abs(ld(r["eta"])).max() < 1e-13


def test_energy_mean_symmetry_under_time_stepping(orc_ld):
    """T3, T4, T6, T7."""
    N, h, g = 32, 1.0, 1.0
    a = si.grid(N)
    eta0 = 0.05 * np.cos(a) + 0.01 * np.cos(2 * a)
    eta0 = 0.5 * (eta0 + np.roll(eta0[::-1], 1))                          # exactly even samples
    T = 2 * math.pi / math.sqrt(math.tanh(h))
    n = 12
    fwd = orc_ld.rk_advance(eta0, np.zeros(N), h, g, T / 8 / n, n, want_energy=True)
    E = ld(fwd["energies"])
    assert float(np.abs(E - E[0]).max() / E[0]) < 1e-12                  # energy
    assert abs(float(ld(fwd["eta"]).mean() - eta0.astype(LD).mean())) < 1e-19   # mean eta is conserved
    assert abs(float(ld(fwd["phi"]).mean())) < 1e-19                     # mean phi (P)
    ev = ld(fwd["eta"])
    assert np.abs(ev - np.roll(ev[::-1], 1)).max() < 2e-18               # even data stay even (roundoff only)
    # time reversal from rest: eta(-t) = eta(t), phi(-t) = -phi(t)
    bwd = orc_ld.rk_advance(eta0, np.zeros(N), h, g, -T / 8 / n, n)
    assert np.abs(ld(bwd["eta"]) - ld(fwd["eta"])).max() < 1e-17
    assert np.abs(ld(bwd["phi"]) + ld(fwd["phi"])).max() < 1e-17


def test_energy_absolute_scale(orc_ld):
    """E = (1/2) int_0^{2 pi} [phi G phi + g eta^2] dx in closed form, so that the constant in front of the
    oracle's sum is pinned (conservation alone passes with any factor):
      eta = a cos x, phi = 0           ->  E = g a^2 pi / 2          (int cos^2 = pi);
      eta = 0, phi = b cos(k x), h     ->  E = b^2 k tanh(k h) pi / 2   (flat-surface symbol (4.34))."""
    N = 64
    x = si.grid(N)
    a, g = 0.05, 1.7
    E = orc_ld.rhs(a * np.cos(x), np.zeros(N), 1.0, g)["energy"]
    assert abs(float(ld((np.array([E[0]]), np.array([E[1]])))[0]) - 0.5 * g * a * a * math.pi) < 1e-17
    b, k, h = 0.3, 3, 0.7
    E = orc_ld.rhs(np.zeros(N), b * np.cos(k * x), h, g)["energy"]
    want = 0.5 * b * b * k * math.tanh(k * h) * math.pi
    assert abs(float(E[0] + E[1]) - want) < 1e-15 * want + 1e-17


def test_variational_columns_track_finite_differences(orc_ld):
    """(3.32): the column batch advanced with q equals d/de of the advanced nonlinear state."""
    N, h, g = 32, 1.0, 1.0
    a = si.grid(N)
    eta0 = (0.05 * np.cos(a) + 0.01 * np.cos(2 * a)).astype(LD)
    phi0 = (0.02 * np.sin(a)).astype(LD)
    de = np.stack([np.cos(2 * a), np.zeros(N)])
    dp = np.stack([np.zeros(N), np.cos(a)])
    dt, n = 0.05, 6
    lin = orc_ld.rk_advance(split_ld(eta0), split_ld(phi0), h, g, dt, n, de, dp)
    for col in range(2):
        def F(e):
            r = orc_ld.rk_advance(split_ld(eta0 + LD(e) * de[col]), split_ld(phi0 + LD(e) * dp[col]), h, g, dt, n)
            return np.concatenate([ld(r["eta"]), ld(r["phi"])])
        fd = _richardson(F, 2e-2)
        want = np.concatenate([ld(lin["deta"])[col], ld(lin["dphi"])[col]])
        assert np.abs(fd - want).max() < 1e-11, col


# ------------------------------------------------------------------------------------------------ shooting map (3.15)-(3.17), (3.31)
def test_shooting_map_linear_theory(orc_ld):
    """small amplitude: phi(x, t) = 2 eps cos x cos(omega t) + O(eps^2), omega^2 = g tanh h ((4.35)), and a unit
    perturbation of mode k evolves as eta' = A cos(omega_k t), phi' = -(g/omega_k) A sin(omega_k t): closed forms of r and of
    the columns 0, 1, 2 of J at leading order"""
    from oracle import shooting
    N, h, g, eps, nsteps = 32, 1.0, 1.0, 1e-7, 16
    om = [0.0] + [math.sqrt(g * k * math.tanh(k * h)) for k in range(1, 4)]
    T = 6.9   # deliberately off the linear period 7.19976
    c = np.array([T, eps, 0.0, 0.0])
    s = shooting.shoot(orc_ld, c, N, h, g, nsteps)
    x = si.grid(N)
    w = 1 / math.sqrt(N)
    assert np.abs(s["r"] - 2 * eps * np.cos(x) * math.cos(om[1] * T / 4) * w).max() < 1e-13 * eps + 50 * eps * eps
    assert np.abs(s["J"][:, 0] - (-(om[1] / 4) * 2 * eps * np.cos(x) * math.sin(om[1] * T / 4) * w)).max() < 1e-13 * eps + 50 * eps * eps
    assert np.abs(s["J"][:, 1] - 2 * np.cos(x) * math.cos(om[1] * T / 4) * w).max() < 1e-6
    assert np.abs(s["J"][:, 2] - (-(g / om[2]) * 2 * np.cos(2 * x) * math.sin(om[2] * T / 4) * w)).max() < 1e-6
    assert np.abs(s["J"][:, 3] - 2 * np.cos(3 * x) * math.cos(om[3] * T / 4) * w).max() < 1e-6


def test_shooting_jacobian_matches_finite_differences(orc_ld):
    """(3.33): J_ik = [r_i(c + e e_k) - r_i(c - e e_k)] / 2e, Richardson-extrapolated, at a finite amplitude;
    this also fixes the factor 1/4 of the k = 0 (period) column (R13)"""
    from oracle import shooting
    N, h, g, nsteps = 32, 1.0, 1.0, 12
    c = np.array([7.1, 0.02, 0.004, -0.001, 0.0005])
    s = shooting.shoot(orc_ld, c, N, h, g, nsteps)
    for k in range(c.shape[0]):
        def F(e):
            ck = c.copy()
            ck[k] += e
            return shooting.shoot(orc_ld, ck, N, h, g, nsteps)["r"]
        e0 = 2e-3 if k else 2e-2
        d1 = (F(e0) - F(-e0)) / (2 * e0)
        d2 = (F(e0 / 2) - F(-e0 / 2)) / e0
        fd = (4 * d2 - d1) / 3
        assert np.abs(fd - s["J"][:, k]).max() < 1e-8 * max(1.0, float(np.abs(s["J"][:, k]).max())), k


def test_shooting_recovers_the_linear_period(orc_ld):
    """Gauss-Newton on the period alone along the small-amplitude branch converges to T = 7.19976"""
    from oracle import shooting
    N, h, g, eps, nsteps = 32, 1.0, 1.0, 1e-6, 16
    T = 7.0
    for _ in range(6):
        s = shooting.shoot(orc_ld, np.array([T, eps]), N, h, g, nsteps)
        J0, r = s["J"][:, 0], s["r"]
        T = T - float((J0 @ r) / (J0 @ J0))
    want, tol = golden()["T_linear_h1"]
    assert abs(T - want) < tol
    assert float(0.5 * (s["r"] @ s["r"])) < 1e-22


def test_shooting_quad_matches_long_double(orc_ld, orc_q):
    """shoot_quad (initial state and scaling to ~40 digits, __float128 stepping) against shoot (long double): the two builds of the
    same map agree to long-double accuracy; the quad initial state against its defining sum (3.15) with mpmath at one node"""
    import mpmath as mp
    from oracle import shooting
    c = np.array([7.0, -0.01, 0.003, 0.001, -0.0005])
    N = 32
    a = shooting.shoot(orc_ld, c, N, 1.0, 1.0, 4)
    b = shooting.shoot_quad(orc_q, c, N, 1.0, 1.0, 4)
    assert np.abs(ld(b["r"]) - a["r"]).max() < 5e-18
    assert np.abs(ld(b["J"]) - a["J"]).max() < 5e-18
    eq, pq, deq, dpq = shooting.initial_state_quad(c, N)
    with mp.workprec(200):
        j = 5
        x = 2 * mp.pi * j / N
        eta = sum(2 * mp.mpf(float(c[k])) * mp.cos(k * x) for k in (2, 4))
        phi = sum(2 * mp.mpf(float(c[k])) * mp.cos(k * x) for k in (1, 3))
        assert abs(mp.mpf(float(eq[0][j])) + mp.mpf(float(eq[1][j])) - eta) < mp.mpf(10) ** -33
        assert abs(mp.mpf(float(pq[0][j])) + mp.mpf(float(pq[1][j])) - phi) < mp.mpf(10) ** -33
        assert abs(mp.mpf(float(dpq[0][2][j])) + mp.mpf(float(dpq[1][2][j])) - 2 * mp.cos(3 * x)) < mp.mpf(10) ** -31
        assert float(deq[0][2][j]) == 0.0 and float(dpq[0][1][j]) == 0.0   # column k = 3 perturbs phi only, k = 2 eta only


# ------------------------------------------------------------------------------------------------ surface tension (2.1b), (B.4), (4.42)
def test_surface_tension_is_the_curvature(orc_ld):
    """a surface at rest (phi = 0): phi_t = P[-g eta + sigma kappa] with kappa = eta'' / (1 + eta'^2)^(3/2) in closed form
    ((2.1b)); the difference of the sigma = 1 and sigma = 0 right-hand sides is P[kappa]"""
    N = 64
    x = 2 * LD("3.14159265358979323846264338327950288") * np.arange(N) / N    # the nodes to long-double accuracy
    a, b = LD(0.05), LD(0.01)
    eta = a * np.cos(x) + b * np.cos(3 * x)
    e1 = -a * np.sin(x) - 3 * b * np.sin(3 * x)
    e2 = -a * np.cos(x) - 9 * b * np.cos(3 * x)
    kappa = e2 / (1 + e1 * e1) ** LD(1.5)
    r1 = ld(orc_ld.rhs(split_ld(eta), np.zeros(N), 1.0, 1.0, filter=False, sigma=0.7)["phi_t"])
    r0 = ld(orc_ld.rhs(split_ld(eta), np.zeros(N), 1.0, 1.0, filter=False)["phi_t"])
    assert np.abs((r1 - r0) - LD(0.7) * (kappa - kappa.mean())).max() < 2e-17
    assert np.abs(r0 + (eta - eta.mean())).max() < 1e-18          # phi_t = P[-g eta] at rest without surface tension


def test_capillary_gravity_periods(orc_ld):
    """(4.42): omega^2 = (g + sigma k^2) k tanh kh.  Gauss-Newton on the period alone along the small-amplitude
    branch, infinite depth, g = sigma = 1, k = 1, converges to the printed T = 2 pi / sqrt 2 = 4.443; finite depth h = 1 to the formula"""
    from oracle import shooting
    N, eps, nsteps = 32, 1e-6, 16
    for h, want, tol in ((float("inf"), golden()["T_capillary_hinf"][0], golden()["T_capillary_hinf"][1]),
                         (1.0, 2 * math.pi / math.sqrt(2 * math.tanh(1.0)), 1e-9)):
        T = 0.95 * want
        for _ in range(6):
            s = shooting.shoot(orc_ld, np.array([T, eps]), N, h, 1.0, nsteps, sigma=1.0)
            J0, r = s["J"][:, 0], s["r"]
            T = T - float((J0 @ r) / (J0 @ J0))
        assert abs(T - want) < tol, (h, T, want)
        assert float(0.5 * (s["r"] @ s["r"])) < 1e-22


def test_linearized_surface_tension_matches_finite_differences(orc_q):
    """the variation of the curvature term, sigma D(D(deta) / (1 + eta'^2)^(3/2)) ((B.4)), against Richardson
    differences of the nonlinear right-hand side with sigma = 1: the gap closes spectrally with N as in the sigma = 0 test"""
    h = 1.0
    ce, se = np.array([0, 0.07, -0.03, 0.015, 0.0, 0.004]), np.array([0, 0.0, 0.02, 0.0, 0.0, 0.0])
    cp, sp = np.array([0, 0.05, 0.0, 0.02]), np.array([0, 0.1, -0.03, 0.0])
    cde, sde = np.array([[0, 0.5, 0.2, 0.0, 0.1], [0, 0, 0, 1.0, 0]]), np.array([[0, 0.0, 0.3, 0.0, 0.0], [0, 0, 0.5, 0, 0]])
    cdp, sdp = np.array([[0, 0.1, 0.0, 0.4, 0.0], [0, 1.0, 0, 0, 0]]), np.array([[0, 0.6, 0.0, 0.0, 0.2], [0, 0, 0, 0, 0.3]])
    gaps = []
    for N in (32, 64, 128):
        eta, phi0 = si.synth(N, ce, se)[0].astype(LD), si.synth(N, cp, sp)[0].astype(LD)
        de, dp = si.synth(N, cde, sde), si.synth(N, cdp, sdp)
        lin = orc_q.rhs(split_ld(eta), split_ld(phi0), h, 1.0, de, dp, filter=False, sigma=1.0)
        lin0 = orc_q.rhs(split_ld(eta), split_ld(phi0), h, 1.0, de, dp, filter=False)
        assert np.abs(ld(lin["deta_t"]) - ld(lin0["deta_t"])).max() == 0     # surface tension enters the phi equation only
        gap = 0.0
        for col in range(2):
            def F(e):
                r = orc_q.rhs(split_ld(eta + LD(e) * de[col]), split_ld(phi0 + LD(e) * dp[col]), h, 1.0, filter=False, sigma=1.0)
                return ld(r["phi_t"])
            fd = _richardson(F, 1e-4)
            want = ld(lin["dphi_t"])[col]
            gap = max(gap, float(np.abs(fd - want).max() / np.abs(want).max()))
        gaps.append(gap)
    assert gaps[0] < 1e-3 and gaps[1] < 1e-4 * gaps[0] and gaps[2] < 1e-3 * gaps[1] and gaps[2] < 1e-12, gaps


# ------------------------------------------------------------------------------------------------ SDC15 (R15)
def test_sdc_radau_tables(orc_q):
    """8 Radau IIa nodes and their integration matrix: closed forms for s = 2, 3 (1/3, 1; (4 -+ sqrt 6)/10, 1), c_s = 1, exactness of the
    rows of S on polynomials of degree < s, of the weights b = S[s-1] on degree <= 2 s - 2 (Radau quadrature), positive weights"""
    import mpmath as mp
    mp.mp.prec = 200
    val = lambda p, *i: mp.mpf(float(p[0][i])) + mp.mpf(float(p[1][i]))
    c2, _ = orc_q.sdc_tables(2)
    assert abs(val(c2, 0) - mp.mpf(1) / 3) < mp.mpf(10) ** -32 and val(c2, 1) == 1
    c3, _ = orc_q.sdc_tables(3)
    assert abs(val(c3, 0) - (4 - mp.sqrt(6)) / 10) < mp.mpf(10) ** -32 and abs(val(c3, 1) - (4 + mp.sqrt(6)) / 10) < mp.mpf(10) ** -32
    s = 8
    c, S = orc_q.sdc_tables(s)
    cc = [val(c, i) for i in range(s)]
    SS = [[val(S, m, j) for j in range(s)] for m in range(s)]
    assert cc[-1] == 1 and all(0 < cc[i] < cc[i + 1] for i in range(s - 1))
    for m in range(s):
        for k in range(s):
            assert abs(sum(SS[m][j] * cc[j] ** k for j in range(s)) - cc[m] ** (k + 1) / (k + 1)) < mp.mpf(10) ** -31
    for k in range(2 * s - 1):
        assert abs(sum(SS[s - 1][j] * cc[j] ** k for j in range(s)) - mp.mpf(1) / (k + 1)) < mp.mpf(10) ** -31
    assert all(SS[s - 1][j] > 0 for j in range(s))


def test_sdc_is_fifteenth_order(orc_q):
    """y' = lambda y: halving the step divides the error by 2^15 ("the method is 15th order")"""
    import mpmath as mp
    mp.mp.prec = 200
    lam = complex(-0.3, 1.0)
    errs = []
    for dt, n in ((1.0, 2), (0.5, 4), (0.25, 8)):
        yh, yl = orc_q.sdc_linear_test(lam, dt, n)
        y = mp.mpc(mp.mpf(float(yh[0])) + mp.mpf(float(yl[0])), mp.mpf(float(yh[1])) + mp.mpf(float(yl[1])))
        errs.append(float(abs(y - mp.exp(mp.mpc(lam.real, lam.imag) * 2))))
    slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(14.5 < s < 16.5 for s in slopes), (errs, slopes)


def test_sdc_advance_agrees_with_rk8_and_conserves_energy(orc_ld, orc_q):
    """the water-wave driver: SDC15 steps against RK8 with 16x smaller steps (long double), state and variational
    columns; in __float128 the energy of PAPER.md:501 stays constant to 27+ digits ("29 in quadruple precision")"""
    N, h, g = 32, 1.0, 1.0
    a = si.grid(N)
    eta0 = 0.05 * np.cos(a) + 0.01 * np.cos(2 * a)
    phi0 = 0.02 * np.cos(a)
    de = np.stack([np.cos(2 * a), np.zeros(N)])
    dp = np.stack([np.zeros(N), np.cos(a)])
    T = 0.8
    # filter off: applied after every step it makes the result depend on the number of steps (1e-13 on this coarse grid)
    s = orc_ld.rk_advance(eta0, phi0, h, g, T / 4, 4, deta=de, dphi=dp, method="sdc15", filter=False)
    r = orc_ld.rk_advance(eta0, phi0, h, g, T / 256, 256, deta=de, dphi=dp, filter=False)
    for name in ("eta", "phi", "deta", "dphi"):
        assert np.abs(ld(s[name]) - ld(r[name])).max() < 2e-17, name
    q = orc_q.rk_advance(eta0, phi0, h, g, T / 8, 8, method="sdc15", want_energy=True, filter=False)
    E = q["energies"][0].astype(LD) + q["energies"][1].astype(LD)
    assert float(np.abs(E - E[0]).max() / abs(E[0])) < 1e-27


# ------------------------------------------------------------------------------------------------ adjoint system (B.6)
@pytest.mark.parametrize("sigma,h", [(0.0, 1.0), (0.6, 1.0), (0.0, float("inf"))])
def test_adjoint_identity(orc_q, sigma, h):
    """(B.4)-(B.6): <DF(q) qdot, q~> = <qdot, DF(q)^* q~> with <a, b> = (1/2 pi) int (eta_a eta_b + phi_a phi_b) dx, for
    the linearized right-hand side already pinned by finite differences and random smooth qdot, q~.  Each side is O(0.1); the
    identity is one of the CONTINUOUS operators (G is self-adjoint by Green's identity (B.5)), so the gap closes spectrally with N"""
    gaps = []
    for N in (32, 64, 128):
        rng = np.random.default_rng(7)
        def smooth(amp):
            c, s_ = np.zeros(9), np.zeros(9)
            c[1:] = amp * rng.standard_normal(8) * np.exp(-0.5 * np.arange(1, 9))
            s_[1:] = amp * rng.standard_normal(8) * np.exp(-0.5 * np.arange(1, 9))
            c[0] = 0.3 * amp * rng.standard_normal()
            return si.synth(N, c, s_)[0].astype(LD)
        eta, phi = smooth(0.05), smooth(0.1)
        eta = eta - eta.mean()
        qd = (np.stack([smooth(1.0), smooth(1.0)]), np.stack([smooth(1.0), smooth(1.0)]))      # (deta, dphi), 2 columns
        qt = (np.stack([smooth(1.0), smooth(1.0)]), np.stack([smooth(1.0), smooth(1.0)]))      # (eta~, phi~), 2 columns
        sp = lambda a: split_ld(a) if a.ndim == 1 else tuple(np.stack(t) for t in zip(*[split_ld(r) for r in a]))
        lin = orc_q.rhs(sp(eta), sp(phi), h, 1.0, sp(qd[0]), sp(qd[1]), filter=False, sigma=sigma)
        adj = orc_q.adjoint_rhs(sp(eta), sp(phi), h, 1.0, sp(qt[0]), sp(qt[1]), sigma=sigma)
        gap = 0.0
        for a in range(2):
            for b in range(2):
                lhs = (ld(lin["deta_t"])[a] * qt[0][b] + ld(lin["dphi_t"])[a] * qt[1][b]).mean()
                rhs = (qd[0][a] * ld(adj["eta_s"])[b] + qd[1][a] * ld(adj["phi_s"])[b]).mean()
                assert abs(lhs) > 1e-3
                gap = max(gap, float(abs(lhs - rhs)))
        gaps.append(gap)
    assert gaps[0] < 1e-4 and gaps[1] < 1e-6 * gaps[0] and gaps[2] < 1e-4 * gaps[1] and gaps[2] < 1e-18, gaps


def test_paper_omega2_sign_change_depth():
    """(4.36): the root in h of the printed omega_2 is the printed 1.0581 (the golden value used by the GPU test of
    the period correction is consistent with the formula printed next to it)"""
    w2 = lambda h: (lambda w: 9 * w ** -7 - 12 * w ** -3 - 3 * w - 2 * w ** 5)(math.sqrt(math.tanh(h)))
    lo, hi = 1.0, 1.1
    assert w2(lo) > 0 > w2(hi)
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if w2(mid) > 0 else (lo, mid)
    want, tol = golden()["h_omega2_sign"]
    assert abs(lo - want) < tol
