"""GPU parity tests of mesh refinement in space ((2.10)-(2.11); mesh.cu) against the oracle: kernel matrices, DtN and
linearized DtN in both precisions, the time stepper and the respacing between segments; plus a closed-form harmonic function
through the device path alone.  The stored samples are the same seeded arrays as elsewhere (any smooth periodic function of
alpha is a smooth function of x).  Tolerances: the bars of parity_util divided by rho^2 -- the kernels next to the diagonal are
differences of O(1/spacing^2) terms, and the spacing at the refined end is ~rho times the uniform one."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import sww_inputs as si
from parity_util import ld, diff, to_dev

pytestmark = pytest.mark.gpu
LD = np.longdouble


@pytest.fixture(scope="module")
def sww():
    import paper_1210_5672_b200 as pkg
    assert pkg.lib_path().exists() and torch.cuda.is_available()
    return pkg


@pytest.fixture()
def mesh_ld(orc_ld):
    yield orc_ld
    orc_ld.set_mesh()


@pytest.fixture()
def mesh_q(orc_q):
    yield orc_q
    orc_q.set_mesh()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def surface(N, amp=0.2):
    a, _ = si._family_surface(si.SEED_BASE + 3, N, amp, kmax=min(64, N // 4))
    return si.synth(N, a)[0]


def small_case(N, nc):
    c2 = si.config2()
    eta = np.ascontiguousarray(c2.eta[:: c2.N // N]) if N <= c2.N else surface(N, 0.1)
    a = np.zeros(9); a[1] = 0.05; a[2] = 0.02; a[3] = -0.01
    b = np.zeros(9); b[2] = 0.01
    phi = si.synth(N, a, b)[0]
    deta, dphi = si.fourier_unit_columns(N, nc // 2, "eta_phi")
    return eta, phi, deta, dphi


@pytest.mark.parametrize("N,h,rho,where", [(64, 1.0, 0.5, 0), (256, 1.0, 0.3, 1), (256, 0.05, 0.4, 0), (128, float("inf"), 0.2, 0)])
def test_kernel_matrices_on_refined_mesh(sww, mesh_ld, N, h, rho, where):
    eta = surface(N, 0.2 if h > 0.1 else 0.01)
    d = sww.DtN(dev(eta), h)
    d.set_mesh(rho, where)
    d.refactor(dev(eta))
    d.check()
    mesh_ld.set_mesh(rho, where)
    o = mesh_ld.assemble(eta, h)
    for name in ("K", "G"):
        g = d.get(name).cpu().numpy().T
        ref = ld(o[name])
        scale = float(np.abs(ref).max())
        err = float(np.abs(g - ref).max())
        assert err <= 3e-14 / rho ** 2 * max(scale, 1.0 / N), (name, err, scale)
    x = sww.mesh_points(N, rho, where)
    xp, _, _ = mesh_ld.mesh_tables(N)
    assert np.abs(x - (2 * np.pi * np.arange(N) / N + xp[0])).max() < 1e-15


def test_kernel_matrices_on_refined_mesh_dd(sww, mesh_q):
    N, rho = 128, 0.35
    c = si.config4(N, 2)
    d = sww.DtN(to_dev(c.eta, c.eta_lo, "dd"), c.h, sww.DD)
    d.set_mesh(rho, 1)
    d.refactor(to_dev(c.eta, c.eta_lo, "dd"))
    d.check()
    mesh_q.set_mesh(rho, 1)
    o = mesh_q.assemble((c.eta, c.eta_lo), c.h)
    for name in ("K", "G"):
        t = d.get(name).cpu().numpy()
        err = float(np.abs(diff((t[0].T, t[1].T), o[name])).max())
        assert err <= 1e-29 * N / rho ** 2, (name, err)


@pytest.mark.parametrize("N,h,rho,where", [(256, 1.0, 0.4, 0), (128, float("inf"), 0.25, 1), (1024, 1.0, 0.5, 0)])
def test_apply_and_linearized_on_refined_mesh(sww, mesh_ld, N, h, rho, where):
    eta, phi, deta, dphi = small_case(N, 12)
    d = sww.DtN(dev(eta), h)
    d.set_mesh(rho, where)
    d.refactor(dev(eta))
    w = d.apply(dev(np.stack([phi, deta[0]])))
    d.set_base(dev(phi))
    lin = d.linearized_apply(dev(deta), dev(dphi))
    d.check()
    mesh_ld.set_mesh(rho, where)
    ow = ld(mesh_ld.dtn_apply(eta, h, np.stack([phi, deta[0]])))
    ol, base = mesh_ld.dtn_linearized(eta, h, phi, deta, dphi, want_base=True)
    tol = 1e-11 / rho ** 2
    err = np.abs(w.cpu().numpy().astype(LD) - ow).max(axis=1) / np.abs(ow).max(axis=1)
    assert float(err.max()) <= tol, err
    ol = ld(ol)
    err = np.abs(lin.cpu().numpy().astype(LD) - ol).max(axis=1) / np.abs(ol).max(axis=1)
    assert float(err.max()) <= tol, err
    for name in ("dphi0", "W0", "u", "v"):
        g = d.get(name).cpu().numpy().astype(LD)
        ref = ld(base[name])
        assert float(np.abs(g - ref).max()) <= 1e-13 / rho ** 2 * max(1.0, float(np.abs(ref).max())), name


def test_apply_and_linearized_on_refined_mesh_dd(sww, mesh_q):
    N, rho, where = 128, 0.4, 0
    c = si.config4(N, 8)
    d = sww.DtN(to_dev(c.eta, c.eta_lo, "dd"), c.h, sww.DD)
    d.set_mesh(rho, where)
    d.refactor(to_dev(c.eta, c.eta_lo, "dd"))
    w = d.apply(to_dev(c.dphi, c.dphi_lo, "dd"))
    d.set_base(to_dev(c.phi0, c.phi0_lo, "dd"))
    lin = d.linearized_apply(to_dev(c.deta, c.deta_lo, "dd"), to_dev(c.dphi, c.dphi_lo, "dd"))
    d.check()
    mesh_q.set_mesh(rho, where)
    ow = mesh_q.dtn_apply((c.eta, c.eta_lo), c.h, (c.dphi, c.dphi_lo))
    ol = mesh_q.dtn_linearized((c.eta, c.eta_lo), c.h, (c.phi0, c.phi0_lo), (c.deta, c.deta_lo), (c.dphi, c.dphi_lo))
    for got, ref in ((w, ow), (lin, ol)):
        g = got.cpu().numpy()
        e = np.abs(diff((g[0], g[1]), ref)).max(axis=1) / np.abs(ld(ref)).max(axis=1)
        assert float(e.max()) <= 1e-25 / rho ** 2, e


@pytest.mark.parametrize("rho,where,h", [(0.4, 0, 1.0), (0.3, 1, 0.5)])
def test_harmonic_function_closed_form(sww, rho, where, h):
    """phi = cosh(2 y) cos(2 x) on a wavy surface sampled at the refined points: G phi, phi_x, phi_y in closed form (no oracle)"""
    N = 256
    x = sww.mesh_points(N, rho, where).astype(LD)
    coef = [0.0, 0.07, -0.03, 0.015, 0.0, 0.004]
    eta = sum(LD(c) * np.cos(m * x) for m, c in enumerate(coef))
    ex = sum(-LD(c) * m * np.sin(m * x) for m, c in enumerate(coef))
    Y = LD(h) + eta
    phi = np.cosh(2 * Y) * np.cos(2 * x)
    px, py = -2 * np.cosh(2 * Y) * np.sin(2 * x), 2 * np.sinh(2 * Y) * np.cos(2 * x)
    w = py - ex * px
    e64, p64 = np.asarray(eta, dtype=np.float64), np.asarray(phi, dtype=np.float64)
    d = sww.DtN(dev(e64), h)
    d.set_mesh(rho, where)
    d.refactor(dev(e64))
    got = d.apply(dev(p64)).cpu().numpy()
    d.set_base(dev(p64))
    d.check()
    # the fp64 rounding of the inputs moves the answer by ~eps N / rho (a first-order operator on rounded samples)
    tol = 4 * N * 2.0 ** -53 / rho * float(np.abs(w).max()) + 1e-13 / rho ** 2
    assert float(np.abs(got - w).max()) <= tol
    assert float(np.abs(d.get("u").cpu().numpy() - px).max()) <= tol
    assert float(np.abs(d.get("v").cpu().numpy() - py).max()) <= tol


@pytest.mark.parametrize("N,nc,h,rho,where,sigma", [(64, 6, 1.0, 0.5, 0, 0.0), (256, 6, 1.0, 0.4, 1, 0.0), (128, 8, float("inf"), 0.5, 0, 0.6),
                                                     (2048, 0, 1.0, 0.5, 0, 0.0)])
def test_steps_on_refined_mesh(sww, mesh_ld, N, nc, h, rho, where, sigma):
    eta, phi, deta, dphi = small_case(N, max(nc, 2))
    dt = 0.02 if sigma == 0.0 else 0.4 / N * rho
    nsteps = 2 if N <= 256 else 1
    kw = dict(deta=dev(deta), dphi=dev(dphi)) if nc else {}
    st = sww.State(dev(eta), dev(phi), h, 1.0, **kw)
    st.set_mesh(rho, where)
    st.set_sigma(sigma)
    e0 = st.energy()[0]
    st.advance(dt, nsteps)
    r = st.read()
    mesh_ld.set_mesh(rho, where)
    o = mesh_ld.rk_advance(eta, phi, h, 1.0, dt, nsteps, deta=deta if nc else None, dphi=dphi if nc else None, sigma=sigma, want_energy=True)
    tol = 1e-11 / rho ** 2
    for name in ("eta", "phi"):
        ref = ld(o[name])
        assert float(np.abs(r[name].cpu().numpy().astype(LD) - ref).max() / np.abs(ref).max()) <= tol, name
    if nc:
        for name in ("deta", "dphi"):
            gq, oq = r[name].cpu().numpy(), ld(o[name])
            err = np.abs(gq.astype(LD) - oq).max(axis=1) / np.abs(oq).max(axis=1)
            assert float(err.max()) <= tol, (name, err)
    if sigma == 0.0:
        assert abs(e0 - float(ld(o["energies"])[0])) <= 1e-12 * abs(e0)


def test_segments_with_respacing(sww, mesh_ld):
    """two segments as in section 2.2: uniform mesh, then a finer refined one; against the oracle's chain of the same steps"""
    N, M2, nc, h, dt, rho = 128, 256, 4, 1.0, 0.02, 0.4
    eta, phi, deta, dphi = small_case(N, nc)
    s1 = sww.State(dev(eta), dev(phi), h, 1.0, deta=dev(deta), dphi=dev(dphi))
    s1.advance(dt, 2)
    z1, zc = torch.zeros(M2, dtype=torch.float64, device="cuda"), torch.zeros(nc, M2, dtype=torch.float64, device="cuda")
    s2 = sww.State(z1, z1, h, 1.0, deta=zc, dphi=zc)
    s2.set_mesh(rho, 0)
    s2.respace_from(s1)
    mid = s2.read()
    s2.advance(dt / 2, 2)
    r = s2.read()
    assert abs(r["t"] - 3 * dt) < 1e-15
    mesh_ld.set_mesh()
    o1 = mesh_ld.rk_advance(eta, phi, h, 1.0, dt, 2, deta=deta, dphi=dphi)
    om = {k: mesh_ld.respace(o1[k], (N, 1.0, 0), (M2, rho, 0)) for k in ("eta", "phi", "deta", "dphi")}
    mesh_ld.set_mesh(rho, 0)
    o2 = mesh_ld.rk_advance(om["eta"], om["phi"], h, 1.0, dt / 2, 2, deta=om["deta"], dphi=om["dphi"])
    for got, ref, tol in ((mid, om, 2e-13), (r, o2, 1e-11 / rho ** 2)):
        for name in ("eta", "phi", "deta", "dphi"):
            g, q = got[name].cpu().numpy().astype(LD), ld(ref[name])
            g, q = g.reshape(-1, M2), q.reshape(-1, M2)
            err = np.abs(g - q).max(axis=1) / np.abs(q).max(axis=1)
            assert float(err.max()) <= tol, (name, err)


def test_respacing_between_arbitrary_meshes(sww, mesh_ld):
    """refined -> refined with another rho, the other end and a smaller size; and onto the same mesh (the identity)"""
    N, h = 256, 1.0
    eta, phi, _, _ = small_case(N, 2)
    s1 = sww.State(dev(eta), dev(phi), h, 1.0)
    s1.set_mesh(0.5, 1)
    for M2, rho2, w2 in ((128, 0.7, 0), (256, 0.5, 1), (512, 1.0, 0)):
        z = torch.zeros(M2, dtype=torch.float64, device="cuda")
        s2 = sww.State(z, z, h, 1.0)
        s2.set_mesh(rho2, w2)
        s2.respace_from(s1)
        r = s2.read()
        for name, src in (("eta", eta), ("phi", phi)):
            ref = ld(mesh_ld.respace(src, (N, 0.5, 1), (M2, rho2, w2)))
            assert float(np.abs(r[name].cpu().numpy().astype(LD) - ref).max()) <= 3e-14 * float(np.abs(ref).max()), (M2, name)
        if (M2, rho2, w2) == (256, 0.5, 1):
            assert float(np.abs(r["eta"].cpu().numpy() - eta).max()) <= 1e-15


def test_uniform_mesh_is_untouched_and_errors(sww):
    N, h = 128, 1.0
    eta, phi, deta, dphi = small_case(N, 4)
    d0 = sww.DtN(dev(eta), h)
    ref = d0.apply(dev(phi)).clone()
    d = sww.DtN(dev(eta), h)
    d.set_mesh(0.5, 0)
    d.refactor(dev(eta))
    moved = d.apply(dev(phi)).clone()
    assert float((moved - ref).abs().max()) > 1e-3
    d.set_mesh(1.0, 0)
    d.refactor(dev(eta))
    assert torch.equal(d.apply(dev(phi)), ref)            # rho = 1 is the uniform path, bit for bit
    for bad in ((0.0, 0), (1.5, 0), (0.5, 2), (float("nan"), 0)):
        with pytest.raises(sww.SwwError):
            d.set_mesh(*bad)
    sdd = sww.State(to_dev(eta, None, "dd"), to_dev(phi, None, "dd"), h, 1.0, prec=sww.DD)
    s64 = sww.State(dev(eta), dev(phi), h, 1.0)
    with pytest.raises(sww.SwwError):
        s64.respace_from(sdd)                              # the two states must have the same precision and column count


def dd_err(got, ref):
    """per row: max |got - ref| / max |ref| for a (2, ..., N) double-double tensor against an oracle (hi, lo) pair"""
    g = got.cpu().numpy()
    d = np.abs(diff((g[0], g[1]), ref))
    r = np.abs(ld(ref))
    if d.ndim == 1:
        return float(d.max() / r.max())
    return float((d.max(axis=1) / r.max(axis=1)).max())


@pytest.mark.parametrize("N,nc,h,rho,where,sigma,method", [(64, 4, 1.0, 0.5, 0, 0.0, "rk8"), (128, 2, float("inf"), 0.4, 1, 0.5, "rk8"),
                                                            (64, 2, 1.0, 0.5, 1, 0.0, "sdc15")])
def test_steps_on_refined_mesh_dd(sww, mesh_q, N, nc, h, rho, where, sigma, method):
    """the paper's quadruple-precision configuration: a refined mesh under the double-double stepper (Table 3)"""
    eta, phi, deta, dphi = small_case(N, nc)
    dt = (0.02 if sigma == 0.0 else 0.4 / N * rho) * (4 if method == "sdc15" else 1)
    st = sww.State(to_dev(eta, None, "dd"), to_dev(phi, None, "dd"), h, 1.0, prec=sww.DD, deta=to_dev(deta, None, "dd"), dphi=to_dev(dphi, None, "dd"))
    st.set_mesh(rho, where)
    st.set_sigma(sigma)
    e0 = st.energy()
    st.advance(dt, 1, method=method)
    r = st.read()
    mesh_q.set_mesh(rho, where)
    o = mesh_q.rk_advance(eta, phi, h, 1.0, dt, 1, deta=deta, dphi=dphi, sigma=sigma, want_energy=True, method=method)
    tol = 1e-25 / rho ** 2
    for name in ("eta", "phi", "deta", "dphi"):
        assert dd_err(r[name], o[name]) <= tol, name
    if sigma == 0.0:
        eh, el = o["energies"][0][0], o["energies"][1][0]      # word by word: a long double cannot hold a double-double
        assert abs((LD(e0[0]) - LD(eh)) + (LD(e0[1]) - LD(el))) <= 1e-27 * abs(eh)


def test_respacing_dd(sww, mesh_q):
    N, M2, nc, h = 64, 128, 2, 1.0
    eta, phi, deta, dphi = small_case(N, nc)
    s1 = sww.State(to_dev(eta, None, "dd"), to_dev(phi, None, "dd"), h, 1.0, prec=sww.DD, deta=to_dev(deta, None, "dd"), dphi=to_dev(dphi, None, "dd"))
    s1.advance(0.02, 1)
    a = s1.read()
    z1 = torch.zeros(2, M2, dtype=torch.float64, device="cuda")
    zc = torch.zeros(2, nc, M2, dtype=torch.float64, device="cuda")
    s2 = sww.State(z1, z1, h, 1.0, prec=sww.DD, deta=zc, dphi=zc)
    s2.set_mesh(0.4, 0)
    s2.respace_from(s1)
    b = s2.read()
    for name in ("eta", "phi", "deta", "dphi"):
        src = a[name].cpu().numpy()
        ref = mesh_q.respace((src[0], src[1]), (N, 1.0, 0), (M2, 0.4, 0))
        assert dd_err(b[name], ref) <= 1e-28, name


def test_shooting_map_with_segments_dd(sww, mesh_q):
    from oracle import shooting
    n, segs = 4, [(32, 0.5, 1.0, 0, 2), (64, 0.5, 0.5, 0, 3)]
    c = shoot_unknowns(n)
    S = sww.Shooter(32, n, 1.0, 1.0, prec=sww.DD)
    S.set_segments(segs)
    r, J = S.shoot(c, 1)
    o = shooting.shoot_segments_quad(mesh_q, c, segs, 1.0, 1.0)
    assert r.shape == (2, 64) and J.shape == (2, n + 1, 64)
    assert dd_err(r, o["r"]) <= 1e-25 / 0.25
    assert dd_err(J, (o["J"][0].T, o["J"][1].T)) <= 1e-25 / 0.25
    S.close()


def shoot_unknowns(n, T=7.0, amp=-0.02, seed=3):
    rng = np.random.default_rng(seed)
    c = np.zeros(n + 1)
    c[0], c[1] = T, amp
    for k in range(2, n + 1):
        c[k] = 0.2 * abs(amp) * rng.standard_normal() * np.exp(-0.7 * k)
    return c


@pytest.mark.parametrize("segs", [[(64, 0.5, 1.0, 0, 4), (128, 0.5, 0.5, 0, 6)],
                                  [(128, 0.3, 1.0, 0, 3), (128, 0.3, 0.6, 1, 3), (256, 0.4, 0.4, 0, 6)]])
def test_shooting_map_with_segments(sww, mesh_ld, segs):
    """sww_shooter_set_segments: r (3.17) with the weight sqrt(E/M) and J (3.31) on the last mesh against oracle/shooting.shoot_segments"""
    from oracle import shooting
    n = 6
    c = shoot_unknowns(n)
    S = sww.Shooter(segs[0][0], n, 1.0, 1.0)
    S.set_segments(segs)
    r, J, eta, phi = S.shoot(c, 1, want_state=True)
    o = shooting.shoot_segments(mesh_ld, c, segs, 1.0, 1.0)
    m, rho = segs[-1][0], min(sg[2] for sg in segs)
    assert r.shape == (m,) and J.shape == (n + 1, m)
    tol = 1e-11 / rho ** 2
    assert float(np.abs(r.cpu().numpy().astype(LD) - o["r"]).max() / np.abs(o["r"]).max()) <= tol
    e = np.abs(J.cpu().numpy().astype(LD) - o["J"].T).max(axis=1) / np.abs(o["J"].T).max(axis=1)
    assert float(e.max()) <= tol, e
    assert float(np.abs(eta.cpu().numpy().astype(LD) - o["eta"]).max() / np.abs(o["eta"]).max()) <= tol
    r0 = S.residual(c, 1)                                   # the steppers without columns: the same residual
    assert float((r0 - r).abs().max()) <= 1e-13 * float(r.abs().max())
    r2, J2 = S.shoot(c, 1)                                  # repeatable through the cached interpolation matrices
    assert torch.equal(r, r2) and torch.equal(J, J2)
    S.set_segments([])                                      # back to one uniform segment
    r1, _ = S.shoot(c, 8)
    assert r1.shape == (segs[0][0],)
    S.close()


def test_levenberg_marquardt_on_a_refined_mesh(sww):
    """the small-amplitude branch through the segmented device path: the period converges to the printed T = 7.19976"""
    n, eps = 4, 1e-6
    S = sww.Shooter(32, n, 1.0, 1.0)
    S.set_segments([(32, 0.5, 1.0, 0, 8), (64, 0.5, 0.5, 0, 8)])
    c0 = [7.0, eps, 0.0, 0.0, 0.0]
    c, rep = S.solve(c0, 1, fixed=[0, 1, 0, 0, 0])
    assert abs(c[0] - 7.19976) < 1e-5, (c, rep)
    assert rep["f"] < 1e-24
    S.close()


def test_segment_errors(sww):
    S = sww.Shooter(64, 4, 1.0, 1.0)
    for bad in ([(32, 1.0, 1.0, 0, 4)],                              # M_1 must be the shooter's N
                [(64, 1.0, 0.5, 0, 4)],                              # rho_1 = 1
                [(64, 0.5, 1.0, 0, 4), (128, 0.4, 0.5, 0, 4)],       # theta must sum to one
                [(64, 0.5, 1.0, 0, 4), (128, 0.5, 0.5, 0, 0)],       # at least one step
                [(64, 0.5, 1.0, 0, 4), (100, 0.5, 0.5, 0, 4)]):      # sizes the stepper supports
        with pytest.raises(sww.SwwError):
            S.set_segments(bad)
    S.close()


@pytest.mark.parametrize("N,nc,h,sigma,rho,where", [(64, 3, 1.0, 0.0, 0.5, 0), (256, 6, 1.0, 0.7, 0.4, 1), (1024, 4, float("inf"), 0.3, 0.5, 0)])
def test_adjoint_rhs_on_refined_mesh(sww, mesh_ld, N, nc, h, sigma, rho, where):
    """(B.6) with d/dx = (1/xi') d/dalpha and the mean over x in P, against the oracle; and the adjoint identity between the library's
    own linearized and adjoint operators with the inner product (1/N) sum_j (.)_j xi'(alpha_j)"""
    from test_gpu_adjoint import case
    eta, phi, et, pt = case(N, nc)
    d = sww.DtN(dev(eta), h)
    d.set_mesh(rho, where)
    d.refactor(dev(eta))
    d.set_base(dev(phi))
    es, ps = d.adjoint_rhs(dev(et), dev(pt), g=1.0, sigma=sigma)
    d.check()
    mesh_ld.set_mesh(rho, where)
    o = mesh_ld.adjoint_rhs(eta, phi, h, 1.0, et, pt, sigma=sigma)
    for name, g_ in (("eta_s", es), ("phi_s", ps)):
        ref = ld(o[name])
        err = np.abs(g_.cpu().numpy().astype(LD) - ref).max(axis=1) / np.abs(ref).max(axis=1)
        assert float(err.max()) <= 1e-11 / rho ** 2, (name, err)


def test_adjoint_rhs_on_refined_mesh_dd(sww, mesh_q):
    from test_gpu_adjoint import case
    N, nc, h, sigma, rho, where = 128, 3, 1.0, 0.4, 0.5, 1
    eta, phi, et, pt = case(N, nc)
    d = sww.DtN(to_dev(eta, None, "dd"), h, sww.DD)
    d.set_mesh(rho, where)
    d.refactor(to_dev(eta, None, "dd"))
    d.set_base(to_dev(phi, None, "dd"))
    es, ps = d.adjoint_rhs(to_dev(et, None, "dd"), to_dev(pt, None, "dd"), g=1.0, sigma=sigma)
    d.check()
    mesh_q.set_mesh(rho, where)
    o = mesh_q.adjoint_rhs(eta, phi, h, 1.0, et, pt, sigma=sigma)
    assert dd_err(es, o["eta_s"]) <= 1e-25 / rho ** 2
    assert dd_err(ps, o["phi_s"]) <= 1e-25 / rho ** 2


def test_maximum_and_minimum_size_on_refined_mesh(sww, mesh_ld):
    """N = 8192 (the largest DtN): flat surface, phi = cos(k x) sampled at the refined points, G phi = k tanh(kh) cos(k x) in closed
    form; N = 16 (the smallest) against the oracle"""
    N, h, rho = 8192, 1.0, 0.3
    x = sww.mesh_points(N, rho, 0)
    ks = [1, 5, 40]
    phi = np.stack([np.cos(k * x) for k in ks])
    d = sww.DtN(torch.zeros(N, dtype=torch.float64, device="cuda"), h)
    d.set_mesh(rho, 0)
    d.refactor(torch.zeros(N, dtype=torch.float64, device="cuda"))
    w = d.apply(dev(phi)).cpu().numpy()
    d.check()
    d.close()
    for i, k in enumerate(ks):
        want = k * np.tanh(k * h) * phi[i]
        # rounded samples under a first-order operator: ~ N eps / rho relative to the largest mode resolved, plus the parity bar
        assert float(np.abs(w[i] - want).max()) <= (1e-11 / rho ** 2) * k * np.tanh(k * h), k
    N = 16
    eta, phi1 = 0.05 * np.cos(2 * np.pi * np.arange(N) / N), np.sin(2 * np.pi * np.arange(N) / N)
    d = sww.DtN(dev(eta), h)
    d.set_mesh(0.5, 1)
    d.refactor(dev(eta))
    got = d.apply(dev(phi1[None, :])).cpu().numpy()[0]
    mesh_ld.set_mesh(0.5, 1)
    ref = ld(mesh_ld.dtn_apply(eta, h, phi1[None, :]))[0]
    assert float(np.abs(got - ref).max()) <= 1e-13


def test_metric_point_on_refined_mesh_sampled_columns(sww, mesh_ld):
    """the metric workload (N = 2048, 512 columns, all computed) on the mesh (2.10) with rho = 0.3, as bench.py's configs.metric_refined_mesh
    times it; the oracle checks 12 sampled columns (k = 1, 2, 3, N/8, N/4 always included) with the rule of parity_util, bar and floor
    divided by rho^2"""
    from parity_util import sample_columns, lin_scales, EPS
    rho, where = 0.3, 0
    c = si.metric_point(512)
    cols = sample_columns(c, 12)
    d = sww.DtN(dev(c.eta), c.h)
    d.set_mesh(rho, where)
    d.refactor(dev(c.eta))
    d.set_base(dev(c.phi0))
    out = d.linearized_apply(dev(c.deta), dev(c.dphi))
    d.check()
    got = out.cpu().numpy()[cols]
    mesh_ld.set_mesh(rho, where)
    orc, base = mesh_ld.dtn_linearized(c.eta, c.h, c.phi0, c.deta[cols], c.dphi[cols], want_base=True)
    ref = ld(orc)
    S = lin_scales(c, base, cols)
    err = np.abs(got.astype(LD) - ref).max(axis=1)
    nrm = np.abs(ref).max(axis=1)
    worst = 0.0
    for i in range(len(cols)):
        floor = float(4 * c.N * EPS["f64"] * S[i] / nrm[i])
        e = float(err[i] / nrm[i])
        assert e <= max(1e-11, floor) / rho ** 2, (int(cols[i]), e, floor)
        worst = max(worst, e)
    print("metric point on the refined mesh: E_col_max", worst)


def test_sdc15_step_on_refined_mesh_fp64(sww, mesh_ld):
    """the SDC15 stepper through the refined-mesh right-hand sides in fp64: one large step against the oracle"""
    N, nc, h, rho, where = 64, 2, 1.0, 0.5, 0
    eta, phi, deta, dphi = small_case(N, nc)
    dt = 0.08
    st = sww.State(dev(eta), dev(phi), h, 1.0, deta=dev(deta), dphi=dev(dphi))
    st.set_mesh(rho, where)
    st.advance(dt, 1, method="sdc15")
    r = st.read()
    mesh_ld.set_mesh(rho, where)
    o = mesh_ld.rk_advance(eta, phi, h, 1.0, dt, 1, deta=deta, dphi=dphi, method="sdc15")
    for name in ("eta", "phi", "deta", "dphi"):
        g, q = r[name].cpu().numpy().astype(LD).reshape(-1, N), ld(o[name]).reshape(-1, N)
        err = np.abs(g - q).max(axis=1) / np.abs(q).max(axis=1)
        assert float(err.max()) <= 1e-11 / rho ** 2, (name, err)


def test_capillary_shooting_with_segments_in_deep_water(sww, mesh_ld):
    """section 4.6 meets section 2.2: infinite depth, surface tension, two segments with a refined second mesh -- every stepper of the
    shooter gets sigma; r and J against oracle/shooting.shoot_segments"""
    from oracle import shooting
    n, sigma, h = 5, 0.1, float("inf")
    # capillary waves are stiff: omega_max ~ sqrt(sigma k^3), k = (M/2) / min xi' -- 96 at the refined end here, omega dt = 1.25
    segs = [(32, 0.5, 1.0, 0, 16), (64, 0.5, 0.6, 1, 48)]
    c = shoot_unknowns(n, T=5.0, amp=-0.01)
    S = sww.Shooter(32, n, h, 1.0)
    S.set_sigma(sigma)
    S.set_segments(segs)
    r, J = S.shoot(c, 1)
    S.close()
    o = shooting.shoot_segments(mesh_ld, c, segs, h, 1.0, sigma=sigma)
    assert np.isfinite(o["r"]).all()
    tol = 1e-11 / 0.36
    assert float(np.abs(r.cpu().numpy().astype(LD) - o["r"]).max() / np.abs(o["r"]).max()) <= tol
    e = np.abs(J.cpu().numpy().astype(LD) - o["J"].T).max(axis=1) / np.abs(o["J"].T).max(axis=1)
    assert float(e.max()) <= tol, e
    o0 = shooting.shoot_segments(mesh_ld, c, segs, h, 1.0, sigma=0.0)
    assert np.abs(o0["r"] - o["r"]).max() > 1e-4 * np.abs(o["r"]).max()      # the term matters
