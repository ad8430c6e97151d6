"""GPU parity tests of the time stepper (sww_state_create / sww_rk_advance / sww_state_read / sww_state_energy) against the
long-double oracle, plus the invariants the paper states for time stepping (energy, mean, evenness)."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import sww_inputs as si
from parity_util import ld

pytestmark = pytest.mark.gpu
LD = np.longdouble


@pytest.fixture(scope="module")
def sww():
    import paper_1210_5672_b200 as pkg
    assert pkg.lib_path().exists() and torch.cuda.is_available()
    return pkg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(gpu, ref):
    ref = ld(ref)
    return float(np.abs(gpu.astype(LD) - ref).max() / np.abs(ref).max())


def small_case(N=64, nc=6):
    c2 = si.config2()
    eta = np.ascontiguousarray(c2.eta[:: c2.N // N])
    a = np.zeros(9); a[1] = 0.05; a[2] = 0.02; a[3] = -0.01
    b = np.zeros(9); b[2] = 0.01
    phi = si.synth(N, a, b)[0]
    deta, dphi = si.fourier_unit_columns(N, nc // 2, "eta_phi")
    return eta, phi, deta, dphi, c2.h, c2.g, c2.meta["dt"]


@pytest.mark.parametrize("filt", [True, False])
def test_steps_with_variational_columns(sww, orc_ld, filt):
    """3 RK8 steps of (q, Qdot) together (3.32): state and every variational column against the oracle"""
    eta, phi, deta, dphi, h, g, dt = small_case()
    st = sww.State(dev(eta), dev(phi), h, g, deta=dev(deta), dphi=dev(dphi), filter=filt)
    st.advance(dt, 3)
    r = st.read()
    assert abs(r["t"] - 3 * dt) < 1e-15
    o = orc_ld.rk_advance(eta, phi, h, g, dt, 3, deta=deta, dphi=dphi, filter=filt)
    for name in ("eta", "phi"):
        assert rel(r[name].cpu().numpy(), o[name]) <= 1e-11, name
    for name in ("deta", "dphi"):
        gq, oq = r[name].cpu().numpy(), ld(o[name])
        err = np.abs(gq.astype(LD) - oq).max(axis=1) / np.abs(oq).max(axis=1)   # per column
        assert float(err.max()) <= 1e-11, (name, float(err.max()))


@pytest.mark.parametrize("N,nc", [(128, 8), (256, 10)])
def test_steps_with_variational_columns_tiled_sizes(sww, orc_ld, N, nc):
    """(3.32), PAPER.md:294-305 at sizes that run the persistent dataflow LU and triangular solves (N > 64) together with
    k_rhs_cols: 2 RK8 steps of config 2's surface family with a moving potential, error PER COLUMN
    E_col(c) = ||gpu_c - orc_c||_inf / ||orc_c||_inf"""
    eta, phi, deta, dphi, h, g, dt = small_case(N, nc)
    st = sww.State(dev(eta), dev(phi), h, g, deta=dev(deta), dphi=dev(dphi))
    st.advance(dt, 2)
    r = st.read()
    o = orc_ld.rk_advance(eta, phi, h, g, dt, 2, deta=deta, dphi=dphi)
    for name in ("eta", "phi"):
        assert rel(r[name].cpu().numpy(), o[name]) <= 1e-11, name
    worst = 0.0
    for name in ("deta", "dphi"):
        gq, oq = r[name].cpu().numpy(), ld(o[name])
        ref = np.abs(oq).max(axis=1)
        err = np.abs(gq.astype(LD) - oq).max(axis=1)
        for c in range(nc):
            if ref[c] == 0:
                assert err[c] <= 1e-11 * 4 * N, (name, c)
            else:
                worst = max(worst, float(err[c] / ref[c]))
                assert err[c] <= 1e-11 * ref[c], (name, c, float(err[c] / ref[c]))
    print(f"stepper with columns N={N}: worst E_col {worst:.2e}")


def test_ragged_odd_column_count(sww, orc_ld):
    """an odd number of columns (the FFT kernels work on column pairs)"""
    eta, phi, deta, dphi, h, g, dt = small_case(64, 6)
    deta, dphi = deta[:5].copy(), dphi[:5].copy()
    st = sww.State(dev(eta), dev(phi), h, g, deta=dev(deta), dphi=dev(dphi))
    st.advance(dt, 1)
    r = st.read()
    o = orc_ld.rk_advance(eta, phi, h, g, dt, 1, deta=deta, dphi=dphi)
    for name in ("eta", "phi", "deta", "dphi"):
        assert rel(r[name].cpu().numpy(), o[name]) <= 1e-11, name


def test_config2_full_period(sww, orc_ld):
    """BASELINE.json config 2: N = 256, 256 steps of the 11-stage RK8 over one linear period, one DtN setup + solve per stage.
    Parity of the final state; energy to ~13 digits, mean eta, evenness."""
    c = si.config2()
    dt, n = c.meta["dt"], c.meta["nsteps"]
    st = sww.State(dev(c.eta), dev(c.phi0), c.h, c.g)
    e0 = st.energy()[0]
    st.advance(dt, n)
    r = st.read()
    e1 = st.energy()[0]
    eta, phi = r["eta"].cpu().numpy(), r["phi"].cpu().numpy()
    assert abs(e1 - e0) <= 5e-13 * abs(e0), (e0, e1)
    assert abs(eta.mean()) <= 1e-14
    assert np.abs(eta[1:] - eta[1:][::-1]).max() <= 1e-12 * np.abs(eta).max()  # even data stay even
    o = orc_ld.rk_advance(c.eta, c.phi0, c.h, c.g, dt, n, want_energy=True)
    assert rel(eta, o["eta"]) <= 1e-11
    assert rel(phi, o["phi"]) <= 1e-11
    eo = ld(o["energies"])
    assert abs(e0 - float(eo[0])) <= 1e-13 * abs(e0) and abs(e1 - float(eo[-1])) <= 1e-12 * abs(e0)
    print("cfg2: eta err %.2e phi err %.2e energy drift %.2e" % (rel(eta, o["eta"]), rel(phi, o["phi"]), abs(e1 - e0) / abs(e0)))


def test_small_amplitude_wave_returns_after_linear_period(sww):
    """(4.35): an amplitude-1e-6 standing wave started at rest returns to its initial state after T = 2 pi / sqrt(tanh h)
    up to O(amp^2)"""
    N, h, amp = 64, 1.0, 1e-6
    al = si.grid(N)
    eta0 = amp * np.cos(al)
    T = 2 * np.pi / np.sqrt(np.tanh(h))
    st = sww.State(dev(eta0), dev(np.zeros(N)), h, 1.0)
    st.advance(T / 64, 64)
    r = st.read()
    assert np.abs(r["eta"].cpu().numpy() - eta0).max() <= 50 * amp * amp
    assert np.abs(r["phi"].cpu().numpy()).max() <= 50 * amp * amp


def _dd(hi, lo=None):
    hi = np.ascontiguousarray(hi, dtype=np.float64)
    lo = np.zeros_like(hi) if lo is None else np.ascontiguousarray(lo, dtype=np.float64)
    return torch.from_numpy(np.stack([hi, lo])).cuda().contiguous()


def _dd_err(t, ref):
    """max |gpu - oracle| / max |oracle| for a planar (2, ...) tensor against an oracle (hi, lo) pair, word by word"""
    g = t.cpu().numpy()
    d = (g[0].astype(LD) - ref[0].astype(LD)) + (g[1].astype(LD) - ref[1].astype(LD))
    return np.abs(d), np.abs(ld(ref))


@pytest.mark.parametrize("N,nc,nsteps", [(64, 4, 2), (256, 6, 1)])
def test_double_double_stepper(sww, orc_q, N, nc, nsteps):
    """the quadruple-precision time stepping of PAPER.md:163-165, 314: sww_state_create(prec = SWW_DD) advances (q, Qdot) with
    every kernel in double-double; state and every variational column against the __float128 oracle, bar 1e-25 per column"""
    c4 = si.config4(N, max(nc, 2))
    eta = (0.25 * c4.eta, 0.25 * c4.eta_lo)           # exact scaling of a double-double pair
    phi = (c4.phi0, c4.phi0_lo)
    deta = (c4.deta[:nc] * 2.0 ** -4, c4.deta_lo[:nc] * 2.0 ** -4)
    dphi = (c4.dphi[:nc] * 2.0 ** -4, c4.dphi_lo[:nc] * 2.0 ** -4)
    h, g, dt = 1.0, 1.0, si.config2().meta["dt"]
    st = sww.State(_dd(*eta), _dd(*phi), h, g, prec=sww.DD, deta=_dd(*deta), dphi=_dd(*dphi))
    e0 = st.energy()
    st.advance(dt, nsteps)
    r = st.read()
    e1 = st.energy()
    o = orc_q.rk_advance(eta, phi, h, g, dt, nsteps, deta=deta, dphi=dphi, want_energy=True)
    for name in ("eta", "phi"):
        d, ref = _dd_err(r[name], o[name])
        assert float(d.max() / ref.max()) <= 1e-25, (name, float(d.max() / ref.max()))
    worst = 0.0
    for name in ("deta", "dphi"):
        d, ref = _dd_err(r[name], o[name])
        e = (d.max(axis=1) / ref.max(axis=1)).astype(np.float64)
        worst = max(worst, float(e.max()))
        assert float(e.max()) <= 1e-25, (name, e)
    # energy against the oracle's, and conserved to ~29 digits over the step(s)
    eo = o["energies"]
    for mine, k in ((e0, 0), (e1, nsteps)):
        ref = LD(eo[0][k]) + LD(eo[1][k])
        assert abs((LD(mine[0]) - LD(eo[0][k])) + (LD(mine[1]) - LD(eo[1][k]))) <= 1e-27 * abs(ref)
    print(f"dd stepper N={N}: worst column E_col {worst:.2e}")


def test_double_double_energy_conservation(sww):
    """E(t) constant "to 29 digits in quadruple precision": a smooth standing wave, 4 steps of dt = 1e-3 (the
    order-8 truncation error is far below the double-double rounding level there)"""
    N, h, g = 32, 1.0, 1.0
    a = si.grid(N)
    eta0 = 0.05 * np.cos(a) + 0.01 * np.cos(2 * a)
    st = sww.State(_dd(eta0), _dd(np.zeros(N)), h, g, prec=sww.DD)
    e0 = st.energy()
    st.advance(1e-3, 4)
    e1 = st.energy()
    drift = abs((LD(e1[0]) - LD(e0[0])) + (LD(e1[1]) - LD(e0[1]))) / abs(LD(e0[0]))
    assert float(drift) <= 1e-28, float(drift)
    print(f"dd energy drift over 4 steps: {float(drift):.2e}")


def test_double_double_stepper_tracks_fp64(sww):
    """the same initial state through the fp64 and the double-double stepper: they agree to fp64 accuracy"""
    eta, phi, deta, dphi, h, g, dt = small_case(64, 4)
    a = sww.State(dev(eta), dev(phi), h, g, deta=dev(deta), dphi=dev(dphi))
    b = sww.State(_dd(eta), _dd(phi), h, g, prec=sww.DD, deta=_dd(deta), dphi=_dd(dphi))
    a.advance(dt, 2)
    b.advance(dt, 2)
    ra, rb = a.read(), b.read()
    for name in ("eta", "phi", "deta", "dphi"):
        x, y = ra[name].cpu().numpy(), rb[name].cpu().numpy()[0]
        assert np.abs(x - y).max() <= 1e-11 * np.abs(y).max(), name


def test_state_errors(sww):
    N = 64
    z = torch.zeros(N, dtype=torch.float64, device="cuda")
    with pytest.raises(sww.SwwError) as e:   # the double-double stepper stops at N = 2048 (include/sww.h)
        sww.State(torch.zeros((2, 4096), dtype=torch.float64, device="cuda"), torch.zeros((2, 4096), dtype=torch.float64, device="cuda"), 1.0, prec=sww.DD)
    assert e.value.status == -1
    st = sww.State(z - 2.0, z, 1.0)  # surface below the bottom
    with pytest.raises(sww.SwwError) as e:
        st.read()
    assert e.value.status == -4
