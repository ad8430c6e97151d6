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


def test_state_errors(sww):
    N = 64
    z = torch.zeros(N, dtype=torch.float64, device="cuda")
    with pytest.raises(sww.SwwError) as e:
        sww.State(torch.zeros((2, N), dtype=torch.float64, device="cuda"), torch.zeros((2, N), dtype=torch.float64, device="cuda"), 1.0, prec=sww.DD)
    assert e.value.status == -1  # the double-double stepper is not built
    st = sww.State(z - 2.0, z, 1.0)  # surface below the bottom
    with pytest.raises(sww.SwwError) as e:
        st.read()
    assert e.value.status == -4
