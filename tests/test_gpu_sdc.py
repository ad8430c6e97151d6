"""GPU parity tests of the SDC15 stepper (sww_sdc_advance, R15) against the oracle's sdc_advance, in fp64
and in double-double (the paper's quadruple-precision time stepping), and the energy the paper monitors."""
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


def small_case(N, nc):
    c2 = si.config2()
    eta = np.ascontiguousarray(c2.eta[:: c2.N // N])
    a = np.zeros(9); a[1] = 0.05; a[2] = 0.02; a[3] = -0.01
    b = np.zeros(9); b[2] = 0.01
    phi = si.synth(N, a, b)[0]
    deta, dphi = si.fourier_unit_columns(N, nc // 2, "eta_phi") if nc else (None, None)
    return eta, phi, deta, dphi


@pytest.mark.parametrize("N,nc,filt", [(64, 4, True), (128, 6, False)])
def test_sdc_steps_fp64(sww, orc_ld, N, nc, filt):
    eta, phi, deta, dphi = small_case(N, nc)
    dt = 0.05
    st = sww.State(dev(eta), dev(phi), 1.0, 1.0, deta=dev(deta), dphi=dev(dphi), filter=filt)
    st.advance(dt, 2, method="sdc15")
    r = st.read()
    assert abs(r["t"] - 2 * dt) < 1e-15
    o = orc_ld.rk_advance(eta, phi, 1.0, 1.0, dt, 2, deta=deta, dphi=dphi, filter=filt, method="sdc15")
    for name in ("eta", "phi"):
        ref = ld(o[name])
        assert float(np.abs(r[name].cpu().numpy().astype(LD) - ref).max() / np.abs(ref).max()) <= 1e-11, name
    for name in ("deta", "dphi"):
        gq, oq = r[name].cpu().numpy(), ld(o[name])
        err = np.abs(gq.astype(LD) - oq).max(axis=1) / np.abs(oq).max(axis=1)
        assert float(err.max()) <= 1e-11, (name, err)


def test_sdc_steps_dd_and_energy(sww, orc_q):
    """double-double: state and columns to 1e-25 against the __float128 oracle; the energy stays constant to the digits the paper
    quotes for quadruple precision ("29 in quadruple precision") once the filter is off on this coarse grid"""
    N, nc = 64, 2
    eta, phi, deta, dphi = small_case(N, nc)
    z1, zc = np.zeros(N), np.zeros_like(deta)
    pk = lambda hi, lo: torch.from_numpy(np.stack([hi, lo])).cuda().contiguous()
    dt = 0.05
    st = sww.State(pk(eta, z1), pk(phi, z1), 1.0, 1.0, prec=sww.DD, deta=pk(deta, zc), dphi=pk(dphi, zc), filter=False)
    e0 = st.energy()
    st.advance(dt, 2, method="sdc15")
    r = st.read()
    e1 = st.energy()
    o = orc_q.rk_advance(eta, phi, 1.0, 1.0, dt, 2, deta=deta, dphi=dphi, filter=False, method="sdc15")
    for name in ("eta", "phi", "deta", "dphi"):
        g = r[name].cpu().numpy()
        d = (g[0].astype(LD) - o[name][0].astype(LD)) + (g[1].astype(LD) - o[name][1].astype(LD))
        d, ref = d.reshape(-1, N), o[name][0].reshape(-1, N)
        err = np.abs(d).max(axis=1) / np.abs(ref).max(axis=1)
        assert float(err.max()) <= 1e-25, (name, err)
    drift = abs((LD(e1[0]) - LD(e0[0])) + (LD(e1[1]) - LD(e0[1]))) / abs(LD(e0[0]))
    assert float(drift) < 1e-27, float(drift)


def test_sdc_agrees_with_rk8_on_the_device(sww):
    """the two steppers of the library against each other: 2 SDC15 steps = 64 RK8 steps to fp64 roundoff (filter off)"""
    N = 128
    eta, phi, _, _ = small_case(N, 0)
    a = sww.State(dev(eta), dev(phi), 1.0, 1.0, filter=False)
    b = sww.State(dev(eta), dev(phi), 1.0, 1.0, filter=False)
    a.advance(0.1, 2, method="sdc15")
    b.advance(0.2 / 64, 64)
    ra, rb = a.read(), b.read()
    for name in ("eta", "phi"):
        assert float((ra[name] - rb[name]).abs().max() / rb[name].abs().max()) < 2e-13, name
