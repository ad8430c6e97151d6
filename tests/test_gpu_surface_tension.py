"""GPU parity tests of the surface-tension terms of the stepper ((2.1b); (B.4)) against the oracle, and
the capillary-gravity standing waves of section 4.6 through the device path: the printed linear period 2 pi / sqrt 2 = 4.443 (4.42)
and Concus' prediction T = sqrt 2 pi (1 + 197/320 c_1^2) (4.43), infinite depth, g = sigma / rho = 1."""
from __future__ import annotations

import math
from pathlib import Path

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
    deta, dphi = si.fourier_unit_columns(N, nc // 2, "eta_phi")
    return eta, phi, deta, dphi


@pytest.mark.parametrize("N,nc,h", [(64, 6, 1.0), (128, 8, float("inf")), (256, 6, 1.0)])
def test_steps_with_surface_tension_fp64(sww, orc_ld, N, nc, h):
    eta, phi, deta, dphi = small_case(N, nc)
    dt, sigma = 0.4 / N, 0.8                       # capillary waves are stiff: omega_max ~ (N/2)^(3/2)
    st = sww.State(dev(eta), dev(phi), h, 1.0, deta=dev(deta), dphi=dev(dphi))
    st.set_sigma(sigma)
    st.advance(dt, 2)
    r = st.read()
    o = orc_ld.rk_advance(eta, phi, h, 1.0, dt, 2, deta=deta, dphi=dphi, sigma=sigma)
    o0 = orc_ld.rk_advance(eta, phi, h, 1.0, dt, 2, deta=deta, dphi=dphi)
    assert np.abs(ld(o["phi"]) - ld(o0["phi"])).max() > 1e-6          # the term matters at this size
    for name in ("eta", "phi"):
        ref = ld(o[name])
        assert float(np.abs(r[name].cpu().numpy().astype(LD) - ref).max() / np.abs(ref).max()) <= 1e-11, name
    for name in ("deta", "dphi"):
        gq, oq = r[name].cpu().numpy(), ld(o[name])
        err = np.abs(gq.astype(LD) - oq).max(axis=1) / np.abs(oq).max(axis=1)
        assert float(err.max()) <= 1e-11, (name, err)


def test_steps_with_surface_tension_dd(sww, orc_q):
    N, nc = 64, 4
    eta, phi, deta, dphi = small_case(N, nc)
    z1, zc = np.zeros(N), np.zeros_like(deta)
    pk = lambda hi, lo: torch.from_numpy(np.stack([hi, lo])).cuda().contiguous()
    dt, sigma = 0.4 / N, 0.8
    st = sww.State(pk(eta, z1), pk(phi, z1), 1.0, 1.0, prec=sww.DD, deta=pk(deta, zc), dphi=pk(dphi, zc))
    st.set_sigma(sigma)
    st.advance(dt, 2)
    r = st.read()
    o = orc_q.rk_advance(eta, phi, 1.0, 1.0, dt, 2, deta=deta, dphi=dphi, sigma=sigma)
    for name in ("eta", "phi", "deta", "dphi"):
        g = r[name].cpu().numpy()
        d = (g[0].astype(LD) - o[name][0].astype(LD)) + (g[1].astype(LD) - o[name][1].astype(LD))
        d, ref = d.reshape(-1, N), o[name][0].reshape(-1, N)
        err = np.abs(d).max(axis=1) / np.abs(ref).max(axis=1)
        assert float(err.max()) <= 1e-25, (name, err)


def _golden(key):
    for line in (Path(__file__).parent / "golden" / "paper_values.txt").read_text().splitlines():
        line = line.split("#")[0].split()
        if line and line[0] == key:
            return float(line[1]), float(line[2])
    raise KeyError(key)


def test_capillary_gravity_standing_waves_follow_concus(sww):
    """Section 4.6: Levenberg-Marquardt on the device shooting map, h = infinity, g = sigma = 1, c_1 held fixed.  The period tends to the
    printed 2 pi / sqrt 2 = 4.443 as c_1 -> 0 and follows T = sqrt 2 pi (1 + 197/320 c_1^2) (4.43): the fitted coefficient of c_1^2
    from two amplitudes agrees with 197/320 to the size of the next-order term"""
    N, n, nsteps = 64, 8, 160                       # dt omega_max(capillary, k = 32) well inside the stability interval
    T0 = math.sqrt(2.0) * math.pi
    want, tol = _golden("T_capillary_hinf")
    assert abs(T0 - want) < tol
    S = sww.Shooter(N, n, float("inf"), 1.0)
    S.set_sigma(1.0)
    found = {}
    for c1 in (-0.02, -0.04):
        c0 = np.zeros(n + 1)
        c0[0], c0[1] = T0, c1
        fixed = [0] * (n + 1)
        fixed[1] = 1
        c, rep = S.solve(c0, nsteps, fixed=fixed, delta0=0.1, f_tol=1e-26, max_iter=60)
        assert rep["f"] < 1e-22, rep
        found[c1] = c[0]
    S.close()
    coef = {c1: (T / T0 - 1) / c1 ** 2 for c1, T in found.items()}
    for c1, k in coef.items():
        assert abs(k - 197 / 320) < 40 * c1 ** 2, (c1, k)        # 197/320 = 0.6156 up to the O(c_1^2) correction of the coefficient
    assert abs(coef[-0.02] - 197 / 320) < abs(coef[-0.04] - 197 / 320) + 1e-6
