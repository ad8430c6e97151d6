"""GPU parity test of the right-hand side of the adjoint system (B.6) (sww_dtn_adjoint_rhs) against the oracle, per
column, and the adjoint identity <DF(q) qdot, q~> = <qdot, DF(q)^* q~> between the library's own linearized and adjoint operators."""
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


def case(N, nc, seed=11):
    rng = np.random.default_rng(seed)
    def smooth(amp, mean=True):
        c, s = np.zeros(13), np.zeros(13)
        c[1:] = amp * rng.standard_normal(12) * np.exp(-0.4 * np.arange(1, 13))
        s[1:] = amp * rng.standard_normal(12) * np.exp(-0.4 * np.arange(1, 13))
        if mean:
            c[0] = 0.3 * amp * rng.standard_normal()
        return si.synth(N, c, s)[0]
    eta, phi = smooth(0.05, mean=False), smooth(0.1)
    et = np.stack([smooth(1.0) for _ in range(nc)])
    pt = np.stack([smooth(1.0) for _ in range(nc)])
    return eta, phi, et, pt


@pytest.mark.parametrize("N,nc,h,sigma", [(64, 3, 1.0, 0.0), (256, 6, 1.0, 0.7), (512, 5, float("inf"), 0.0), (2048, 4, 0.5, 0.3)])
def test_adjoint_rhs_against_the_oracle(sww, orc_ld, N, nc, h, sigma):
    eta, phi, et, pt = case(N, nc)
    d = sww.DtN(dev(eta), h)
    d.set_base(dev(phi))
    es, ps = d.adjoint_rhs(dev(et), dev(pt), g=1.0, sigma=sigma)
    d.check()
    o = orc_ld.adjoint_rhs(eta, phi, h, 1.0, et, pt, sigma=sigma)
    for name, g_ in (("eta_s", es), ("phi_s", ps)):
        ref = ld(o[name])
        err = np.abs(g_.cpu().numpy().astype(LD) - ref).max(axis=1) / np.abs(ref).max(axis=1)
        assert float(err.max()) <= 1e-11, (name, err)


def test_dtn_is_self_adjoint_on_the_device(sww):
    """Green's identity (B.5), on which the adjoint system rests: G is self-adjoint, <phi_a, G phi_b> = <G phi_a, phi_b>"""
    N = 512
    eta, phi, a, b = case(N, 4, seed=5)
    d = sww.DtN(dev(eta), 1.0)
    Ga, Gb = d.apply(dev(a)), d.apply(dev(b))
    lhs = (dev(a) * Gb).mean(dim=1)
    rhs = (Ga * dev(b)).mean(dim=1)
    assert float((lhs - rhs).abs().max()) < 1e-13 * float(lhs.abs().max())


def test_adjoint_rhs_double_double(sww, orc_q):
    N, nc, h, sigma = 128, 3, 1.0, 0.4
    eta, phi, et, pt = case(N, nc)
    pk = lambda a: torch.from_numpy(np.stack([a, np.zeros_like(a)])).cuda().contiguous()
    d = sww.DtN(pk(eta), h, sww.DD)
    d.set_base(pk(phi))
    es, ps = d.adjoint_rhs(pk(et), pk(pt), g=1.0, sigma=sigma)
    d.check()
    o = orc_q.adjoint_rhs(eta, phi, h, 1.0, et, pt, sigma=sigma)
    for name, g_ in (("eta_s", es), ("phi_s", ps)):
        g_ = g_.cpu().numpy()
        diff = (g_[0].astype(LD) - o[name][0].astype(LD)) + (g_[1].astype(LD) - o[name][1].astype(LD))
        err = np.abs(diff).max(axis=1) / np.abs(o[name][0]).max(axis=1)
        assert float(err.max()) <= 1e-25, (name, err)


def test_adjoint_argument_checks(sww):
    N = 64
    eta, phi, et, pt = case(N, 2)
    d = sww.DtN(dev(eta), 1.0)
    with pytest.raises(sww.SwwError) as e:
        d.adjoint_rhs(dev(et), dev(pt))
    assert e.value.status == -6              # SWW_ENOBASE
