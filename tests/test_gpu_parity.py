"""GPU parity tests: the CUDA path (through the C ABI of include/sww.h) against the CPU oracle on the same seeded inputs.
fp64 results are judged against the long-double oracle (bar 1e-11), double-double results against the __float128 oracle
(bar 1e-25); the rule is in tests/parity_util.py.  Run on the B200 box with `pytest -m gpu`."""
from __future__ import annotations

import math

import numpy as np
import pytest
import torch

import sww_inputs as si
from parity_util import (BAR, LD, check_columns, diff, from_dev, gpu_linearized, ld, lin_scales, oracle_linearized,
                         sample_columns, to_dev)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sww():
    import paper_1210_5672_b200 as pkg
    assert pkg.lib_path().exists(), "libsww.so missing: the GPU tests never fall back"
    assert torch.cuda.is_available()
    return pkg


# ------------------------------------------------------------------------------------------------ config 1
def test_cfg1_flat_surface_symbol(sww):
    """eta = 0, phi = cos 3a -> 3 tanh 3 cos 3a  ((4.34); BASELINE.json config 1)"""
    c = si.config1_flat()
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    out = d.apply(to_dev(c.dphi, None, "f64")).cpu().numpy()[0]
    d.check()
    exact = 3.0 * math.tanh(3.0) * c.phi0
    assert np.abs(out - exact).max() <= 1e-11 * np.abs(exact).max()


@pytest.mark.parametrize("h", [1.0, 0.05, float("inf")])
def test_flat_symbol_all_modes(sww, h):
    """G e^{ikx} = k tanh(kh) e^{ikx} for every resolved k at once (a multi-column apply with a ragged column count).
    The trapezoid rule on the image kernel aliases at the e^{-2hN} level, so the shallow case needs N = 512 (e^{-51})."""
    N = 512 if h < 0.1 else 128
    ks = np.arange(1, N // 2)
    j = np.arange(N)
    phi = np.cos(2 * np.pi * ((ks[:, None] * j[None, :]) % N) / N)
    d = sww.DtN(torch.zeros(N, dtype=torch.float64, device="cuda"), h)
    out = d.apply(torch.from_numpy(phi).cuda()).cpu().numpy()
    d.check()
    sym = ks * (np.tanh(ks * h) if math.isfinite(h) else 1.0)
    err = np.abs(out - sym[:, None] * phi).max(axis=1) / sym
    assert err.max() <= 1e-11, err.max()


def test_maximum_size_flat_symbol(sww):
    """N = 8192, the largest size the ABI accepts (128 x 128 tiles in the LU, 128-link solve chains): G cos(kx) = k tanh(kh) cos(kx)
    on the flat surface for low, middle and near-Nyquist modes, and a wavy surface must still report a clean status"""
    N, h = 8192, 1.0
    ks = np.array([1, 2, 3, 17, 500, 2047, 4000])
    j = np.arange(N)
    phi = np.cos(2 * np.pi * ((ks[:, None] * j[None, :]) % N) / N)
    d = sww.DtN(torch.zeros(N, dtype=torch.float64, device="cuda"), h)
    out = d.apply(torch.from_numpy(phi).cuda()).cpu().numpy()
    d.check()
    sym = ks * np.tanh(ks * h)
    err = np.abs(out - sym[:, None] * phi).max(axis=1) / sym
    assert err.max() <= 1e-11, err
    a, _ = si._family_surface(si.SEED_BASE + 3, N, 0.2, kmax=64)
    d.refactor(torch.from_numpy(si.synth(N, a)[0]).cuda())
    w = d.apply(torch.from_numpy(phi[:2]).cuda())
    d.check()
    assert torch.isfinite(w).all() and abs(float(w.mean())) < 1e-12   # mean(G phi) = 0


def test_cfg1_single_rhs(sww, orc_ld):
    c = si.config1()
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    out = from_dev(d.apply(to_dev(c.dphi, None, "f64")), "f64")
    d.check()
    orc = orc_ld.dtn_apply(c.eta, c.h, c.dphi)
    r = check_columns(out, orc, "f64", c.N, np.abs(c.dphi).max(axis=1), "cfg1")
    assert r["E_col_max"] <= 1e-12  # N = 64 has three digits of margin


# ------------------------------------------------------------------------------------------------ assembly, entry by entry
@pytest.mark.parametrize("N,h", [(64, 1.0), (256, 1.0), (256, 0.05), (128, float("inf"))])
def test_kernel_matrices_entrywise(sww, orc_ld, N, h):
    """K, G of (2.13) and eta', eta'' against the oracle: N |dK_ij|, N |dG_ij| at the 1e-13 level"""
    a, _ = si._family_surface(si.SEED_BASE + 3, N, 0.2 if h > 0.1 else 0.01, kmax=min(64, N // 4))
    eta = si.synth(N, a)[0]
    d = sww.DtN(torch.from_numpy(eta).cuda(), h)
    d.check()
    o = orc_ld.assemble(eta, h)
    for name in ("d1", "d2"):
        g = d.get(name).cpu().numpy()
        ref = ld(o[name])
        assert np.abs(g - ref).max() <= 4e-16 * max(1.0, float(np.abs(ref).max())), name
    scale = {n: float(np.abs(ld(o[n])).max()) for n in ("K", "G")}
    for name in ("K", "G"):
        g = d.get(name).cpu().numpy().T  # column-major storage -> [i, j]
        err = float(np.abs(g - ld(o[name])).max())
        assert err <= 3e-14 * max(scale[name], 1.0 / N), (name, err, scale[name])


def test_kernel_matrices_entrywise_dd(sww, orc_q):
    N = 128
    c = si.config4(N, 2)
    d = sww.DtN(to_dev(c.eta, c.eta_lo, "dd"), c.h, sww.DD)
    d.check()
    o = orc_q.assemble((c.eta, c.eta_lo), c.h)
    for name in ("K", "G"):
        t = d.get(name).cpu().numpy()
        g = (t[0].T, t[1].T)
        err = float(np.abs(diff(g, o[name])).max())
        assert err <= 1e-29 * N, (name, err)


# ------------------------------------------------------------------------------------------------ config 3 (fp64 batch)
def test_cfg3_linearized_batch(sww, orc_ld):
    c = si.config3()
    out, d = gpu_linearized(c)
    orc, base = oracle_linearized(orc_ld, c)
    r = check_columns(out, orc, "f64", c.N, lin_scales(c, base), "cfg3")
    assert r["cols_with_floor_above_bar"] == 0
    for name in ("dphi0", "W0", "u", "v"):
        g = d.get(name).cpu().numpy()
        ref = ld(base[name])
        assert np.abs(g - ref).max() <= 1e-13 * np.abs(ref).max(), name
    print("cfg3", r)


@pytest.mark.parametrize("nrhs", [1, 2, 3, 63, 65, 130])
def test_ragged_column_counts(sww, orc_ld, nrhs):
    """column counts that are not multiples of any tile: every column must match, and nothing is written past nrhs"""
    c = si.config3(256, 256)
    sel = np.arange(nrhs) * (256 // nrhs)
    c.deta, c.dphi = np.ascontiguousarray(c.deta[sel]), np.ascontiguousarray(c.dphi[sel])
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    d.set_base(to_dev(c.phi0, None, "f64"))
    buf = torch.full((nrhs + 2, c.N), 777.0, dtype=torch.float64, device="cuda")
    d.linearized_apply(to_dev(c.deta, None, "f64"), to_dev(c.dphi, None, "f64"), out=buf[:nrhs])
    d.check()
    assert bool((buf[nrhs:] == 777.0).all()), "wrote past the last column"
    orc, base = oracle_linearized(orc_ld, c)
    check_columns(from_dev(buf[:nrhs], "f64"), orc, "f64", c.N, lin_scales(c, base), f"ragged{nrhs}")


def test_apply_is_pure_and_repeatable(sww):
    c = si.config3(256, 64)
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    phi = to_dev(c.dphi, None, "f64")
    a = d.apply(phi).clone()
    d.set_base(to_dev(c.phi0, None, "f64"))
    d.linearized_apply(to_dev(c.deta, None, "f64"), phi)
    b = d.apply(phi)
    assert torch.equal(a, b)
    inplace = phi.clone()
    d.apply(inplace, out=inplace)
    assert torch.equal(a, inplace)


def test_refactor_matches_fresh_setup(sww):
    c3, c4 = si.config3(256, 16), si.config4(256, 2)
    d = sww.DtN(to_dev(c4.eta, None, "f64"), 1.0)
    d.refactor(to_dev(c3.eta, None, "f64"))
    fresh = sww.DtN(to_dev(c3.eta, None, "f64"), 1.0)
    phi = to_dev(c3.dphi, None, "f64")
    assert torch.equal(d.apply(phi), fresh.apply(phi))


# ------------------------------------------------------------------------------------------------ config 4 (double-double)
def test_cfg4_double_double_batch(sww, orc_q):
    c = si.config4()
    out, d = gpu_linearized(c)
    orc, base = oracle_linearized(orc_q, c)
    r = check_columns(out, orc, "dd", c.N, lin_scales(c, base), "cfg4")
    assert r["cols_with_floor_above_bar"] == 0
    for name in ("dphi0", "W0", "u", "v"):
        t = d.get(name).cpu().numpy()
        err = np.abs(diff((t[0], t[1]), base[name])).max()
        assert err <= 1e-27 * float(np.abs(ld(base[name])).max()), name
    print("cfg4", r)


def test_dd_plain_apply_and_fp64_consistency(sww, orc_q):
    """dd apply against the __float128 oracle, and the fp64 handle on the rounded inputs agrees with it to fp64 accuracy"""
    c = si.config4(256, 6)
    d = sww.DtN(to_dev(c.eta, c.eta_lo, "dd"), c.h, sww.DD)
    out = from_dev(d.apply(to_dev(c.dphi, c.dphi_lo, "dd")), "dd")
    d.check()
    orc = orc_q.dtn_apply((c.eta, c.eta_lo), c.h, (c.dphi, c.dphi_lo))
    check_columns(out, orc, "dd", c.N, np.abs(c.dphi).max(axis=1), "dd apply")
    d64 = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    out64 = d64.apply(to_dev(c.dphi, None, "f64")).cpu().numpy()
    assert np.abs(out64 - out[0]).max() <= 1e-11 * np.abs(out[0]).max()


# ------------------------------------------------------------------------------------------------ full sizes, sampled columns
def test_metric_point_sampled_columns(sww, orc_ld):
    """BASELINE.json metric point, N = 2048, nrhs = 512, in the launch configuration bench.py times; the oracle checks a
    seeded subset of 32 columns (k = 1, 2, 3, N/8, N/4 always included)"""
    c = si.metric_point(512)
    cols = sample_columns(c, 32)
    out, d = gpu_linearized(c, cols)
    orc, base = oracle_linearized(orc_ld, c, cols)
    r = check_columns(out, orc, "f64", c.N, lin_scales(c, base, cols), "metric")
    assert r["cols_with_floor_above_bar"] == 0
    print("metric point", r)


@pytest.mark.parametrize("amp1,variant", [(0.1, 0), (0.3, 0), (0.1, 1), (0.2, 1), (0.3, 1), (0.1, 2), (0.2, 2), (0.3, 2)])
def test_metric_point_other_seeds_and_amplitudes(sww, orc_ld, amp1, variant):
    """the metric point on other draws of the seeded surface / potential and at amplitudes 0.1, 0.2, 0.3 of the cos(alpha) mode
    ((0.2, seed 0) is test_metric_point_sampled_columns): all 512 columns computed, 12 sampled ones against the oracle"""
    c = si.metric_point(512, amp1, variant)
    cols = sample_columns(c, 12, seed=11 + variant)
    out, d = gpu_linearized(c, cols)
    orc, base = oracle_linearized(orc_ld, c, cols)
    r = check_columns(out, orc, "f64", c.N, lin_scales(c, base, cols), f"metric amp {amp1} variant {variant}")
    # where the floor F_c exceeds the bar at all, it is on the k = 1 surface-perturbation column only (output small against
    # (|u| + |v|) |deta|: the two terms of (B.2) nearly cancel there)
    assert all(int(cols[i]) == 0 for i in r["floor_cols"]), [int(cols[i]) for i in r["floor_cols"]]
    print(f"metric point amp1={amp1} variant={variant}", r)


def test_metric_point_dd_sampled_columns(sww, orc_q):
    """the double-double leg of the metric as bench.py times it: N = 2048, 128 columns (config-4 family), all computed; the
    __float128 oracle checks 8 sampled columns (k = 1, 2, 3 always included); bar 1e-25"""
    c = si.metric_point_dd(128, 2048)
    cols = sample_columns(c, 8)
    out, d = gpu_linearized(c, cols)
    orc, base = oracle_linearized(orc_q, c, cols)
    r = check_columns(out, orc, "dd", c.N, lin_scales(c, base, cols), "metric dd")
    assert r["cols_with_floor_above_bar"] == 0
    print("metric dd (N=2048, 128 columns)", r)


def test_gemm_128x128_tiles(sww):
    """the 128 x 128 tile instantiation of the G product (taken when (N/128) * ceil(nrhs/128) >= 148: N = 4096 with 640 columns):
    (a) flat surface: G cos(kx) = k tanh(kh) cos(kx) for k = 1..640 ((4.34));
    (b) wavy surface: the same 640 columns applied in two halves of 320 go through the 64 x 64 tiles -- same result to rounding"""
    N, h, nc = 4096, 1.0, 640
    ks = np.arange(1, nc + 1)
    j = np.arange(N)
    phi = torch.from_numpy(np.cos(2 * np.pi * ((ks[:, None] * j[None, :]) % N) / N)).cuda()
    d = sww.DtN(torch.zeros(N, dtype=torch.float64, device="cuda"), h)
    out = d.apply(phi)
    d.check()
    sym = torch.from_numpy(ks * np.tanh(ks * h)).cuda()
    err = ((out - sym[:, None] * phi).abs().max(dim=1).values / sym).max()
    assert float(err) <= 1e-11, float(err)
    a, _ = si._family_surface(si.SEED_BASE + 3, N, 0.2, kmax=64)
    d.refactor(torch.from_numpy(si.synth(N, a)[0]).cuda())
    wide = d.apply(phi)
    halves = torch.cat([d.apply(phi[:320].contiguous()), d.apply(phi[320:].contiguous())])
    d.check()
    scale = wide.abs().max(dim=1).values
    assert float(((wide - halves).abs().max(dim=1).values / scale).max()) <= 1e-12


def test_dd_maximum_size_flat_symbol_and_small_sizes(sww, orc_q):
    """the ends of the double-double size range (include/sww.h: 16 <= N <= 4096).  N = 4096 runs the one-multiplier spectral
    passes: flat surface, G cos(kx) = k tanh(kh) cos(kx) ((4.34)) with the symbol from mpmath and the columns
    synthesised in double-double; N = 16 and 32 (the small-size dd products) against the __float128 oracle"""
    import mpmath
    N, h = 4096, 1.0
    ks = [1, 2, 37, 1000, 2047]
    coef = np.zeros((len(ks), max(ks) + 1))
    for r, k in enumerate(ks):
        coef[r, k] = 1.0
    phi_hi, phi_lo = si.synth_dd(N, coef)
    d = sww.DtN(torch.zeros((2, N), dtype=torch.float64, device="cuda"), h, sww.DD)
    out = d.apply(to_dev(phi_hi, phi_lo, "dd")).cpu().numpy()
    d.check()
    del d
    for r, k in enumerate(ks):
        with mpmath.workdps(50):   # 97 sampled entries of the column, everything in 50-digit arithmetic
            sym = mpmath.mpf(k) * mpmath.tanh(mpmath.mpf(k) * h)
            worst = max(abs((mpmath.mpf(float(out[0][r][j])) + mpmath.mpf(float(out[1][r][j])))
                            - sym * (mpmath.mpf(float(phi_hi[r][j])) + mpmath.mpf(float(phi_lo[r][j])))) for j in range(0, N, 43))
            assert worst <= mpmath.mpf(1e-25) * sym, (k, float(worst / sym))
    for Ns in (16, 32):
        c = si.config4(Ns, 4)
        eta = (0.1 * c.eta, np.zeros(Ns))   # a gentle surface that N = 16 resolves
        dd_ = sww.DtN(to_dev(*eta, "dd"), c.h, sww.DD)
        res = from_dev(dd_.apply(to_dev(c.dphi * 2.0 ** -3, c.dphi_lo * 2.0 ** -3, "dd")), "dd")
        dd_.check()
        orc = orc_q.dtn_apply(eta, c.h, (c.dphi * 2.0 ** -3, c.dphi_lo * 2.0 ** -3))
        check_columns(res, orc, "dd", Ns, np.abs(c.dphi * 2.0 ** -3).max(axis=1), f"dd N={Ns}")


def test_cfg5_shallow_sampled_columns(sww, orc_ld):
    """config 5: N = 4096, h = 0.05, phi0 = 0 (u = v = 0: the deta part of every column has no effect); the fp64 floor binds
    on the lowest wavenumbers only"""
    c = si.config5()
    cols = sample_columns(c, 16)
    out, d = gpu_linearized(c, cols)
    orc, base = oracle_linearized(orc_ld, c, cols)
    r = check_columns(out, orc, "f64", c.N, lin_scales(c, base, cols), "cfg5")
    # F_c = 4 N eps S_c / ||orc_c|| = 1.8e-12 / (k tanh(k h)) exceeds the bar for k = 1 only (3.6e-11; k = 2: 9.1e-12): the two
    # k = 1 columns of the sample (cos and sin), as DESIGN.md section 6 states
    assert r["cols_with_floor_above_bar"] == 2, r
    print("cfg5", r)


def test_properties_at_full_size(sww):
    """properties that hold at any size, on all 512 columns of the metric point: mean(G phi) = 0 (T4) and
    self-adjointness int chi G phi = int phi G chi ((B.5))"""
    c = si.metric_point(512)
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    phi = to_dev(c.dphi + c.deta, None, "f64")
    w = d.apply(phi)
    d.check()
    assert float(w.mean(dim=1).abs().max()) <= 1e-12 * float(w.abs().max())
    a = phi @ w.T
    assert float((a - a.T).abs().max()) <= 1e-11 * float(a.abs().max())


# ------------------------------------------------------------------------------------------------ degenerate cases and errors
def test_zero_columns_and_zero_rhs(sww):
    c = si.config3(256, 4)
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    d.set_base(to_dev(c.phi0, None, "f64"))
    empty = torch.empty((0, c.N), dtype=torch.float64, device="cuda")
    assert d.apply(empty).shape == (0, c.N)
    z = torch.zeros((3, c.N), dtype=torch.float64, device="cuda")
    assert float(d.linearized_apply(z, z).abs().max()) == 0.0
    d.check()


@pytest.mark.parametrize("N", [128, 256, 1024, 4096])
def test_single_column_solver_matches_batch_solver(sww, orc_ld, N):
    """One right-hand side runs through the 8-column slab instantiation of the dataflow solver, a wider batch through another:
    the same column must come out of both to rounding, from the smallest tiled size (2 tiles) to N = 4096; N <= 256 is also
    checked against the oracle."""
    c = si.config3(N, 80) if N < 4096 else si.config5(N, 80)
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    cols = to_dev(c.dphi, None, "f64")
    batch = d.apply(cols).cpu().numpy()
    single = np.stack([d.apply(cols[i:i + 1].contiguous()).cpu().numpy()[0] for i in range(2)])
    d.check()
    scale = np.abs(batch[:2]).max(axis=1, keepdims=True)
    assert np.abs(single - batch[:2]).max() <= 4.0 * N * 2.0 ** -53 * float(np.abs(c.dphi).max() / scale.min()) * scale.max()
    if N <= 256:
        orc = orc_ld.dtn_apply(c.eta, c.h, c.dphi[:2])
        check_columns((single, None), orc, "f64", N, np.abs(c.dphi[:2]).max(axis=1), f"single N={N}")


def test_nan_column_stays_in_its_column(sww):
    """a non-finite right-hand side must neither hang the dataflow solves (they poll the data itself) nor leak beyond the column
    it shares a complex FFT with (columns 2c and 2c + 1 are transformed as one complex vector)"""
    c = si.config3(256, 8)
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    good = d.apply(to_dev(c.dphi, None, "f64")).cpu().numpy()
    bad_in = c.dphi.copy()
    bad_in[2, 17] = np.nan
    bad_in[4, :] = np.inf
    out = d.apply(to_dev(bad_in, None, "f64")).cpu().numpy()
    d.check()
    for col in (0, 1, 6, 7):
        assert np.array_equal(out[col], good[col])
    assert not np.isfinite(out[2]).any() and not np.isfinite(out[4]).any()


def test_all_ones_payload_column(sww):
    """a right-hand side filled with 0xFF bytes is a NaN with the payload the triangular solves reserve for "not computed yet":
    it must behave like any other NaN column (no hang, no give-up status, its FFT partner spoiled, all other columns exact)"""
    c = si.config3(256, 40)
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    good = d.apply(to_dev(c.dphi, None, "f64")).cpu().numpy()
    bad_in = to_dev(c.dphi, None, "f64")
    bad_in[6].view(torch.int64).fill_(-1)
    out = d.apply(bad_in).cpu().numpy()
    assert d.status() == 0
    for col in range(40):
        if col not in (6, 7):
            assert np.array_equal(out[col], good[col]), col
    assert np.isnan(out[6]).all()
    assert np.array_equal(d.apply(to_dev(c.dphi, None, "f64")).cpu().numpy(), good)


def test_repeated_solves_are_bit_identical_under_concurrent_copies(sww):
    """the dataflow kernels hand tiles over through L2 without grid barriers: 500 repeated setup-free applies of the metric-point
    batch (N = 2048, 512 columns) and 40 refactor + apply rounds while a second stream keeps copying 64 MB buffers must all
    return the same bits, with a clean status"""
    c = si.metric_point(512)
    d = sww.DtN(to_dev(c.eta, None, "f64"), c.h)
    phi = to_dev(c.dphi + c.deta, None, "f64")
    ref = d.apply(phi).clone()
    side = torch.cuda.Stream()
    src = torch.empty(8 << 20, dtype=torch.float64, device="cuda").normal_()
    dst = torch.empty_like(src)
    out = torch.empty_like(ref)
    bad = 0
    for it in range(500):
        with torch.cuda.stream(side):
            dst.copy_(src, non_blocking=True)
        if it % 12 == 11 and it < 480:
            d.refactor(to_dev(c.eta, None, "f64"))
        d.apply(phi, out=out)
        bad += int(not torch.equal(out, ref))
    torch.cuda.synchronize()
    d.check()
    assert bad == 0, f"{bad} of 500 repeated applies differed"


def test_minimum_size(sww, orc_ld):
    N = 16
    a = np.zeros(4); a[1] = 0.05
    eta = si.synth(N, a)[0]
    phi = si.synth(N, np.array([0, 0.3, 0.1]), np.array([0, 0.0, 0.2]))
    d = sww.DtN(torch.from_numpy(eta).cuda(), 1.0)
    out = from_dev(d.apply(torch.from_numpy(phi).cuda()), "f64")
    d.check()
    check_columns(out, orc_ld.dtn_apply(eta, 1.0, phi), "f64", N, np.abs(phi).max(axis=1), "N16")


def test_error_codes(sww):
    N = 64
    eta = torch.zeros(N, dtype=torch.float64, device="cuda")
    d = sww.DtN(eta, 1.0)
    z = torch.zeros((1, N), dtype=torch.float64, device="cuda")
    with pytest.raises(sww.SwwError) as e:
        d.linearized_apply(z, z)
    assert e.value.status == -6  # SWW_ENOBASE
    bad = sww.DtN(eta - 2.0, 1.0)  # h + eta < 0
    assert bad.status() == -4       # SWW_EBOTTOM
    with pytest.raises(sww.SwwError) as e:
        sww.DtN(torch.zeros(48, dtype=torch.float64, device="cuda"), 1.0)
    assert e.value.status == -1


def test_host_buffer_entry_point(sww):
    c = si.config3(256, 32)
    dev, _ = gpu_linearized(c)
    host = sww.dtn_linearized_host(*(torch.from_numpy(np.ascontiguousarray(a)) for a in (c.eta, c.phi0, c.deta, c.dphi)), c.h)
    assert np.array_equal(host.numpy(), dev[0])
    # the library caches one context between host calls: a second surface, another depth, fewer / more columns, another N
    # must each give exactly what a fresh device-side handle gives
    for case in (si.config3(256, 8), si.config3(256, 64), si.config5(256, 16), si.config3(128, 32), si.config3(512, 256), si.config3(512, 300), c):
        dev, _ = gpu_linearized(case)
        args = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (case.eta, case.phi0, case.deta, case.dphi)]
        out = torch.empty_like(args[3]).pin_memory()
        host = sww.dtn_linearized_host(*args, case.h, out=out)
        assert host is out and np.array_equal(host.numpy(), dev[0]), case.name
    # a failing call (surface below the bottom) reports its status and does not poison the next one
    with pytest.raises(sww.SwwError) as e:
        sww.dtn_linearized_host(torch.from_numpy(c.eta - 2.0), *(torch.from_numpy(np.ascontiguousarray(a)) for a in (c.phi0, c.deta, c.dphi)), c.h)
    assert e.value.status == -4
    dev, _ = gpu_linearized(c)
    host = sww.dtn_linearized_host(*(torch.from_numpy(np.ascontiguousarray(a)) for a in (c.eta, c.phi0, c.deta, c.dphi)), c.h)
    assert np.array_equal(host.numpy(), dev[0])
    sww.host_cache_clear()
