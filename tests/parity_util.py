"""Helpers shared by the GPU parity tests: run a Case through the C ABI, run it through the oracle, apply the parity rule.

Parity rule.  Per column c:
    E_col(c) = ||gpu_c - orc_c||_inf / ||orc_c||_inf  <=  max(bar, F_c),
    F_c = 4 N eps S_c / ||orc_c||_inf,   S_c = ||dphi_c||_inf + (||u||_inf + ||v||_inf) ||deta_c||_inf   (||phi_c||_inf for a plain apply),
bar = 1e-11 / eps = 2^-53 in fp64, bar = 1e-25 / eps = 2^-104 in double-double.  F_c is the floor of a first-order operator
applied to a density stored in working precision; it exceeds the bar only on shallow-water low-k columns (config 5, k <= 3).
A zero oracle column must come back below bar * 4 N ||inputs||_inf in absolute value.
"""
from __future__ import annotations

import numpy as np
import torch

import sww_inputs as si

LD = np.longdouble
BAR = {"f64": 1e-11, "dd": 1e-25}
EPS = {"f64": 2.0 ** -53, "dd": 2.0 ** -104}


def ld(x):
    if isinstance(x, tuple):
        return np.asarray(x[0], dtype=LD) + (0 if x[1] is None else np.asarray(x[1], dtype=LD))
    return np.asarray(x, dtype=LD)


def to_dev(hi, lo, prec):
    """numpy hi (+lo) -> CUDA tensor in the ABI layout (dd: planar (2, ...))"""
    hi = np.ascontiguousarray(hi, dtype=np.float64)
    if prec == "dd":
        lo = np.zeros_like(hi) if lo is None else np.ascontiguousarray(lo, dtype=np.float64)
        return torch.from_numpy(np.stack([hi, lo])).cuda().contiguous()
    return torch.from_numpy(hi).cuda().contiguous()


def from_dev(t, prec):
    a = t.detach().cpu().numpy()
    return (a[0], a[1]) if prec == "dd" else (a, None)


def diff(gpu, orc):
    """gpu - orc for (hi, lo) pairs, formed word by word so that double-double differences survive the 64-bit long double"""
    d = np.asarray(gpu[0], dtype=LD) - np.asarray(orc[0], dtype=LD)
    if gpu[1] is not None:
        d = d + np.asarray(gpu[1], dtype=LD)
    if orc[1] is not None:
        d = d - np.asarray(orc[1], dtype=LD)
    return d


def gpu_linearized(case: si.Case, cols=None):
    """setup + set_base + linearized_apply through the C ABI; returns (out (hi, lo), handle)"""
    import paper_1210_5672_b200 as sww
    prec = sww.DD if case.prec == "dd" else sww.F64
    d = sww.DtN(to_dev(case.eta, case.eta_lo, case.prec), case.h, prec)
    d.set_base(to_dev(case.phi0, case.phi0_lo, case.prec))
    out = d.linearized_apply(to_dev(case.deta, case.deta_lo, case.prec), to_dev(case.dphi, case.dphi_lo, case.prec))
    d.check()
    o = from_dev(out, case.prec)
    if cols is not None:
        o = (o[0][cols], None if o[1] is None else o[1][cols])
    return o, d


def oracle_linearized(orc, case: si.Case, cols=None, want_base=True):
    sel = (lambda a: None if a is None else a[cols]) if cols is not None else (lambda a: a)
    pair = lambda hi, lo: (hi, lo) if lo is not None else hi
    return orc.dtn_linearized(pair(case.eta, case.eta_lo), case.h, pair(case.phi0, case.phi0_lo),
                              pair(sel(case.deta), sel(case.deta_lo)), pair(sel(case.dphi), sel(case.dphi_lo)), want_base=want_base)


def check_columns(gpu, orc, prec, N, S, what=""):
    """apply the parity rule; S: per-column input scale S_c.  Returns a dict of summary numbers."""
    bar, eps = BAR[prec], EPS[prec]
    d = np.abs(diff(gpu, orc)).max(axis=1)
    ref = np.abs(ld(orc)).max(axis=1)
    S = np.asarray(S, dtype=LD)
    worst, nfloor, floor_cols = 0.0, 0, []
    for c in range(d.shape[0]):
        if ref[c] == 0:
            assert d[c] <= bar * 4 * N * S[c], f"{what} column {c}: zero oracle column, |gpu| = {float(d[c]):.3e}"
            continue
        e = float(d[c] / ref[c])
        floor = float(4 * N * eps * S[c] / ref[c])
        nfloor += floor > bar
        if floor > bar:
            floor_cols.append(c)
        assert e <= max(bar, floor), f"{what} column {c}: E_col = {e:.3e} > max(bar {bar:.1e}, floor {floor:.3e})"
        worst = max(worst, e)
    e_blk = float(d.max() / ref.max()) if ref.max() > 0 else 0.0
    return {"E_col_max": worst, "E_blk": e_blk, "cols_with_floor_above_bar": int(nfloor), "floor_cols": floor_cols}


def lin_scales(case: si.Case, base, cols=None):
    """S_c = ||dphi_c||_inf + (||u||_inf + ||v||_inf) ||deta_c||_inf"""
    de = case.deta if cols is None else case.deta[cols]
    dp = case.dphi if cols is None else case.dphi[cols]
    uv = float(np.abs(ld(base["u"])).max() + np.abs(ld(base["v"])).max())
    return np.abs(dp).max(axis=1) + uv * np.abs(de).max(axis=1)


def sample_columns(case: si.Case, n=32, seed=7):
    """seeded subset of columns for the large cases, always with k = 1, 2, 3, N/8, N/4 of both field types"""
    nrhs, N = case.nrhs, case.N
    must = []
    for k in (1, 2, 3, N // 8, N // 4):
        for t in (0, 1):
            c = 2 * k - 2 + t
            if 0 <= c < nrhs:
                must.append(c)
    rng = np.random.default_rng(seed)
    rest = [c for c in rng.permutation(nrhs) if c not in must]
    cols = sorted(set(must + [int(c) for c in rest[:max(0, n - len(must))]]))
    return np.array(cols, dtype=np.int64)
