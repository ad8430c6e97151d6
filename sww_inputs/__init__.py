"""Seeded synthetic inputs for the DtN hot path (shared by the oracle tests and the CUDA tests/bench).

This module holds NONE of the method's arithmetic: it only synthesises surfaces, potentials and
right-hand-side columns with the shapes, sizes and spectra of the paper's workloads
(unit depth PAPER.md:320-332, shallow h=0.05 PAPER.md:517-533, sizes from Tables 1-3
PAPER.md:491-497, 572-593) following the recipe in BASELINE.json `configs` / DESIGN.md §4.
Neither `oracle/` nor the CUDA package is imported here.

Layout: a batch of nrhs columns of N reals is a C-contiguous numpy array of shape (nrhs, N)
(= column-major N x nrhs: column c starts at offset c*N).
A double-double quantity is a pair (hi, lo) of such arrays, value = hi + lo exactly.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from fractions import Fraction
from functools import lru_cache

import numpy as np

SEED_BASE = 12105672 * 10  # seed = SEED_BASE + config number

_M64 = (1 << 64) - 1


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """Counter-based 64-bit mixer (splitmix64 finaliser) on uint64 arrays."""
    x = (x + np.uint64(0x9E3779B97F4A7C15)) & np.uint64(_M64)
    z = x
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def uniforms(seed: int, stream: int, n: int) -> np.ndarray:
    """n uniforms in (0,1), a pure function of (seed, stream, index)."""
    with np.errstate(over="ignore"):
        ctr = np.arange(n, dtype=np.uint64)
        key = _splitmix64(np.full(1, (seed * 0x100000001B3 + stream) & _M64, dtype=np.uint64))[0]
        bits = _splitmix64(_splitmix64(ctr ^ key) + np.uint64(stream))
    return ((bits >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normals(seed: int, stream: int, n: int) -> np.ndarray:
    """n standard normals (Box-Muller on the counter-based uniforms)."""
    u1 = uniforms(seed, 2 * stream, n)
    u2 = uniforms(seed, 2 * stream + 1, n)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def grid(N: int) -> np.ndarray:
    return 2.0 * np.pi * np.arange(N) / N


def _trig_int_tables(N: int, bits: int = 160):
    """cos(2 pi m/N), sin(2 pi m/N), m=0..N-1 as Python ints scaled by 2**bits (mpmath, 60 digits)."""
    import mpmath

    with mpmath.workdps(70):
        two_pi = 2 * mpmath.pi
        scale = mpmath.mpf(2) ** bits
        cs = [int(mpmath.nint(mpmath.cos(two_pi * m / N) * scale)) for m in range(N)]
        sn = [int(mpmath.nint(mpmath.sin(two_pi * m / N) * scale)) for m in range(N)]
    return cs, sn


@lru_cache(maxsize=8)
def _trig_tables_cached(N: int):
    return _trig_int_tables(N)


def _split_hi_lo(num: int, shift: int):
    """Exact integer num / 2**shift -> (hi, lo) doubles, hi = RN(x), lo = RN(x - hi)."""
    x = Fraction(num, 1 << shift)
    hi = float(x)
    lo = float(x - Fraction(hi))
    return hi, lo


def synth_dd(N: int, cos_coef: np.ndarray, sin_coef: np.ndarray | None = None):
    """Trigonometric synthesis sum_k (a_k cos k alpha_j + b_k sin k alpha_j) carried to ~2**-150,
    returned as a (hi, lo) pair of float64 arrays.  cos_coef/sin_coef: (ncol, kmax+1) float64
    (index = wavenumber k).  Exact integer fixed-point accumulation; input recipe only."""
    cos_coef = np.atleast_2d(np.asarray(cos_coef, dtype=np.float64))
    ncol, kdim = cos_coef.shape
    if sin_coef is None:
        sin_coef = np.zeros_like(cos_coef)
    sin_coef = np.atleast_2d(np.asarray(sin_coef, dtype=np.float64))
    cs, sn = _trig_tables_cached(N)
    CB = 120  # coefficient fixed-point bits
    fix = lambda v: int(round(Fraction(float(v)) * (1 << CB)))
    ai = np.array([[fix(v) for v in row] for row in cos_coef], dtype=object)
    bi = np.array([[fix(v) for v in row] for row in sin_coef], dtype=object)
    idx = (np.arange(kdim, dtype=np.int64)[:, None] * np.arange(N, dtype=np.int64)[None, :]) % N
    acc = ai.dot(np.array(cs, dtype=object)[idx]) + bi.dot(np.array(sn, dtype=object)[idx])
    hi = np.zeros((ncol, N))
    lo = np.zeros((ncol, N))
    for c in range(ncol):
        for j in range(N):
            hi[c, j], lo[c, j] = _split_hi_lo(acc[c, j], CB + 160)
    return hi, lo


def synth(N: int, cos_coef: np.ndarray, sin_coef: np.ndarray | None = None) -> np.ndarray:
    """Plain float64 trigonometric synthesis (phase reduced exactly: cos(2 pi (k j mod N)/N))."""
    cos_coef = np.atleast_2d(np.asarray(cos_coef, dtype=np.float64))
    ncol, kdim = cos_coef.shape
    j = np.arange(N, dtype=np.int64)
    k = np.arange(kdim, dtype=np.int64)
    ph = 2.0 * np.pi * ((k[:, None] * j[None, :]) % N) / N
    out = cos_coef @ np.cos(ph)
    if sin_coef is not None:
        out = out + np.atleast_2d(np.asarray(sin_coef, dtype=np.float64)) @ np.sin(ph)
    return np.ascontiguousarray(out)


@dataclass
class Case:
    """One workload: base surface, base potential, and the (deta, dphi) column batch."""
    name: str
    N: int
    h: float
    g: float = 1.0
    prec: str = "f64"                      # "f64" | "dd"
    eta: np.ndarray | None = None          # (N,)
    phi0: np.ndarray | None = None         # (N,)
    deta: np.ndarray | None = None         # (nrhs, N)
    dphi: np.ndarray | None = None         # (nrhs, N)
    eta_lo: np.ndarray | None = None       # dd low words (None => zeros)
    phi0_lo: np.ndarray | None = None
    deta_lo: np.ndarray | None = None
    dphi_lo: np.ndarray | None = None
    meta: dict = field(default_factory=dict)

    @property
    def nrhs(self) -> int:
        return 0 if self.dphi is None else self.dphi.shape[0]


def fourier_unit_columns(N: int, kmax: int, pattern: str = "eta_phi") -> tuple[np.ndarray, np.ndarray]:
    """Jacobian-style unit perturbations of one Fourier coefficient each (
    SURVEY.md §8(c)-A11).  pattern "eta_phi": col 2k-2 = (2cos k a, 0), col 2k-1 = (0, 2cos k a).
    pattern "phi_only" (config 5): col 2k-2: dphi = 2cos k a, col 2k-1: dphi = 2sin k a, deta the
    same with cos<->sin."""
    a = grid(N)
    j = np.arange(N, dtype=np.int64)
    deta = np.zeros((2 * kmax, N))
    dphi = np.zeros((2 * kmax, N))
    for k in range(1, kmax + 1):
        ph = 2.0 * np.pi * ((k * j) % N) / N
        c, s = 2.0 * np.cos(ph), 2.0 * np.sin(ph)
        if pattern == "eta_phi":
            deta[2 * k - 2] = c
            dphi[2 * k - 1] = c
        else:
            dphi[2 * k - 2] = c
            deta[2 * k - 2] = s
            dphi[2 * k - 1] = s
            deta[2 * k - 1] = c
    del a
    return deta, dphi


def config1() -> Case:
    """Config 1: N=64, h=1, single DtN evaluation, 1 RHS."""
    seed, N = SEED_BASE + 1, 64
    k = np.arange(0, 9)
    dec = np.exp(-k.astype(float))
    a = np.zeros(9); b = np.zeros(9); c = np.zeros(9)
    a[1:] = 0.05 * normals(seed, 0, 8) * dec[1:]
    b[1:] = 0.1 * normals(seed, 1, 8) * dec[1:]
    c[1:] = 0.1 * normals(seed, 2, 8) * dec[1:]
    eta = synth(N, a)[0]
    phi = synth(N, b, c)[0]
    return Case("cfg1", N, 1.0, eta=eta, phi0=phi, deta=np.zeros((1, N)), dphi=phi[None, :].copy())


def config1_flat() -> Case:
    """Config 1 flat-surface check: eta=0, phi=cos(3 alpha) -> 3 tanh(3) cos(3 alpha) (4.34)."""
    N = 64
    a = np.zeros(4); a[3] = 1.0
    phi = synth(N, a)[0]
    return Case("cfg1_flat", N, 1.0, eta=np.zeros(N), phi0=phi, deta=np.zeros((1, N)), dphi=phi[None, :].copy())


def config2() -> Case:
    """Config 2: N=256 standing wave started at rest; meta has dt, nsteps for one linear period."""
    seed, N = SEED_BASE + 2, 256
    a = np.zeros(17)
    a[1] = 0.1
    kk = np.arange(2, 17)
    a[2:] = 0.01 * normals(seed, 0, 15) * np.exp(-kk.astype(float))
    eta = synth(N, a)[0]
    T = 2.0 * math.pi / math.sqrt(math.tanh(1.0))
    return Case("cfg2", N, 1.0, eta=eta, phi0=np.zeros(N), meta={"T": T, "nsteps": 256, "dt": T / 256})


def _family_surface(seed: int, N: int, amp1: float, kmax: int = 64):
    a = np.zeros(kmax + 1)
    a[1] = amp1
    kk = np.arange(2, kmax + 1)
    a[2:] = 0.01 * normals(seed, 0, kmax - 1) * np.exp(-kk / 8.0)
    b = np.zeros(kmax + 1)
    b[1] = 0.1
    ko = np.arange(3, kmax, 2)
    b[3:kmax:2] = 0.01 * normals(seed, 1, len(ko)) * np.exp(-ko / 8.0)
    return a, b


def config3(N: int = 512, ncols: int = 256, amp1: float = 0.2, variant: int = 0) -> Case:
    """Config 3 (N=512, 256 columns) and, with N=2048, ncols=512, the fp64 metric point.  amp1: amplitude of the cos(alpha)
    mode of the surface; variant > 0: another draw of the seeded modes (seed + 1000 variant) for the multi-seed parity runs."""
    seed = SEED_BASE + 3 + 1000 * variant
    a, b = _family_surface(seed, N, amp1)
    eta = synth(N, a)[0]
    phi0 = synth(N, b)[0]
    deta, dphi = fourier_unit_columns(N, ncols // 2, "eta_phi")
    return Case(f"cfg3_N{N}", N, 1.0, eta=eta, phi0=phi0, deta=deta, dphi=dphi)


def config4(N: int = 512, ncols: int = 128) -> Case:
    """Config 4 (double-double): 0.4 cos(alpha) family, seeded smooth columns, hi/lo pairs."""
    seed = SEED_BASE + 4
    a, b = _family_surface(seed, N, 0.4)
    eta_hi, eta_lo = synth_dd(N, a)
    phi_hi, phi_lo = synth_dd(N, b)
    kmax = 64
    dec = np.exp(-np.arange(kmax + 1) / 8.0)
    ce = np.zeros((ncols, kmax + 1)); se = np.zeros((ncols, kmax + 1))
    cp = np.zeros((ncols, kmax + 1)); sp = np.zeros((ncols, kmax + 1))
    for c in range(ncols):
        ne = normals(seed, 10 + 2 * c, kmax) * dec[1:]
        npv = normals(seed, 11 + 2 * c, kmax) * dec[1:]
        if c % 2 == 0:
            ce[c, 1:] = ne; cp[c, 1:] = npv
        else:
            se[c, 1:] = ne; sp[c, 1:] = npv
    dehi, delo = synth_dd(N, ce, se)
    dphi_hi, dphi_lo = synth_dd(N, cp, sp)
    return Case(f"cfg4_N{N}", N, 1.0, prec="dd", eta=eta_hi[0], eta_lo=eta_lo[0], phi0=phi_hi[0], phi0_lo=phi_lo[0],
                deta=dehi, deta_lo=delo, dphi=dphi_hi, dphi_lo=dphi_lo)


def config5(N: int = 4096, ncols: int = 512) -> Case:
    """Config 5: shallow water h=0.05, two sech^2 humps (periodised, +-1% seeded), phi0 = 0, dphi-type columns."""
    seed = SEED_BASE + 5
    xi = 2.0 * uniforms(seed, 0, 4) - 1.0
    al = grid(N)
    eta = np.zeros(N)
    for i, c in enumerate((0.5 * math.pi, 1.5 * math.pi)):
        amp = 0.02 * (1.0 + 0.01 * xi[2 * i])
        w = 0.3 * (1.0 + 0.01 * xi[2 * i + 1])
        for m in range(-2, 3):
            eta += amp / np.cosh((al - c - 2.0 * math.pi * m) / w) ** 2
    eta -= eta.mean()
    deta, dphi = fourier_unit_columns(N, ncols // 2, "phi_only")
    return Case(f"cfg5_N{N}", N, 0.05, eta=eta, phi0=np.zeros(N), deta=deta, dphi=dphi)


def metric_point(ncols: int = 512, amp1: float = 0.2, variant: int = 0) -> Case:
    """BASELINE.json metric point: N=2048, config-3 family, fp64."""
    c = config3(2048, ncols, amp1, variant)
    c.name = f"metric_N2048_nrhs{ncols}"
    return c


def metric_point_dd(ncols: int = 128, N: int = 2048) -> Case:
    c = config4(N, ncols)
    c.name = f"metric_dd_N{N}_nrhs{ncols}"
    return c
