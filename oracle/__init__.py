"""ctypes front end of the CPU oracle (oracle/sww_oracle.c) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
It shares nothing with the CUDA path.  Three builds of the one C source: "f64" (double), "ld" (x87 long
double, the oracle for the fp64 bar) and "q" (__float128, the oracle for the double-double bar).

Every quantity goes in and comes out as float64 `hi` (+ optional `lo`) arrays, value = hi + lo.
Batches are C-contiguous (nrhs, N) arrays (= column-major N x nrhs).  K, G come back row-major (N, N).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sww_oracle.c"
_FLAGS = {"f64": ["-DORC_F64"], "ld": ["-DORC_LD"], "q": ["-DORC_Q"]}
_LIBS: dict[str, ctypes.CDLL] = {}

MUL_D, MUL_H, MUL_ABSD, MUL_FILTER, MUL_P, MUL_PFILTER = 1, 2, 3, 4, 5, 6


def lib_path(prec: str) -> Path:
    return _HERE / f"liborc_{prec}.so"


def build(force: bool = False) -> None:
    """Compile the three oracle libraries with gcc (no GPU involved)."""
    for prec, defs in _FLAGS.items():
        out = lib_path(prec)
        if not force and out.exists() and out.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", *defs, str(_SRC), "-o", str(out), "-lm"]
        if prec != "f64":
            cmd.append("-lquadmath")
        subprocess.run(cmd, check=True)


def _lib(prec: str) -> ctypes.CDLL:
    if prec not in _LIBS:
        build()
        _LIBS[prec] = ctypes.CDLL(str(lib_path(prec)))
    return _LIBS[prec]


_DP = ctypes.POINTER(ctypes.c_double)


def _split(x, shape=None):
    """array | (hi, lo) -> contiguous float64 hi, lo-or-None"""
    if isinstance(x, tuple):
        hi, lo = x
    else:
        hi, lo = x, None
    hi = np.ascontiguousarray(hi, dtype=np.float64)
    if lo is not None:
        lo = np.ascontiguousarray(lo, dtype=np.float64)
        assert lo.shape == hi.shape
    if shape is not None:
        assert hi.shape == shape, (hi.shape, shape)
    return hi, lo


def _p(a):
    return None if a is None else a.ctypes.data_as(_DP)


class OracleError(RuntimeError):
    pass


def _check(rc: int, what: str):
    if rc != 0:
        raise OracleError(f"{what}: oracle status {rc}")


class Oracle:
    def __init__(self, prec: str = "ld"):
        assert prec in _FLAGS
        self.prec = prec
        self.lib = _lib(prec)
        self._f = lambda name: getattr(self.lib, f"orc_{prec}_{name}")

    def set_num_threads(self, n: int) -> None:
        """OpenMP threads of the following calls of this build (small N: 1 is fastest)"""
        self._f("set_num_threads")(ctypes.c_int(int(n)))

    def num_threads(self) -> int:
        return int(self._f("num_threads")())

    def sizeof_real(self) -> int:
        return int(self._f("sizeof_real")())

    def set_mesh(self, rho: float = 1.0, where: int = 0) -> None:
        """Mesh refinement (2.10) for the following calls of this build: rho in (0, 1] (1 = uniform), where = 0 refines near
        x = pi, 1 near x = 0.  Reset with set_mesh() when done."""
        _check(self._f("set_mesh")(ctypes.c_double(rho), ctypes.c_int(where)), "set_mesh")

    def mesh_tables(self, N: int):
        """-> xp = xi - alpha, E = xi', E1 = xi'' (each (hi, lo)) of the current mesh setting at alpha_j = 2 pi j / N"""
        o = [(np.empty(N), np.empty(N)) for _ in range(3)]
        _check(self._f("mesh_tables")(ctypes.c_int(N), _p(o[0][0]), _p(o[0][1]), _p(o[1][0]), _p(o[1][1]), _p(o[2][0]), _p(o[2][1])), "mesh_tables")
        return tuple(o)

    def respace(self, f, old, new):
        """Values on the mesh `new` = (M, rho, where) of the functions stored on the mesh `old`; f: (ncols, M_old)"""
        fhi, flo = _split(f)
        one = fhi.ndim == 1
        if one:
            fhi = fhi[None, :]
            flo = None if flo is None else flo[None, :]
        Mo, Mn = int(old[0]), int(new[0])
        ncols = fhi.shape[0]
        assert fhi.shape == (ncols, Mo)
        ohi, olo = np.empty((ncols, Mn)), np.empty((ncols, Mn))
        _check(self._f("respace")(ctypes.c_int(Mo), ctypes.c_double(old[1]), ctypes.c_int(old[2]), ctypes.c_int(Mn), ctypes.c_double(new[1]),
                                  ctypes.c_int(new[2]), ctypes.c_int(ncols), _p(fhi), _p(flo), _p(ohi), _p(olo)), "respace")
        return (ohi[0], olo[0]) if one else (ohi, olo)

    def multiplier(self, which: int, f):
        hi, lo = _split(f)
        N = hi.shape[-1]
        assert hi.ndim == 1
        ohi, olo = np.empty(N), np.empty(N)
        _check(self._f("multiplier")(ctypes.c_int(N), ctypes.c_int(which), _p(hi), _p(lo), _p(ohi), _p(olo)), "multiplier")
        return ohi, olo

    def assemble(self, eta, h: float):
        ehi, elo = _split(eta)
        N = ehi.shape[0]
        out = {k: (np.empty(s), np.empty(s)) for k, s in (("K", (N, N)), ("G", (N, N)), ("d1", (N,)), ("d2", (N,)))}
        _check(self._f("assemble")(ctypes.c_int(N), ctypes.c_double(h), _p(ehi), _p(elo),
                                   _p(out["K"][0]), _p(out["K"][1]), _p(out["G"][0]), _p(out["G"][1]),
                                   _p(out["d1"][0]), _p(out["d1"][1]), _p(out["d2"][0]), _p(out["d2"][1])), "assemble")
        return out

    def dtn_apply(self, eta, h: float, phi, want_mu: bool = False):
        ehi, elo = _split(eta)
        N = ehi.shape[0]
        phi_hi, phi_lo = _split(phi)
        if phi_hi.ndim == 1:
            phi_hi = phi_hi[None, :]
            phi_lo = None if phi_lo is None else phi_lo[None, :]
        nrhs = phi_hi.shape[0]
        assert phi_hi.shape == (nrhs, N)
        ohi, olo = np.empty((nrhs, N)), np.empty((nrhs, N))
        mhi = np.empty((nrhs, N)) if want_mu else None
        mlo = np.empty((nrhs, N)) if want_mu else None
        _check(self._f("dtn_apply")(ctypes.c_int(N), ctypes.c_double(h), _p(ehi), _p(elo), ctypes.c_int(nrhs),
                                    _p(phi_hi), _p(phi_lo), _p(ohi), _p(olo), _p(mhi), _p(mlo)), "dtn_apply")
        return ((ohi, olo), (mhi, mlo)) if want_mu else (ohi, olo)

    def dtn_linearized(self, eta, h: float, phi0, deta, dphi, want_base: bool = False):
        ehi, elo = _split(eta)
        N = ehi.shape[0]
        p0hi, p0lo = _split(phi0, (N,))
        dehi, delo = _split(deta)
        dphi_hi, dphi_lo = _split(dphi)
        nrhs = dehi.shape[0]
        assert dehi.shape == (nrhs, N) and dphi_hi.shape == (nrhs, N)
        ohi, olo = np.empty((nrhs, N)), np.empty((nrhs, N))
        bhi, blo = np.empty((4, N)), np.empty((4, N))
        _check(self._f("dtn_linearized")(ctypes.c_int(N), ctypes.c_double(h), _p(ehi), _p(elo), _p(p0hi), _p(p0lo),
                                         ctypes.c_int(nrhs), _p(dehi), _p(delo), _p(dphi_hi), _p(dphi_lo),
                                         _p(ohi), _p(olo), _p(bhi), _p(blo)), "dtn_linearized")
        if want_base:
            base = {k: (bhi[i], blo[i]) for i, k in enumerate(("dphi0", "W0", "u", "v"))}
            return (ohi, olo), base
        return ohi, olo

    def rhs(self, eta, phi, h: float, g: float = 1.0, deta=None, dphi=None, filter: bool = True, sigma: float = 0.0):
        """-> dict eta_t, phi_t, deta_t, dphi_t (each (hi, lo)), energy (hi, lo)"""
        ehi, elo = _split(eta)
        N = ehi.shape[0]
        phi_hi, phi_lo = _split(phi, (N,))
        if deta is None:
            ncols, dehi, delo, dphi_hi, dphi_lo = 0, None, None, None, None
        else:
            dehi, delo = _split(deta)
            dphi_hi, dphi_lo = _split(dphi)
            ncols = dehi.shape[0]
        L = 2 * N * (1 + ncols)
        ohi, olo, E = np.empty(L), np.empty(L), np.empty(2)
        _check(self._f("rhs")(ctypes.c_int(N), ctypes.c_double(h), ctypes.c_double(g), ctypes.c_double(sigma), ctypes.c_int(int(filter)),
                              _p(ehi), _p(elo), _p(phi_hi), _p(phi_lo), ctypes.c_int(ncols),
                              _p(dehi), _p(delo), _p(dphi_hi), _p(dphi_lo), _p(ohi), _p(olo), _p(E)), "rhs")
        cut = lambda a, o, n, shape: a[o:o + n].reshape(shape)
        nc = N * ncols
        res = {
            "eta_t": (cut(ohi, 0, N, (N,)), cut(olo, 0, N, (N,))),
            "phi_t": (cut(ohi, N, N, (N,)), cut(olo, N, N, (N,))),
            "deta_t": (cut(ohi, 2 * N, nc, (ncols, N)), cut(olo, 2 * N, nc, (ncols, N))),
            "dphi_t": (cut(ohi, 2 * N + nc, nc, (ncols, N)), cut(olo, 2 * N + nc, nc, (ncols, N))),
            "energy": (E[0], E[1]),
        }
        return res

    def adjoint_rhs(self, eta, phi, h: float, g: float, eta_t, phi_t, sigma: float = 0.0):
        """(B.6): -> dict eta_s, phi_s (each (hi, lo), shape (ncols, N)) for the adjoint vectors (eta_t, phi_t) at the state (eta, phi)"""
        ehi, elo = _split(eta)
        N = ehi.shape[0]
        phi_hi, phi_lo = _split(phi, (N,))
        ethi, etlo = _split(eta_t)
        pthi, ptlo = _split(phi_t)
        ncols = ethi.shape[0]
        nc = N * ncols
        ohi, olo = np.empty(2 * nc), np.empty(2 * nc)
        _check(self._f("adjoint_rhs")(ctypes.c_int(N), ctypes.c_double(h), ctypes.c_double(g), ctypes.c_double(sigma), _p(ehi), _p(elo),
                                      _p(phi_hi), _p(phi_lo), ctypes.c_int(ncols), _p(ethi), _p(etlo), _p(pthi), _p(ptlo), _p(ohi), _p(olo)),
               "adjoint_rhs")
        return {"eta_s": (ohi[:nc].reshape(ncols, N), olo[:nc].reshape(ncols, N)),
                "phi_s": (ohi[nc:].reshape(ncols, N), olo[nc:].reshape(ncols, N))}

    def rk_tableau(self):
        a = (np.empty((11, 11)), np.empty((11, 11)))
        b = (np.empty(11), np.empty(11))
        c = (np.empty(11), np.empty(11))
        _check(self._f("rk_tableau")(_p(a[0]), _p(a[1]), _p(b[0]), _p(b[1]), _p(c[0]), _p(c[1])), "rk_tableau")
        return a, b, c

    def rk_linear_test(self, lam: complex, dt: float, nsteps: int):
        yh, yl = np.empty(2), np.empty(2)
        _check(self._f("rk_linear_test")(ctypes.c_double(lam.real), ctypes.c_double(lam.imag), ctypes.c_double(dt),
                                         ctypes.c_int(nsteps), _p(yh), _p(yl)), "rk_linear_test")
        return yh, yl

    def sdc_tables(self, s: int = 8):
        """Radau IIa nodes c (s) and the integration matrix S (s x s), each (hi, lo)"""
        c = (np.empty(s), np.empty(s))
        S = (np.empty((s, s)), np.empty((s, s)))
        _check(self._f("sdc_tables")(ctypes.c_int(s), _p(c[0]), _p(c[1]), _p(S[0]), _p(S[1])), "sdc_tables")
        return c, S

    def sdc_linear_test(self, lam: complex, dt: float, nsteps: int):
        yh, yl = np.empty(2), np.empty(2)
        _check(self._f("sdc_linear_test")(ctypes.c_double(lam.real), ctypes.c_double(lam.imag), ctypes.c_double(dt),
                                          ctypes.c_int(nsteps), _p(yh), _p(yl)), "sdc_linear_test")
        return yh, yl

    def rk_riccati_test(self, dt: float, nsteps: int):
        yh, yl = np.empty(1), np.empty(1)
        _check(self._f("rk_riccati_test")(ctypes.c_double(dt), ctypes.c_int(nsteps), _p(yh), _p(yl)), "rk_riccati_test")
        return yh[0], yl[0]

    def rk_advance(self, eta, phi, h: float, g: float, dt: float, nsteps: int, deta=None, dphi=None,
                   filter: bool = True, want_energy: bool = False, sigma: float = 0.0, method: str = "rk8"):
        """-> dict eta, phi, deta, dphi (each (hi, lo)), energies ((hi, lo) arrays of nsteps+1) or None.
        method: "rk8" (the 11-stage order-8 scheme, R6) or "sdc15" (spectral deferred correction on 8 Radau IIa nodes, R15)"""
        ehi, elo = _split(eta)
        N = ehi.shape[0]
        phi_hi, phi_lo = _split(phi, (N,))
        ehi, phi_hi = ehi.copy(), phi_hi.copy()
        elo = np.zeros(N) if elo is None else elo.copy()
        phi_lo = np.zeros(N) if phi_lo is None else phi_lo.copy()
        if deta is None:
            ncols, dehi, delo, dphi_hi, dphi_lo = 0, None, None, None, None
        else:
            dehi, delo = _split(deta)
            dphi_hi, dphi_lo = _split(dphi)
            ncols = dehi.shape[0]
            dehi, dphi_hi = dehi.copy(), dphi_hi.copy()
            delo = np.zeros_like(dehi) if delo is None else delo.copy()
            dphi_lo = np.zeros_like(dphi_hi) if dphi_lo is None else dphi_lo.copy()
        en = np.empty(2 * (nsteps + 1)) if want_energy else None
        _check(self._f({"rk8": "rk_advance", "sdc15": "sdc_advance"}[method])(ctypes.c_int(N), ctypes.c_double(h), ctypes.c_double(g), ctypes.c_double(sigma), ctypes.c_int(int(filter)),
                                     ctypes.c_double(dt), ctypes.c_int(nsteps), _p(ehi), _p(elo), _p(phi_hi), _p(phi_lo),
                                     ctypes.c_int(ncols), _p(dehi), _p(delo), _p(dphi_hi), _p(dphi_lo), _p(en)), "rk_advance")
        return {"eta": (ehi, elo), "phi": (phi_hi, phi_lo), "deta": (dehi, delo), "dphi": (dphi_hi, dphi_lo),
                "energies": None if en is None else (en[:nsteps + 1], en[nsteps + 1:])}


def set_threads(n: int) -> None:
    os.environ["OMP_NUM_THREADS"] = str(n)
