"""ctypes binding of include/sww.h.  Argument marshalling only (see the package docstring)."""
from __future__ import annotations

import ctypes
import math
from pathlib import Path

import torch

F64, DD = 0, 1
_HERE = Path(__file__).resolve().parent
_LIB = None

# every symbol include/sww.h declares (tests check the library exports each of them)
EXPORTS = [
    "sww_dtn_setup", "sww_dtn_refactor", "sww_dtn_apply", "sww_dtn_set_base", "sww_dtn_linearized_apply", "sww_dtn_get",
    "sww_dtn_status", "sww_dtn_destroy", "sww_state_create", "sww_rk_advance", "sww_state_read", "sww_state_energy",
    "sww_state_destroy", "sww_strerror", "sww_last_cuda_error", "sww_launch_count", "sww_probe_fp64_peak",
    "sww_dtn_linearized_host", "sww_host_cache_clear", "sww_timing_enable", "sww_timing_read",
    "sww_shooter_create", "sww_shoot", "sww_shooter_destroy", "sww_shoot_residual", "sww_shooter_dims", "sww_lm_minimize", "sww_lm_shoot",
    "sww_state_set_sigma", "sww_shooter_set_sigma", "sww_sdc_advance", "sww_dtn_adjoint_rhs", "sww_shooter_set_method",
    "sww_dtn_set_mesh", "sww_mesh_points", "sww_state_set_mesh", "sww_state_respace", "sww_shooter_set_segments", "sww_shoot_gradient", "sww_respace_noalloc",
]


class LmOptions(ctypes.Structure):
    _fields_ = [("f_tol", ctypes.c_double), ("g_tol", ctypes.c_double), ("df_tol", ctypes.c_double), ("delta0", ctypes.c_double),
                ("lambda_tol", ctypes.c_double), ("max_stepsJ", ctypes.c_int), ("max_iter", ctypes.c_int)]


class LmReport(ctypes.Structure):
    _fields_ = [("f", ctypes.c_double), ("delta", ctypes.c_double), ("iterations", ctypes.c_int), ("residual_evals", ctypes.c_int),
                ("jacobian_evals", ctypes.c_int), ("status", ctypes.c_int)]


LM_FUN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                          ctypes.POINTER(ctypes.c_double))


def _lm_options(f_tol=1e-26, g_tol=1e-13, df_tol=1e-5, delta0=1.0, lambda_tol=1e-12, max_stepsJ=10, max_iter=100):
    return LmOptions(f_tol, g_tol, df_tol, delta0, lambda_tol, max_stepsJ, max_iter)


def _lm_report(rep: LmReport) -> dict:
    return {k: getattr(rep, k) for k, _ in LmReport._fields_}


class SwwError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        msg = lib().sww_strerror(status).decode()
        if status in (-3, -7):
            msg += ": " + lib().sww_last_cuda_error().decode()
        super().__init__(f"{what}: {msg} (status {status})")


def lib_path() -> Path:
    return _HERE / "libsww.so"


def lib() -> ctypes.CDLL:
    """Load libsww.so (built in-tree by paper_1210_5672_b200.build).  Fails loudly when it is missing."""
    global _LIB
    if _LIB is None:
        p = lib_path()
        if not p.exists():
            raise ImportError(f"{p} is missing: run `python -m paper_1210_5672_b200.build` (there is no fallback path)")
        L = ctypes.CDLL(str(p))
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.sww_dtn_setup.argtypes = [vp, ci, cd, ci, vp, ctypes.POINTER(vp)]
        L.sww_dtn_refactor.argtypes = [vp, vp]
        L.sww_dtn_apply.argtypes = [vp, vp, ci, vp]
        L.sww_dtn_set_base.argtypes = [vp, vp]
        L.sww_dtn_linearized_apply.argtypes = [vp, vp, vp, ci, vp]
        L.sww_dtn_get.argtypes = [vp, ci, vp]
        L.sww_dtn_adjoint_rhs.argtypes = [vp, vp, vp, ci, cd, cd, vp, vp]
        L.sww_dtn_status.argtypes = [vp]
        L.sww_dtn_destroy.argtypes = [vp]
        L.sww_state_create.argtypes = [ci, cd, cd, ci, ci, vp, vp, vp, vp, ctypes.c_uint, vp, ctypes.POINTER(vp)]
        L.sww_rk_advance.argtypes = [vp, cd, ci]
        L.sww_sdc_advance.argtypes = [vp, cd, ci]
        L.sww_state_read.argtypes = [vp, vp, vp, vp, vp, ctypes.POINTER(cd)]
        L.sww_state_energy.argtypes = [vp, ctypes.POINTER(cd)]
        L.sww_state_destroy.argtypes = [vp]
        L.sww_strerror.argtypes = [ci]
        L.sww_strerror.restype = ctypes.c_char_p
        L.sww_last_cuda_error.restype = ctypes.c_char_p
        L.sww_launch_count.restype = ctypes.c_ulonglong
        L.sww_probe_fp64_peak.argtypes = [ci, ctypes.POINTER(cd)]
        L.sww_dtn_linearized_host.argtypes = [vp, vp, vp, vp, vp, ci, cd, ci, ci]
        L.sww_shooter_create.argtypes = [ci, ci, cd, cd, ci, ctypes.c_uint, vp, ctypes.POINTER(vp)]
        L.sww_shoot.argtypes = [vp, ctypes.POINTER(cd), ci, vp, vp, vp, vp]
        L.sww_shooter_destroy.argtypes = [vp]
        L.sww_state_set_sigma.argtypes = [vp, cd]
        L.sww_shooter_set_sigma.argtypes = [vp, cd]
        L.sww_shooter_set_method.argtypes = [vp, ci]
        L.sww_shoot_residual.argtypes = [vp, ctypes.POINTER(cd), ci, vp]
        L.sww_shooter_dims.argtypes = [vp, ctypes.POINTER(ci), ctypes.POINTER(ci), ctypes.POINTER(ci)]
        L.sww_lm_minimize.argtypes = [LM_FUN, vp, ci, ci, ctypes.POINTER(cd), ctypes.POINTER(ci), ctypes.POINTER(LmOptions), ctypes.POINTER(LmReport)]
        L.sww_lm_shoot.argtypes = [vp, ctypes.POINTER(cd), ctypes.POINTER(ci), ci, ctypes.POINTER(LmOptions), ctypes.POINTER(LmReport)]
        L.sww_dtn_set_mesh.argtypes = [vp, cd, ci]
        L.sww_mesh_points.argtypes = [ci, cd, ci, ctypes.POINTER(cd)]
        L.sww_state_set_mesh.argtypes = [vp, cd, ci]
        L.sww_state_respace.argtypes = [vp, vp]
        L.sww_respace_noalloc.argtypes = [ci, cd, ci, ci, cd, ci, ci, vp, vp, vp]
        L.sww_shoot_gradient.argtypes = [vp, ctypes.POINTER(cd), ci, ctypes.POINTER(cd), ctypes.POINTER(cd)]
        L.sww_shooter_set_segments.argtypes = [vp, ci, ctypes.POINTER(ci), ctypes.POINTER(cd), ctypes.POINTER(cd), ctypes.POINTER(ci), ctypes.POINTER(ci)]
        L.sww_timing_enable.argtypes = [ci]
        L.sww_timing_read.argtypes = [ctypes.POINTER(cd), ctypes.POINTER(ctypes.c_ulonglong), ci]
        _LIB = L
    return _LIB


def _check(rc: int, what: str):
    if rc != 0:
        raise SwwError(rc, what)


def _require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1210_5672_b200 needs a CUDA device: there is no CPU path")


def _dev(t: torch.Tensor, n: int, what: str) -> int:
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n):
        raise ValueError(f"{what}: expected a contiguous CUDA float64 tensor of {n} elements, got {tuple(t.shape)} {t.dtype} {t.device}")
    return t.data_ptr()


def dd_pack(hi, lo, device="cuda") -> torch.Tensor:
    """(hi, lo) arrays of equal shape -> planar dd tensor of shape (2, *shape) on the device"""
    hi = torch.as_tensor(hi, dtype=torch.float64)
    lo = torch.zeros_like(hi) if lo is None else torch.as_tensor(lo, dtype=torch.float64)
    return torch.stack([hi, lo]).contiguous().to(device)


def dd_unpack(t: torch.Tensor):
    c = t.detach().cpu().numpy()
    return c[0], c[1]


def launch_count() -> int:
    return int(lib().sww_launch_count())


KERNEL_CLASSES = ("assembly", "lu", "gemm_dmma", "fft", "dd_gemm", "other", "trsm", "trsv")


def timing_enable(on: bool):
    _check(lib().sww_timing_enable(1 if on else 0), "sww_timing_enable")


def timing_read() -> dict:
    """-> {class: (milliseconds, launches)} since the previous read"""
    n = len(KERNEL_CLASSES)
    ms = (ctypes.c_double * n)()
    cnt = (ctypes.c_ulonglong * n)()
    _check(lib().sww_timing_read(ms, cnt, n), "sww_timing_read")
    return {k: (ms[i], int(cnt[i])) for i, k in enumerate(KERNEL_CLASSES)}


def probe_fp64_peak(which: int) -> float:
    """which: 0 = DFMA loop, 1 = DMMA.8x8x4 loop.  Returns FLOP/s."""
    _require_cuda()
    out = ctypes.c_double(0.0)
    _check(lib().sww_probe_fp64_peak(which, ctypes.byref(out)), "sww_probe_fp64_peak")
    return out.value


class DtN:
    """One surface: sww_dtn_setup / apply / set_base / linearized_apply.  Tensors are CUDA float64; batches are (nrhs, N)
    C-contiguous (= column-major N x nrhs); dd quantities are planar (2, ...) tensors (hi plane, lo plane)."""

    def __init__(self, eta: torch.Tensor, h: float, prec: int = F64, stream: torch.cuda.Stream | None = None):
        _require_cuda()
        self.prec = prec
        self.mul = 2 if prec == DD else 1
        self.N = eta.numel() // self.mul
        self.h = float(h)
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        h_ = ctypes.c_void_p()
        _check(lib().sww_dtn_setup(_dev(eta, self.N * self.mul, "eta"), self.N, self.h, prec, self._stream.cuda_stream, ctypes.byref(h_)),
               "sww_dtn_setup")
        self._h = h_

    def _shape(self, nrhs):
        return (2, nrhs, self.N) if self.prec == DD else (nrhs, self.N)

    def refactor(self, eta: torch.Tensor):
        _check(lib().sww_dtn_refactor(self._h, _dev(eta, self.N * self.mul, "eta")), "sww_dtn_refactor")

    def set_mesh(self, rho: float, where: int = 0):
        """sww_dtn_set_mesh: the refined mesh (2.10); follow with refactor(eta) (values at the points mesh_points(N, rho, where))"""
        _check(lib().sww_dtn_set_mesh(self._h, float(rho), int(where)), "sww_dtn_set_mesh")

    def apply(self, phi: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        nrhs = phi.numel() // (self.N * self.mul)
        if out is None:
            out = torch.empty_like(phi)
        _check(lib().sww_dtn_apply(self._h, _dev(phi, nrhs * self.N * self.mul, "phi"), nrhs, _dev(out, phi.numel(), "out")), "sww_dtn_apply")
        return out

    def set_base(self, phi0: torch.Tensor):
        _check(lib().sww_dtn_set_base(self._h, _dev(phi0, self.N * self.mul, "phi0")), "sww_dtn_set_base")

    def linearized_apply(self, deta: torch.Tensor, dphi: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        nrhs = dphi.numel() // (self.N * self.mul)
        if out is None:
            out = torch.empty_like(dphi)
        n = nrhs * self.N * self.mul
        _check(lib().sww_dtn_linearized_apply(self._h, _dev(deta, n, "deta"), _dev(dphi, n, "dphi"), nrhs, _dev(out, n, "out")),
               "sww_dtn_linearized_apply")
        return out

    def adjoint_rhs(self, eta_t: torch.Tensor, phi_t: torch.Tensor, g: float = 1.0, sigma: float = 0.0):
        """(B.6): -> (eta_s, phi_s) for the adjoint vectors (eta_t, phi_t), each (nrhs, N) (double-double: (2, nrhs, N)); base state set"""
        nrhs = phi_t.numel() // (self.N * self.mul)
        n = nrhs * self.N * self.mul
        eta_s, phi_s = torch.empty_like(eta_t), torch.empty_like(phi_t)
        _check(lib().sww_dtn_adjoint_rhs(self._h, _dev(eta_t, n, "eta_t"), _dev(phi_t, n, "phi_t"), nrhs, float(g), float(sigma),
                                         _dev(eta_s, n, "eta_s"), _dev(phi_s, n, "phi_s")), "sww_dtn_adjoint_rhs")
        return eta_s, phi_s

    _WHICH = {"K": 0, "G": 1, "d1": 2, "d2": 3, "dphi0": 4, "W0": 5, "u": 6, "v": 7, "LU": 8}

    def get(self, name: str) -> torch.Tensor:
        """K, G, LU: (N, N) tensors indexed [j, i] (column-major storage: entry (i, j) of the matrix is t[j, i])."""
        which = self._WHICH[name]
        N = self.N
        if name in ("K", "G"):
            shape = (2, N, N) if self.prec == DD else (N, N)
        elif name == "LU":
            shape = (N, N)
        else:
            shape = (2, N) if self.prec == DD else (N,)
        t = torch.empty(shape, dtype=torch.float64, device="cuda")
        _check(lib().sww_dtn_get(self._h, which, t.data_ptr()), "sww_dtn_get")
        return t

    def status(self) -> int:
        return int(lib().sww_dtn_status(self._h))

    def check(self):
        _check(self.status(), "sww_dtn_status")

    def close(self):
        if getattr(self, "_h", None):
            lib().sww_dtn_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class State:
    """Time-stepper state: sww_state_create / sww_rk_advance / sww_state_read / sww_state_energy."""

    def __init__(self, eta, phi, h: float, g: float = 1.0, prec: int = F64, deta=None, dphi=None, filter: bool = True,
                 stream: torch.cuda.Stream | None = None):
        _require_cuda()
        self.prec = prec
        self.mul = 2 if prec == DD else 1
        self.N = eta.numel() // self.mul
        self.ncols = 0 if deta is None else deta.numel() // (self.N * self.mul)
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        h_ = ctypes.c_void_p()
        n1, nc = self.N * self.mul, self.N * self.mul * self.ncols
        _check(lib().sww_state_create(self.N, float(h), float(g), prec, self.ncols, _dev(eta, n1, "eta"), _dev(phi, n1, "phi"),
                                      None if deta is None else _dev(deta, nc, "deta"), None if dphi is None else _dev(dphi, nc, "dphi"),
                                      0 if filter else 1, self._stream.cuda_stream, ctypes.byref(h_)), "sww_state_create")
        self._h = h_

    def set_sigma(self, sigma: float):
        _check(lib().sww_state_set_sigma(self._h, float(sigma)), "sww_state_set_sigma")

    def set_mesh(self, rho: float, where: int = 0):
        _check(lib().sww_state_set_mesh(self._h, float(rho), int(where)), "sww_state_set_mesh")

    def respace_from(self, src: "State"):
        """sww_state_respace: this state <- src's, interpolated to this handle's mesh"""
        _check(lib().sww_state_respace(self._h, src._h), "sww_state_respace")

    def advance(self, dt: float, nsteps: int, method: str = "rk8"):
        """method: "rk8" (sww_rk_advance) or "sdc15" (sww_sdc_advance, the paper's quadruple-precision stepper)"""
        if method == "sdc15":
            _check(lib().sww_sdc_advance(self._h, float(dt), int(nsteps)), "sww_sdc_advance")
        else:
            _check(lib().sww_rk_advance(self._h, float(dt), int(nsteps)), "sww_rk_advance")

    def read(self):
        N, nc = self.N, self.ncols
        sh1 = (2, N) if self.prec == DD else (N,)
        shc = (2, nc, N) if self.prec == DD else (nc, N)
        eta = torch.empty(sh1, dtype=torch.float64, device="cuda")
        phi = torch.empty_like(eta)
        deta = torch.empty(shc, dtype=torch.float64, device="cuda") if nc else None
        dphi = torch.empty_like(deta) if nc else None
        t = ctypes.c_double(0.0)
        _check(lib().sww_state_read(self._h, eta.data_ptr(), phi.data_ptr(), deta.data_ptr() if nc else None,
                                    dphi.data_ptr() if nc else None, ctypes.byref(t)), "sww_state_read")
        return {"eta": eta, "phi": phi, "deta": deta, "dphi": dphi, "t": t.value}

    def energy(self):
        e = (ctypes.c_double * 2)()
        _check(lib().sww_state_energy(self._h, e), "sww_state_energy")
        return e[0], e[1]

    def close(self):
        if getattr(self, "_h", None):
            lib().sww_state_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Shooter:
    """The shooting map (3.15)-(3.17), (3.31): sww_shooter_create / sww_shoot.  c: n + 1 unknowns (c[0] = T)."""

    def __init__(self, N: int, n: int, h: float, g: float = 1.0, prec: int = F64, filter: bool = True,
                 stream: torch.cuda.Stream | None = None):
        _require_cuda()
        self.N, self.n, self.prec = int(N), int(n), prec
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        h_ = ctypes.c_void_p()
        _check(lib().sww_shooter_create(self.N, self.n, float(h), float(g), prec, 0 if filter else 1, self._stream.cuda_stream,
                                        ctypes.byref(h_)), "sww_shooter_create")
        self._h = h_
        self.m = self.N   # number of residuals (M of the last segment)

    def set_sigma(self, sigma: float):
        _check(lib().sww_shooter_set_sigma(self._h, float(sigma)), "sww_shooter_set_sigma")

    def set_segments(self, segments):
        """Mesh-refinement strategy of section 2.2: segments = [(M, theta, rho, where, nsteps), ...] with M_1 = N, rho_1 = 1 and
        sum(theta) = 1; [] returns to one uniform segment.  With segments the nsteps argument of shoot/residual/solve is ignored."""
        nu = len(segments)
        arr = lambda t, col: (t * max(nu, 1))(*[t(sg[col]) for sg in segments])
        _check(lib().sww_shooter_set_segments(self._h, nu, arr(ctypes.c_int, 0), arr(ctypes.c_double, 1), arr(ctypes.c_double, 2),
                                              arr(ctypes.c_int, 3), arr(ctypes.c_int, 4)), "sww_shooter_set_segments")
        self.m = int(segments[-1][0]) if nu else self.N

    def set_method(self, method: str):
        """"rk8" (default) or "sdc15" for the time stepping of every following shot"""
        _check(lib().sww_shooter_set_method(self._h, {"rk8": 0, "sdc15": 1}[method]), "sww_shooter_set_method")

    def shoot(self, c, nsteps: int, want_state: bool = False):
        """-> r (m), J (n + 1, m) [= column-major m x (n + 1)], m = N or the last segment's M; double-double: leading axis 2 (hi, lo)"""
        N, n = self.m, self.n
        cc = (ctypes.c_double * (n + 1))(*[float(x) for x in c])
        lead = (2,) if self.prec == DD else ()
        r = torch.empty(lead + (N,), dtype=torch.float64, device="cuda")
        J = torch.empty(lead + (n + 1, N), dtype=torch.float64, device="cuda")
        eta = torch.empty(lead + (N,), dtype=torch.float64, device="cuda") if want_state else None
        phi = torch.empty_like(eta) if want_state else None
        _check(lib().sww_shoot(self._h, cc, int(nsteps), r.data_ptr(), J.data_ptr(), eta.data_ptr() if want_state else None,
                               phi.data_ptr() if want_state else None), "sww_shoot")
        return (r, J, eta, phi) if want_state else (r, J)

    def residual(self, c, nsteps: int):
        cc = (ctypes.c_double * (self.n + 1))(*[float(x) for x in c])
        lead = (2,) if self.prec == DD else ()
        r = torch.empty(lead + (self.m,), dtype=torch.float64, device="cuda")
        _check(lib().sww_shoot_residual(self._h, cc, int(nsteps), r.data_ptr()), "sww_shoot_residual")
        return r

    def gradient(self, c, nsteps: int):
        """sww_shoot_gradient: (f, grad (numpy, n + 1)) by one backward solve of the adjoint system (section 3.2)"""
        import numpy as np
        cc = (ctypes.c_double * (self.n + 1))(*[float(x) for x in c])
        f = ctypes.c_double(0.0)
        g = (ctypes.c_double * (self.n + 1))()
        _check(lib().sww_shoot_gradient(self._h, cc, int(nsteps), ctypes.byref(f), g), "sww_shoot_gradient")
        return f.value, np.array(list(g))

    def solve(self, c, nsteps: int, fixed=None, **opts):
        """Levenberg-Marquardt with delayed Jacobian updates (Appendix C) on the shooting map: -> (c, report)"""
        n1 = self.n + 1
        cc = (ctypes.c_double * n1)(*[float(x) for x in c])
        fx = (ctypes.c_int * n1)(*([0] * n1 if fixed is None else [int(bool(x)) for x in fixed]))
        opt, rep = _lm_options(**opts), LmReport()
        _check(lib().sww_lm_shoot(self._h, cc, fx, int(nsteps), ctypes.byref(opt), ctypes.byref(rep)), "sww_lm_shoot")
        return list(cc), _lm_report(rep)

    def close(self):
        if getattr(self, "_h", None):
            lib().sww_shooter_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lm_minimize(fun, c0, M: int, fixed=None, **opts):
    """sww_lm_minimize on a Python callback fun(c (numpy, ntot), want_J) -> (r (M), J (M x ntot) or None).  Host-only: needs no GPU."""
    import numpy as np
    ntot = len(c0)
    cc = (ctypes.c_double * ntot)(*[float(x) for x in c0])
    fx = (ctypes.c_int * ntot)(*([0] * ntot if fixed is None else [int(bool(x)) for x in fixed]))

    def cb(_ctx, cp, want_J, rp, Jp):
        try:
            c = np.ctypeslib.as_array(cp, shape=(ntot,)).copy()
            r, J = fun(c, bool(want_J))
            np.ctypeslib.as_array(rp, shape=(M,))[:] = np.asarray(r, dtype=np.float64)
            if want_J:
                np.ctypeslib.as_array(Jp, shape=(ntot, M))[:] = np.asarray(J, dtype=np.float64).T   # column-major M x ntot
            return 0
        except Exception:
            return -1

    opt, rep = _lm_options(**opts), LmReport()
    _check(lib().sww_lm_minimize(LM_FUN(cb), None, int(M), ntot, cc, fx, ctypes.byref(opt), ctypes.byref(rep)), "sww_lm_minimize")
    return np.array(list(cc)), _lm_report(rep)


def mesh_points(N: int, rho: float, where: int = 0):
    """sww_mesh_points: x_j = xi(alpha_j) of the mesh (2.10) as a numpy array (host)"""
    import numpy as np
    x = np.empty(N)
    _check(lib().sww_mesh_points(int(N), float(rho), int(where), x.ctypes.data_as(ctypes.POINTER(ctypes.c_double))), "sww_mesh_points")
    return x


RESPACE_NOALLOC_MAX = 4096


def respace_noalloc(f: torch.Tensor, old, new, out: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None) -> torch.Tensor:
    """sww_respace_noalloc: f (ncol, M_old) on the mesh old = (M_old, rho, where) -> (ncol, M_new) on new = (M_new, rho, where); the library
    allocates nothing (pass `out` to keep torch from allocating as well).  M_new <= RESPACE_NOALLOC_MAX."""
    _require_cuda()
    Mo, Mn = int(old[0]), int(new[0])
    ncol = f.numel() // Mo
    if out is None:
        out = torch.empty((ncol, Mn), dtype=torch.float64, device="cuda")
    st = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().sww_respace_noalloc(Mo, float(old[1]), int(old[2]), Mn, float(new[1]), int(new[2]), ncol, _dev(f, ncol * Mo, "f"),
                                     _dev(out, ncol * Mn, "out"), st.cuda_stream), "sww_respace_noalloc")
    return out


def dtn_linearized_host(eta, phi0, deta, dphi, h: float, prec: int = F64, out=None):
    """HOST-buffer path (sww_dtn_linearized_host): CPU float64 tensors in, CPU tensor out; copies are inside the call.
    out: optional preallocated (ideally pinned) CPU tensor shaped like dphi."""
    _require_cuda()
    mul = 2 if prec == DD else 1
    N = eta.numel() // mul
    nrhs = dphi.numel() // (N * mul)
    for t in (eta, phi0, deta, dphi):
        assert (not t.is_cuda) and t.dtype == torch.float64 and t.is_contiguous()
    if out is None:
        out = torch.empty_like(dphi)
        if dphi.is_pinned():
            out = out.pin_memory()
    else:
        assert (not out.is_cuda) and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == dphi.numel()
    _check(lib().sww_dtn_linearized_host(eta.data_ptr(), phi0.data_ptr(), deta.data_ptr(), dphi.data_ptr(), out.data_ptr(), N, float(h), prec, nrhs),
           "sww_dtn_linearized_host")
    return out


def host_cache_clear():
    """free the context cached by dtn_linearized_host (sww_host_cache_clear)"""
    _check(lib().sww_host_cache_clear(), "sww_host_cache_clear")
