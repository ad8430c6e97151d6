"""Host-side checks that need no GPU: the C-ABI library builds, loads, and exports every symbol include/sww.h declares;
argument validation that returns before any CUDA call; the Python binding refuses to compute without a device."""
from __future__ import annotations

import ctypes
import re
from pathlib import Path

import numpy as np
import pytest
import torch

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def sww():
    from paper_1210_5672_b200 import build
    build.build()
    import paper_1210_5672_b200 as pkg
    return pkg


def declared_symbols():
    text = (ROOT / "include" / "sww.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sww_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for required in ("sww_dtn_setup", "sww_dtn_apply", "sww_dtn_linearized_apply", "sww_rk_advance"):
        assert required in names


def test_library_exports_every_declared_symbol(sww):
    L = sww.lib()
    names = declared_symbols()
    assert names, "no declarations parsed from include/sww.h"
    for n in names:
        assert hasattr(L, n), f"libsww.so does not export {n}"
    assert sorted(sww.EXPORTS) == names, "binding.EXPORTS and include/sww.h disagree"


def test_strerror_and_codes(sww):
    L = sww.lib()
    assert L.sww_strerror(0) == b"ok"
    texts = {L.sww_strerror(c) for c in range(-6, 1)}
    assert len(texts) == 7 and b"unknown status" not in texts
    assert L.sww_strerror(-99) == b"unknown status"


def test_argument_validation_needs_no_device(sww):
    L = sww.lib()
    h = ctypes.c_void_p()
    buf = np.zeros(64)
    p = buf.ctypes.data
    assert L.sww_dtn_setup(None, 64, 1.0, 0, None, ctypes.byref(h)) == -1          # null eta
    assert L.sww_dtn_setup(p, 48, 1.0, 0, None, ctypes.byref(h)) == -1             # N not a power of two
    assert L.sww_dtn_setup(p, 8, 1.0, 0, None, ctypes.byref(h)) == -1              # N too small
    assert L.sww_dtn_setup(p, 16384, 1.0, 0, None, ctypes.byref(h)) == -1          # N too large
    assert L.sww_dtn_setup(p, 64, 1.0, 7, None, ctypes.byref(h)) == -1             # unknown precision
    assert L.sww_dtn_setup(p, 64, -1.0, 0, None, ctypes.byref(h)) == -1            # negative depth
    assert L.sww_dtn_setup(p, 8192, 1.0, 1, None, ctypes.byref(h)) == -1           # double-double stops at N = 4096 (include/sww.h)
    assert L.sww_dtn_apply(None, p, 1, p) == -1
    assert L.sww_dtn_linearized_apply(None, p, p, 1, p) == -1
    assert L.sww_rk_advance(None, 0.1, 1) == -1
    assert L.sww_dtn_linearized_host(p, p, p, p, p, 48, 1.0, 0, 1) == -1


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback(sww):
    eta = torch.zeros(64, dtype=torch.float64)
    with pytest.raises(RuntimeError, match="no CPU path"):
        sww.DtN(eta, 1.0)
    with pytest.raises(RuntimeError, match="no CPU path"):
        sww.State(eta, eta, 1.0)


def test_product_never_imports_the_oracle():
    for p in (ROOT / "paper_1210_5672_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            assert "oracle" not in re.sub(r"(#|//).*", "", p.read_text()).replace("shares nothing with oracle/", ""), p
    for p in (ROOT / "oracle").rglob("*"):
        if p.suffix in (".py", ".c", ".h"):
            assert "paper_1210_5672_b200" not in re.sub(r"(#|//|\*).*", "", p.read_text()), p


def test_mesh_points_host_function(sww):
    """sww_mesh_points is host code: xi(alpha_j) of (2.10) against the oracle's tables, the printed end-point spacings (2.11) by
    differences, monotonicity; argument checks of the mesh entry points that return before any CUDA call"""
    import oracle
    o = oracle.Oracle("ld")
    N = 96   # the host function takes any N
    for rho, where in ((1.0, 0), (0.6, 0), (0.25, 1), (0.05, 0)):
        x = sww.mesh_points(N, rho, where)
        try:
            o.set_mesh(rho, where)
            xp, E, _ = o.mesh_tables(N)
        finally:
            o.set_mesh()
        assert np.abs(x - (2 * np.pi * np.arange(N) / N + xp[0])).max() < 2e-15
        assert np.all(np.diff(x) > 0) and x[0] == 0.0
        ratio = (x[1] - x[0]) / (x[N // 2 + 1] - x[N // 2])          # spacing at x = 0 over spacing at x = pi
        want = (1 / rho) if where == 0 else rho
        assert abs(ratio / want - 1) < 0.02 / rho
    L = sww.lib()
    buf = np.zeros(8)
    px = buf.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    assert L.sww_mesh_points(8, 0.0, 0, px) == -1 and L.sww_mesh_points(8, 1.5, 0, px) == -1 and L.sww_mesh_points(8, 0.5, 2, px) == -1
    assert L.sww_mesh_points(8, 0.5, 0, None) == -1
    assert L.sww_dtn_set_mesh(None, 0.5, 0) == -1 and L.sww_state_set_mesh(None, 0.5, 0) == -1
    assert L.sww_state_respace(None, None) == -1
    assert L.sww_shooter_set_segments(None, 1, None, None, None, None, None) == -1
