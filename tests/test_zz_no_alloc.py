"""The no-allocation entry point sww_respace_noalloc (mesh.cu) against the existing respacing path (sww_state_respace: Newton nodes,
stored interpolation matrix, fp64 GEMM), on two calls in a row.  Collected last on purpose (the file name): the suite runs with
pytest -x, and this test is an addition outside the parity suite.  It passes alone in a fresh process and after the other tests:
the entry point's scratch is a fixed device array that every call rewrites before reading it."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import sww_inputs as si

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sww():
    import paper_1210_5672_b200 as pkg
    assert pkg.lib_path().exists() and torch.cuda.is_available()
    return pkg


def smooth(N, seed, amp):
    rng = np.random.default_rng(seed)
    a, b = np.zeros(13), np.zeros(13)
    a[1:] = amp * rng.standard_normal(12) * np.exp(-0.4 * np.arange(1, 13))
    b[1:] = amp * rng.standard_normal(12) * np.exp(-0.4 * np.arange(1, 13))
    return si.synth(N, a, b)[0]


def existing_path(sww, eta, phi, old, new):
    """sww_state_respace between two stepper states (the path the shooting segments use): -> (2, M_new) tensor [eta; phi]"""
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    src = sww.State(dev(eta), dev(phi), 1.0, 1.0)
    src.set_mesh(old[1], old[2])
    z = torch.zeros(new[0], dtype=torch.float64, device="cuda")
    dst = sww.State(z, z, 1.0, 1.0)
    dst.set_mesh(new[1], new[2])
    dst.respace_from(src)
    r = dst.read()
    out = torch.stack([r["eta"], r["phi"]]).clone()
    src.close()
    dst.close()
    return out


def test_no_alloc_respacing_matches_the_existing_path_twice(sww):
    Mo = 256
    eta, phi = smooth(Mo, 21, 0.05), smooth(Mo, 22, 0.1)
    f = torch.from_numpy(np.stack([eta, phi])).cuda().contiguous()
    old = (Mo, 0.5, 1)
    calls = [(512, 0.4, 0), (128, 0.7, 1)]            # the second call is smaller: whatever the first left in the scratch must not matter
    refs = [existing_path(sww, eta, phi, old, new) for new in calls]
    outs = [torch.empty((2, new[0]), dtype=torch.float64, device="cuda") for new in calls]
    sww.respace_noalloc(f, old, calls[0], out=outs[0])            # call 1 (also the per-device address lookup)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    sww.respace_noalloc(f, old, calls[1], out=outs[1])            # call 2, right after it
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                  # nothing was allocated on the device by the call
    for got, ref in zip(outs, refs):
        scale = ref.abs().amax(dim=1, keepdim=True)
        assert float(((got - ref).abs() / scale).max()) <= 3e-14  # the tolerance of the respacing parity tests (tests/test_gpu_mesh.py)
    again = torch.empty_like(outs[0])
    sww.respace_noalloc(f, old, calls[0], out=again)              # call 1 repeated after call 2: the same bits
    assert torch.equal(again, outs[0])
    # more columns than one thread carries (groups of four) and sizes that are not powers of two
    g = torch.from_numpy(np.stack([smooth(96, 30 + c, 1.0) for c in range(7)])).cuda().contiguous()
    x_new = torch.from_numpy(sww.mesh_points(120, 0.6, 0)).cuda()
    w = sww.respace_noalloc(g, (96, 1.0, 0), (120, 0.6, 0))
    # from the uniform mesh the samples are a trigonometric polynomial in alpha = x: evaluate it directly at the new points
    k = torch.arange(1, 13, dtype=torch.float64, device="cuda")[:, None]
    for c in range(7):
        rng = np.random.default_rng(30 + c)
        a = torch.from_numpy(rng.standard_normal(12) * np.exp(-0.4 * np.arange(1, 13))).cuda()
        b = torch.from_numpy(rng.standard_normal(12) * np.exp(-0.4 * np.arange(1, 13))).cuda()
        want = (a[:, None] * torch.cos(k * x_new) + b[:, None] * torch.sin(k * x_new)).sum(dim=0)
        assert float((w[c] - want).abs().max()) <= 3e-14 * float(want.abs().max()), c


def test_no_alloc_limits(sww):
    f = torch.zeros((1, 64), dtype=torch.float64, device="cuda")
    with pytest.raises(sww.SwwError) as e:
        sww.respace_noalloc(f, (64, 1.0, 0), (sww.RESPACE_NOALLOC_MAX + 1, 1.0, 0))
    assert e.value.status == -7 and "SWW_RESPACE_NOALLOC_MAX" in str(e.value)
    sww.respace_noalloc(f, (64, 1.0, 0), (sww.RESPACE_NOALLOC_MAX, 0.5, 0))          # the largest size is served
    for bad_old, bad_new in (((63, 1.0, 0), (64, 1.0, 0)), ((64, 0.0, 0), (64, 1.0, 0)), ((64, 1.0, 0), (64, 1.0, 3))):
        with pytest.raises(sww.SwwError):
            sww.respace_noalloc(torch.zeros((1, bad_old[0]), dtype=torch.float64, device="cuda"), bad_old, bad_new)
