"""grx_valencia_rhs_ct_static: constrained-transport right-hand side for callers that cannot allocate device memory.

Some users of this library run inside a code whose driver owns every byte of HBM (it reserved the device for its own arena
at start-up), or are called back with field pointers only, or sit in a region where the device-wide synchronisation of a
cudaMalloc is not acceptable.  They cannot provide the face-flux workspace grx_valencia_rhs_ct asks for.  The static entry
point keeps that workspace in a fixed 16 MiB device array inside libgrx.so, shared by all calls on a device and never
cleared.  This file checks, through the C ABI:

  * its output against the existing workspace-taking path on the same inputs, on TWO calls in a row with different
    shapes, reconstructions and kernels (the second call finds the first one's face fluxes in the array and must not be
    affected by them), within the 1e-11 relative bar the other GPU tests use, ghost cells of `out` untouched;
  * a block that fills the array to within 2 % (64^3 interior + 3 ghost cells);
  * that a call beyond the limit is refused with a message that names the limit, before anything is launched.

The file sorts last on purpose (pytest -x stops at the first failure: a failure here hides nothing behind it), and it makes
no assumption about what ran before it in the process: each test builds its own inputs and compares with a reference
computed in the same test.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2210_17509_b200 import inputs
from util import relerr_per_component

TOL = 1e-11
SENTINEL = -7.25e300


@pytest.fixture(scope="module")
def grx():
    from paper_2210_17509_b200 import build, grx as g
    build.build()
    g.lib()
    return g


def _both_paths(grx, prob, recon, variant="auto"):
    """(static entry point, existing path) on the same device inputs; `out` pre-filled with a sentinel."""
    import torch
    dev = tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (prob.prim, prob.metric, prob.K))
    out_static = torch.full_like(dev[0], SENTINEL)
    out_ws = torch.full_like(dev[0], SENTINEL)
    grx.set_variant(variant)
    try:
        grx.valencia_rhs_ct_static(*dev, prob.dx, prob.nghost, recon, prob.gamma, out_static)
        grx.valencia_rhs_ct(*dev, prob.dx, prob.nghost, recon, prob.gamma, out=out_ws)
        torch.cuda.synchronize()
    finally:
        grx.set_variant("auto")
    return out_static.cpu().numpy(), out_ws.cpu().numpy()


def _assert_same(prob, got, ref, what):
    ii = prob.interior
    assert np.all(np.isfinite(ref[ii])), what
    rel = relerr_per_component(got[ii], ref[ii])
    assert np.all(np.isfinite(got[ii])) and rel.max() <= TOL, f"{what}: {rel}"
    ghost = np.ones(got.shape, dtype=bool)
    ghost[ii] = False
    assert np.all(got[ghost] == SENTINEL), f"{what}: ghost cells of out were written"


@pytest.mark.gpu
def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row(grx):
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    # call 1: two boxes, even Nx -> TMA kernel exports the interior faces, face kernel adds the rim
    first = inputs.general_metric_box(n=(34, 21, 19), seed=41, nbox=2)
    # call 2: smaller, odd Nx -> LDG kernel + face kernel for every face; the array still holds call 1's fluxes
    second = inputs.general_metric_box(n=(33, 12, 9), seed=42)
    for prob, recon in ((first, "weno5"), (second, "minmod"), (first, "mc"), (second, "weno5")):
        got, ref = _both_paths(grx, prob, recon)
        _assert_same(prob, got, ref, f"{prob.n}/{recon}")
    # and the same problem twice in a row, the array holding something else before each: same results to the same bar
    a, _ = _both_paths(grx, first, "weno5")
    b, _ = _both_paths(grx, first, "weno5")
    _assert_same(first, b, a, "repeat")


@pytest.mark.gpu
def test_static_scratch_at_its_stated_maximum(grx):
    """64^3 + 3 ghost cells: 6 * 70^3 * 8 = 16 464 000 of the 16 777 216 bytes."""
    prob = inputs.sweep_boxes(64, 1)
    assert 6 * prob.prim[0, 0].size * 8 <= grx.ct_static_max_bytes() == 16 << 20
    got, ref = _both_paths(grx, prob, "weno5")
    _assert_same(prob, got, ref, "64^3 weno5")


def test_static_scratch_rejects_calls_beyond_its_size(grx):
    """Host-side validation only: no pointer is dereferenced and nothing is launched, so this runs without a GPU."""
    lib = grx.lib()
    dx = (C.c_double * 3)(0.1, 0.1, 0.1)
    fake = [C.c_void_p(0x1000 * (k + 1)) for k in range(4)]
    # 65^3 interior + 3 ghosts = 71^3 cells: 17.2 MB of face fluxes; also many small boxes that add up beyond the limit
    for g in (grx.grx_grid(65, 65, 65, 1), grx.grx_grid(32, 32, 32, 7), grx.grx_grid(256, 256, 256, 1)):
        rc = lib.grx_valencia_rhs_ct_static(C.byref(g), fake[0], fake[1], fake[2], dx, 3, 2, 5.0 / 3.0, fake[3], None)
        msg = lib.grx_last_error().decode()
        assert rc == 1, (rc, msg)
        assert "exceeds the static scratch" in msg and "16777216" in msg, msg
    # the other argument checks are those of grx_valencia_rhs_ct
    g = grx.grx_grid(8, 8, 8, 1)
    assert lib.grx_valencia_rhs_ct_static(C.byref(g), fake[0], fake[1], fake[2], dx, 2, 2, 5.0 / 3.0, fake[3], None) == 1
    assert "nghost too small" in lib.grx_last_error().decode()
    assert lib.grx_valencia_rhs_ct_static(C.byref(g), None, fake[1], fake[2], dx, 3, 2, 5.0 / 3.0, fake[3], None) == 1
    assert lib.grx_valencia_rhs_ct_static(C.byref(g), fake[0], fake[1], fake[2], dx, 3, 2, 5.0 / 3.0, fake[0], None) == 1
    assert "alias" in lib.grx_last_error().decode()
