"""NEXT-3 on the GPU: grx_valencia_rhs_vertex and grx_tmunu_vertices against the oracle (R31 / R32), element by element,
through the C ABI.  Bar: 1e-11 of the oracle's per-component maximum; ghost cells of `out` and vertices outside the
interior cells untouched."""
import numpy as np
import pytest

from paper_2210_17509_b200 import inputs
from util import relerr_per_component
from test_oracle_vertex import _both, _smooth_metric, _smooth_K, _linear_metric, _linear_K, G

pytestmark = pytest.mark.gpu
TOL = 1e-11


@pytest.fixture(scope="module")
def grx():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2210_17509_b200 import build, grx as g
    build.build()
    g.lib()
    return g


def _dev(*arrays):
    import torch
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays)


def _vertex_problem(n, nbox=1, seed=0):
    """Config-5 style primitives (seeded) on a smooth analytic metric sampled at centres and vertices."""
    lo, hi = (-1.0, -0.8, -0.7), (1.0, 0.8, 0.7)
    prim, met_c, K_c, met_v, K_v, dx = _both(n, lo, hi, _smooth_metric, _smooth_K)
    if nbox > 1:
        rng = np.random.default_rng(seed)
        prim = np.concatenate([prim * (1 + 0.05 * b * np.array([1, 0.5, -0.5, 0.3, 1, 0.2, -0.2, 0.4])[None, :, None, None, None])
                               for b in range(nbox)])
        met_v = np.concatenate([met_v] * nbox)
        K_v = np.concatenate([K_v * (1 + b) for b in range(nbox)])
        del rng
    return prim, met_v, K_v, dx


@pytest.mark.parametrize("variant", ["auto", "simple"])
@pytest.mark.parametrize("n,nbox", [((20, 12, 9), 2), ((33, 5, 4), 1), ((1, 1, 1), 1), ((130, 3, 2), 1), ((64, 64, 16), 1),
                                    ((70, 25, 40), 1)])
def test_vertex_rhs_parity(grx, oracle, n, nbox, variant):
    """auto = the face-once tile traversal (rhs_fused_kernel with vertex loads: ragged tiles, thin blocks, several z chunks),
    simple = one thread per cell."""
    import torch
    prim, met_v, K_v, dx = _vertex_problem(n, nbox)
    gamma = 5.0 / 3.0
    d = _dev(prim, met_v, K_v)
    ii = (slice(None), slice(None), slice(G, -G), slice(G, -G), slice(G, -G))
    for recon in ("minmod", "mc", "weno5"):
        ref, nfb_ref = oracle.valencia_rhs_vertex(prim, met_v, K_v, dx, G, recon, gamma)
        out = torch.full_like(d[0], -7.25e300)
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        grx.set_fallback_counter(cnt)
        grx.set_variant(variant)
        try:
            grx.valencia_rhs_vertex(*d, dx, G, recon, gamma, out=out)
            torch.cuda.synchronize()
        finally:
            grx.set_fallback_counter(None)
            grx.set_variant("auto")
        got = out.cpu().numpy()
        rel = relerr_per_component(got[ii], ref[ii])
        assert np.all(np.isfinite(got[ii])) and rel.max() <= TOL, f"{n}/{recon}: {rel}"
        ghost = np.ones(got.shape, dtype=bool)
        ghost[ii] = False
        assert np.all(got[ghost] == -7.25e300)
        assert int(cnt.item()) == nfb_ref


def test_vertex_rhs_parity_256_full_block(grx, oracle):
    """The size bench.py times grx_valencia_rhs_vertex at (256^3 interior, 257^3-vertex metric, WENO5): every interior cell
    against the oracle, fallback count included."""
    import torch
    prim, met_v, K_v, dx = _vertex_problem((256, 256, 256))
    gamma = 5.0 / 3.0
    ref, nfb_ref = oracle.valencia_rhs_vertex(prim, met_v, K_v, dx, G, "weno5", gamma)
    d = _dev(prim, met_v, K_v)
    out = torch.full_like(d[0], -7.25e300)
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    grx.set_fallback_counter(cnt)
    try:
        grx.valencia_rhs_vertex(*d, dx, G, "weno5", gamma, out=out)
        torch.cuda.synchronize()
    finally:
        grx.set_fallback_counter(None)
    got = out.cpu().numpy()
    ii = (slice(None), slice(None), slice(G, -G), slice(G, -G), slice(G, -G))
    rel = relerr_per_component(got[ii], ref[ii])
    assert np.all(np.isfinite(got[ii])) and rel.max() <= TOL, rel
    assert int(cnt.item()) == nfb_ref


def test_vertex_rhs_linear_metric_equals_cell_centred_kernel(grx):
    """Pin V1 on the GPU: on a metric linear in the coordinates the vertex kernel reproduces the product (cell-centred)
    kernel to rounding."""
    import torch
    n, lo, hi = (34, 14, 10), (-1.0, -0.8, -0.7), (1.0, 0.8, 0.7)
    prim, met_c, K_c, met_v, K_v, dx = _both(n, lo, hi, _linear_metric, _linear_K)
    p, mc, kc, mv, kv = _dev(prim, met_c, K_c, met_v, K_v)
    a = grx.valencia_rhs(p, mc, kc, dx, G, "weno5", 5.0 / 3.0)
    b = grx.valencia_rhs_vertex(p, mv, kv, dx, G, "weno5", 5.0 / 3.0)
    torch.cuda.synchronize()
    ii = (slice(None), slice(None), slice(G, -G), slice(G, -G), slice(G, -G))
    assert relerr_per_component(b[ii].cpu().numpy(), a[ii].cpu().numpy()).max() < 1e-12


@pytest.mark.parametrize("n,nbox", [((20, 12, 9), 2), ((1, 1, 1), 1), ((130, 6, 5), 1), ((10, 6, 135), 1)])
def test_tmunu_vertices_parity(grx, oracle, n, nbox):
    import torch
    prim, met_v, _, dx = _vertex_problem(n, nbox)
    gamma = 1.4
    ref = oracle.tmunu_vertices(prim, met_v, G, gamma)
    p, mv = _dev(prim, met_v)
    T = torch.full(ref.shape, -7.25e300, dtype=torch.float64, device="cuda")
    grx.tmunu_vertices(p, mv, G, gamma, out=T)
    torch.cuda.synchronize()
    got = T.cpu().numpy()
    defined = np.isfinite(ref)
    assert defined.sum() == nbox * 10 * (n[0] + 1) * (n[1] + 1) * (n[2] + 1)
    for c in range(10):
        scale = np.abs(ref[:, c][defined[:, c]]).max()
        assert np.abs(got[:, c][defined[:, c]] - ref[:, c][defined[:, c]]).max() <= TOL * max(scale, np.abs(ref[defined]).max() * 1e-3)
    assert np.all(got[~defined] == -7.25e300), "only the vertices of the interior cells are written"


def test_vertex_entry_points_reject_bad_arguments(grx):
    import torch
    prim, met_v, K_v, dx = _vertex_problem((8, 6, 5))
    p, mv, kv = _dev(prim, met_v, K_v)
    with pytest.raises(grx.GrxError, match="vertex array"):
        grx.valencia_rhs_vertex(p, mv[:, :, :-1].contiguous(), kv, dx, G, "weno5", 1.4)
    with pytest.raises(grx.GrxError, match="gamma"):
        grx.valencia_rhs_vertex(p, mv, kv, dx, G, "weno5", 1.0)
    with pytest.raises(grx.GrxError, match="2 ghost"):
        grx.tmunu_vertices(p[:, :, 2:-2, 2:-2, 2:-2].contiguous(), mv[:, :, 2:-2, 2:-2, 2:-2].contiguous(), 1, 1.4)
