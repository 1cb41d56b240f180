"""NEXT-2 on the GPU: grx_valencia_rhs_ct (flux-CT of calB, reading R30) against the oracle, element by element, through
the C ABI.  Bar: max|gpu - oracle| <= 1e-11 max|oracle| per component (the calB components of a CT update are sums of up
to 32 face fluxes: same bar), D, S_i, tau bit-identical to grx_valencia_rhs, ghost cells of `out` untouched; the face
fluxes in the workspace match the oracle's on every face flux-CT reads."""
import numpy as np
import pytest

from paper_2210_17509_b200 import inputs
from util import cut_block, relerr_per_component

pytestmark = pytest.mark.gpu
TOL = 1e-11
FB_OF_ORACLE = (1, 2, 3, 5, 6, 7)     # oracle FB[3 d + c] -> library FB[0..5]


@pytest.fixture(scope="module")
def grx():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2210_17509_b200 import build, grx as g
    build.build()
    g.lib()
    return g


def _run(grx, prob, recon, variant):
    import torch
    dev = tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (prob.prim, prob.metric, prob.K))
    out = torch.full_like(dev[0], -7.25e300)
    grx.set_variant(variant)
    try:
        plain = grx.valencia_rhs(*dev, prob.dx, prob.nghost, recon, prob.gamma)
        _, fb = grx.valencia_rhs_ct(*dev, prob.dx, prob.nghost, recon, prob.gamma, out=out)
        torch.cuda.synchronize()
    finally:
        grx.set_variant("auto")
    return out.cpu().numpy(), plain.cpu().numpy(), fb.cpu().numpy()


def _check(prob, recon, got, plain, fb, oracle, check_fb=True):
    g = prob.nghost
    ref, _ = oracle.valencia_rhs_ct(prob.prim, prob.metric, prob.K, prob.dx, g, recon, prob.gamma)
    ii = prob.interior
    rel = relerr_per_component(got[ii], ref[ii])
    assert np.all(np.isfinite(got[ii])) and rel.max() <= TOL, f"{prob.name}/{recon}: {rel}"
    assert np.array_equal(got[ii][:, :5], plain[ii][:, :5]), "D, S_i, tau must be those of grx_valencia_rhs"
    ghost = np.ones(got.shape, dtype=bool)
    ghost[ii] = False
    assert np.all(got[ghost] == -7.25e300), "ghost cells of out were written (R23)"
    if check_fb:
        FBo = oracle.face_bfluxes(prob.prim, prob.metric, g, recon, prob.gamma)[:, FB_OF_ORACLE]
        defined = np.isfinite(FBo)
        scale = np.abs(FBo[defined]).max()
        assert np.abs(fb[defined] - FBo[defined]).max() <= TOL * scale
    return rel.max()


@pytest.mark.parametrize("variant", ["auto", "ldg"])
@pytest.mark.parametrize("name", ["c1", "gen", "c2:small", "c3:small", "c4:small", "c5-32:small"])
def test_ct_parity_small(grx, oracle, name, variant):
    prob = inputs.by_name(name)
    for recon in prob.recons:
        got, plain, fb = _run(grx, prob, recon, variant)
        _check(prob, recon, got, plain, fb, oracle)


@pytest.mark.parametrize("n", [(2, 5, 2), (34, 1, 3), (2, 2, 70), (64, 8, 9), (30, 61, 17), (33, 12, 9), (1, 1, 1)])
def test_ct_parity_ragged_and_thin(grx, oracle, n):
    """Tiles cut by the block edge, single rows / columns / planes (every face then lies on a line next to the block),
    odd Nx (LDG kernel + face kernel for all faces), two boxes, off-diagonal metric."""
    base = inputs.general_metric_box(n=(96, 62, 71), seed=3, nbox=2)
    prob = cut_block(base, (1, 1, 1), n)
    Nx = n[0] + 2 * prob.nghost
    for variant in ("auto", "tma") if Nx % 2 == 0 else ("auto",):     # forced TMA: the fused face export on every shape
        for recon in ("minmod", "mc", "weno5"):
            got, plain, fb = _run(grx, prob, recon, variant)
            _check(prob, recon, got, plain, fb, oracle)


def test_ct_two_and_four_ghosts(grx, oracle):
    """nghost = 2 (the minimum for minmod / MC: the faces of the lines next to the block reach the outermost ghost cells) and
    nghost = 4 (wider than needed)."""
    for g, recons in ((2, ("minmod", "mc")), (4, ("weno5", "minmod"))):
        prob = inputs.general_metric_box(n=(34, 11, 9), seed=27, g=g, nbox=2)
        for variant in ("auto", "tma", "ldg"):
            for recon in recons:
                got, plain, fb = _run(grx, prob, recon, variant)
                _check(prob, recon, got, plain, fb, oracle)


def test_ct_update_is_divergence_free_on_the_gpu(grx):
    """The vertex-centred divergence of the GPU's d calB/dt vanishes to rounding on a multi-tile block."""
    prob = inputs.general_metric_box(n=(70, 30, 21), seed=17)
    got, _, _ = _run(grx, prob, "weno5", "auto")
    dB = got[prob.interior][0, 5:8]
    lo, hi = slice(None, -1), slice(1, None)
    div = 0.0
    for d in range(3):
        tot = 0.0
        for s1 in (lo, hi):
            for s2 in (lo, hi):
                if d == 0:
                    tot = tot + dB[0][s1, s2, hi] - dB[0][s1, s2, lo]
                elif d == 1:
                    tot = tot + dB[1][s1, hi, s2] - dB[1][s1, lo, s2]
                else:
                    tot = tot + dB[2][hi, s1, s2] - dB[2][lo, s1, s2]
        div = div + 0.25 * tot / prob.dx[d]
    assert np.abs(div).max() < 1e-12 * np.abs(dB).max() / min(prob.dx)


def test_ct_repeated_calls_are_bitwise_identical(grx):
    """Every face flux in the workspace has one writer: the faces between two tiles are evaluated by both tiles (with
    different rounding in y, where a row warp and the rim warp meet), and only one of them may store its value.  Several
    row tiles, x tiles and z chunks, two boxes; out and the workspace bit for bit over repeated calls."""
    prob = inputs.general_metric_box(n=(70, 30, 21), seed=23, nbox=2)
    for recon in ("weno5", "minmod"):
        runs = [_run(grx, prob, recon, "tma") for _ in range(4)]
        for got, _, fb in runs[1:]:
            assert np.array_equal(got, runs[0][0]) and np.array_equal(fb, runs[0][2]), recon


def test_ct_parity_config5_128_full_block(grx, oracle):
    """A full-size sweep point (128^3 x 1 of config 5) in the launch geometry bench.py times for the CT entry point."""
    prob = inputs.sweep_boxes(128, 1)
    for recon in ("weno5",):
        got, plain, fb = _run(grx, prob, recon, "auto")
        _check(prob, recon, got, plain, fb, oracle, check_fb=False)


def test_ct_parity_bench_workload_256_full_block(grx, oracle):
    """The block bench.py times the CT entry point on (C5 256^3 x 1, WENO5; 296 CTAs in two waves, one z chunk of 256
    planes per CTA, plus the rim face kernel and the curl kernel): every interior cell against the oracle."""
    prob = inputs.sweep_boxes(256, 1)
    got, plain, fb = _run(grx, prob, "weno5", "auto")
    _check(prob, "weno5", got, plain, fb, oracle, check_fb=False)


def test_ct_invalid_arguments(grx):
    import torch
    prob = inputs.general_metric_box(n=(8, 6, 5), seed=1)
    dev = tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (prob.prim, prob.metric, prob.K))
    small = torch.empty(10, dtype=torch.float64, device="cuda")
    with pytest.raises(grx.GrxError, match="workspace too small"):
        grx.valencia_rhs_ct(*dev, prob.dx, prob.nghost, "weno5", prob.gamma, workspace=small)
    with pytest.raises(grx.GrxError, match="nghost too small"):
        grx.valencia_rhs_ct(*dev, prob.dx, 2, "weno5", prob.gamma)
