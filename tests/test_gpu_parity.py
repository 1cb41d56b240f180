"""Parity of the CUDA path (through the C ABI) with the CPU oracle, on the same seeded inputs.

Bar (BASELINE.json north_star): max|gpu - oracle| <= 1e-11 * max|oracle| per conserved component, over the
interior cells of all boxes of the call; a component that vanishes identically in the oracle is measured
against the largest component (reading R25).  Ghost cells of `out` must stay untouched (R23).
"""
import numpy as np
import pytest

from paper_2210_17509_b200 import inputs
from util import cut_block, relerr_per_component

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


def _to_dev(prob):
    import torch
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (prob.prim, prob.metric, prob.K))


def gpu_rhs(grx, prob, recon, variant="auto", count=False):
    """Runs the CUDA path; `out` is pre-filled with a sentinel so untouched cells are visible."""
    import torch
    prim, met, K = _to_dev(prob)
    out = torch.full_like(prim, -7.25e300)
    grx.set_variant(variant)
    cnt = None
    if count:
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        grx.set_fallback_counter(cnt)
    try:
        grx.valencia_rhs(prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, out=out)
        torch.cuda.synchronize()
        if count:
            assert grx.fallback_count() == int(cnt.item())      # grx_debug_fallback_count reads the same counter
    finally:
        grx.set_fallback_counter(None)
        grx.set_variant("auto")
    res = out.cpu().numpy()
    return (res, int(cnt.item())) if count else res


def check(prob, recon, got, ref, tol=TOL):
    ii = prob.interior
    rel = relerr_per_component(got[ii], ref[ii])
    assert np.all(np.isfinite(got[ii])), f"{prob.name}/{recon}: non-finite output"
    assert rel.max() <= tol, f"{prob.name}/{recon}: per-component rel. error {rel}"
    ghost = np.ones(got.shape, dtype=bool)
    ghost[ii] = False
    assert np.all(got[ghost] == -7.25e300), f"{prob.name}/{recon}: ghost cells of out were written (R23)"
    return rel.max()


SMALL = ["c1", "gen", "c2:small", "c3:small", "c4:small", "c5-32:small"]


@pytest.mark.parametrize("variant", ["auto", "ldg", "simple"])
@pytest.mark.parametrize("name", SMALL)
def test_parity_small(grx, oracle, name, variant):
    """auto = the product path (TMA kernel: every SMALL config has an even Nx), ldg = the round-1 kernel,
    simple = the one-thread-per-cell cross-check."""
    prob = inputs.by_name(name)
    for recon in prob.recons:
        ref, nfb_ref = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
        got, nfb = gpu_rhs(grx, prob, recon, variant, count=True)
        check(prob, recon, got, ref)
        assert nfb == nfb_ref, f"{name}/{recon}: fallback count {nfb} vs oracle {nfb_ref} (R5)"


@pytest.mark.parametrize("n", [(2, 5, 2), (34, 1, 3), (2, 2, 70), (64, 8, 9), (30, 61, 17), (94, 23, 5), (32, 7, 1),
                               (66, 15, 40)])
def test_parity_tma_ragged_and_thin(grx, oracle, n):
    """The TMA kernel (forced) on ragged and thin blocks with an off-diagonal metric, two boxes: tiles cut by the
    block edge in x and y (zero-filled part of the TMA box), single rows and columns, blocks smaller than a TMA
    box, long z chunks, one plane.  All sizes have an even Nx (a TMA requirement)."""
    base = inputs.general_metric_box(n=(96, 62, 71), seed=3, nbox=2)
    prob = cut_block(base, (1, 1, 1), n)
    for recon in ("minmod", "weno5"):
        ref, nfb_ref = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
        got, nfb = gpu_rhs(grx, prob, recon, "tma", count=True)
        check(prob, recon, got, ref)
        assert nfb == nfb_ref


def test_parity_tma_ghost_widths_and_rotor(grx, oracle):
    """nghost = 2 (minmod/MC; the even-start shift of the TMA boxes differs from nghost = 3), nghost = 4 and 5
    (wider than needed), and the rotor's inadmissible WENO5 face states (R5) through the TMA kernel."""
    for g, recons in ((2, ("minmod", "mc")), (4, ("weno5", "mc")), (5, ("weno5", "minmod"))):
        prob = inputs.general_metric_box(n=(18, 10, 7), seed=21, g=g)
        for recon in recons:
            ref, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, g, recon, prob.gamma)
            check(prob, recon, gpu_rhs(grx, prob, recon, "tma"), ref)
    prob = inputs.rotor((96, 80, 1))
    for recon in prob.recons:
        ref, nfb_ref = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
        got, nfb = gpu_rhs(grx, prob, recon, "tma", count=True)
        check(prob, recon, got, ref)
        assert nfb == nfb_ref


def test_auto_takes_the_ldg_kernel_for_odd_nx_and_tma_refuses(grx, oracle):
    """Odd Nx: TMA needs 16-byte global strides, so the product path falls back to the LDG kernel (same bits as
    forcing it) and forcing TMA is refused with GRX_ERR_UNSUPPORTED before any launch."""
    prob = inputs.general_metric_box(n=(37, 19, 11), seed=11, nbox=2)
    for recon in prob.recons:
        ref, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
        a = gpu_rhs(grx, prob, recon, "auto")
        check(prob, recon, a, ref)
        assert np.array_equal(a[prob.interior], gpu_rhs(grx, prob, recon, "ldg")[prob.interior])
    with pytest.raises(grx.GrxError, match="error 3"):
        gpu_rhs(grx, prob, "weno5", "tma")


@pytest.mark.parametrize("n", [(1, 1, 1), (1, 5, 2), (33, 1, 3), (2, 2, 70), (65, 8, 9), (31, 23, 17)])
def test_parity_ragged_and_thin(grx, oracle, n):
    """Degenerate and ragged block shapes (R24) through the product path: single cells, thin directions, sizes off
    the tile grid (odd sizes take the LDG kernel, even ones the TMA kernel)."""
    base = inputs.general_metric_box(n=(66, 24, 71), seed=3, nbox=2)
    prob = cut_block(base, (1, 1, 1), n)
    for recon in ("minmod", "weno5"):
        ref, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
        check(prob, recon, gpu_rhs(grx, prob, recon), ref)


def test_parity_wide_ghosts_and_minmod_two_ghosts(grx, oracle):
    """nghost larger than needed is legal; minmod/MC accept 2 ghosts (R29)."""
    for g, recons in ((5, ("weno5", "minmod")), (2, ("minmod", "mc"))):
        prob = inputs.general_metric_box(n=(18, 10, 7), seed=21, g=g)
        for recon in recons:
            ref, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, g, recon, prob.gamma)
            check(prob, recon, gpu_rhs(grx, prob, recon), ref)


def test_parity_config2_full(grx, oracle):
    """Config 2 at full size (256x256x1): 64 face sides take the R5 fallback under WENO5."""
    prob = inputs.by_name("c2")
    for recon in prob.recons:
        ref, nfb_ref = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
        got, nfb = gpu_rhs(grx, prob, recon, count=True)
        check(prob, recon, got, ref)
        assert nfb == nfb_ref


def test_parity_config3_full(grx, oracle):
    """Config 3 at full size (128^3 curved-spacetime star, WENO5, metric sources)."""
    prob = inputs.by_name("c3")
    ref, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, "weno5", prob.gamma)
    check(prob, "weno5", gpu_rhs(grx, prob, "weno5"), ref)


def test_parity_config5_batches(grx, oracle):
    """Config 5: 32^3 x 64 and 64^3 x 16 batches in full, both reconstructions."""
    for N in (32, 64):
        prob = inputs.by_name(f"c5-{N}")
        for recon in prob.recons:
            ref, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
            check(prob, recon, gpu_rhs(grx, prob, recon), ref)


def _full_block_check(grx, oracle, prob, recon):
    """Full-size check: the oracle evaluates the WHOLE block (about 2 s per 256^3 evaluation on the GPU box's host
    cores, ~6 GB of host memory) and every interior cell is compared, scale = the ORACLE's per-component maxima
    (R25), sentinel check on the ghosts.  Every x/y tile seam and z-chunk seam of the launch bench.py times is covered."""
    ref, nfb_ref = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
    got, nfb = gpu_rhs(grx, prob, recon, count=True)
    worst = check(prob, recon, got, ref)
    assert nfb == nfb_ref, f"{prob.name}/{recon}: fallback count {nfb} vs oracle {nfb_ref} (R5)"
    return worst


def test_parity_config4_full(grx, oracle):
    """Config 4 at full size (256^3 explosion), both reconstructions, every interior cell."""
    prob = inputs.by_name("c4")
    for recon in prob.recons:
        _full_block_check(grx, oracle, prob, recon)


def test_parity_bench_workload_full(grx, oracle):
    """The bench workload (config 5, 256^3 x 1) in the launch configuration bench.py times: every interior
    cell, WENO5 and minmod."""
    prob = inputs.by_name("c5-256")
    for recon in prob.recons:
        _full_block_check(grx, oracle, prob, recon)


def test_parity_config5_128_full(grx, oracle):
    prob = inputs.by_name("c5-128")
    for recon in prob.recons:
        _full_block_check(grx, oracle, prob, recon)


def test_three_traversals_agree(grx):
    """Three traversals of the same arithmetic (TMA kernel, LDG kernel, one thread per cell) agree to rounding on
    a batch."""
    prob = inputs.general_metric_box(n=(40, 17, 13), seed=5, nbox=3)
    for recon in ("minmod", "mc", "weno5"):
        a = gpu_rhs(grx, prob, recon, "tma")
        ii = prob.interior
        for other in ("simple", "ldg"):
            b = gpu_rhs(grx, prob, recon, other)
            assert relerr_per_component(a[ii], b[ii]).max() < 1e-13, other


def test_two_host_threads(grx):
    """The library keeps no per-launch state: two host threads calling concurrently on their own streams get the
    bits of a serial call."""
    import threading
    import torch
    prob = inputs.sweep_boxes(32, 2)
    prim, met, K = _to_dev(prob)
    serial = grx.valencia_rhs(prim, met, K, prob.dx, prob.nghost, "weno5", prob.gamma)
    torch.cuda.synchronize()
    results, errors = [None, None], []

    def work(i):
        try:
            torch.cuda.set_device(0)
            s = torch.cuda.Stream()
            outs = []
            for _ in range(5):
                outs.append(grx.valencia_rhs(prim, met, K, prob.dx, prob.nghost, "weno5", prob.gamma, stream=s))
            s.synchronize()
            results[i] = outs
        except Exception as ex:   # surfaced below
            errors.append(ex)

    threads = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    ii = prob.interior      # ghost cells of `out` are never written (R23): compare the interior
    for outs in results:
        for o in outs:
            assert torch.equal(o[ii], serial[ii])


def test_batch_equals_single_boxes_bitwise(grx):
    """A batched call gives bit-identical results to one call per box (no cross-box coupling)."""
    import torch
    prob = inputs.sweep_boxes(32, 3)
    whole = gpu_rhs(grx, prob, "weno5")
    for b in range(prob.nbox):
        one = inputs.Problem("one", prob.n, 1, prob.nghost, prob.dx, prob.gamma, prob.prim[b:b + 1].copy(),
                             prob.metric[b:b + 1].copy(), prob.K[b:b + 1].copy())
        got = gpu_rhs(grx, one, "weno5")
        assert np.array_equal(got[one.interior], whole[b:b + 1][one.interior])
    torch.cuda.synchronize()


def test_stream_ordering_and_determinism(grx):
    """Calls on a side stream are ordered with work on that stream; repeated calls are bit-identical."""
    import torch
    prob = inputs.sweep_boxes(32, 2)
    prim, met, K = _to_dev(prob)
    s = torch.cuda.Stream()
    outs = []
    with torch.cuda.stream(s):
        for _ in range(3):
            out = torch.zeros_like(prim)
            grx.valencia_rhs(prim, met, K, prob.dx, prob.nghost, "weno5", prob.gamma, out=out, stream=s)
            outs.append(out)
    s.synchronize()
    assert torch.equal(outs[0], outs[1]) and torch.equal(outs[1], outs[2])


def test_guard_bands_no_out_of_bounds_access(grx):
    """Bounds evidence without a sanitizer (compute-sanitizer is closed on this GPU pool): every array of a call sits
    inside a larger allocation whose guard bands hold NaN (inputs) or a sentinel (out).  A read outside an input array
    that reaches the arithmetic turns a result into NaN, a write outside `out` changes a guard: the results must be the
    bits of the plain call and the guards untouched -- for the TMA kernel (whose boxes and L2 prefetches run over the
    tile edge), the LDG kernel (software prefetch of later planes) and the host entry point's slab calls."""
    import torch
    GUARD = 4096          # doubles on each side (32 KB: more than any halo'd row, plane tail or prefetch distance)
    cases = [(inputs.general_metric_box(n=(34, 9, 11), seed=9, nbox=2), "tma"),
             (inputs.general_metric_box(n=(30, 16, 40), seed=10, nbox=1), "tma"),
             (inputs.general_metric_box(n=(33, 12, 9), seed=12, nbox=2), "ldg"),
             (inputs.general_metric_box(n=(2, 2, 3), seed=13, nbox=1), "auto")]
    for prob, variant in cases:
        plain = _to_dev(prob)

        def guarded(a, fill):
            buf = torch.full((a.numel() + 2 * GUARD,), fill, dtype=torch.float64, device="cuda")
            view = buf[GUARD:GUARD + a.numel()].view(a.shape)
            view.copy_(a)
            return buf, view

        bufs = [guarded(a, float("nan")) for a in plain]
        obuf = torch.full((plain[0].numel() + 2 * GUARD,), -7.25e300, dtype=torch.float64, device="cuda")
        out = obuf[GUARD:GUARD + plain[0].numel()].view(plain[0].shape)
        grx.set_variant(variant)
        try:
            for recon in ("minmod", "weno5"):
                ref = grx.valencia_rhs(*plain, prob.dx, prob.nghost, recon, prob.gamma)
                obuf.fill_(-7.25e300)
                grx.valencia_rhs(bufs[0][1], bufs[1][1], bufs[2][1], prob.dx, prob.nghost, recon, prob.gamma, out=out)
                torch.cuda.synchronize()
                ii = prob.interior
                assert torch.equal(out[ii], ref[ii]), f"{prob.name}/{variant}/{recon}: guarded call differs"
                assert bool((obuf[:GUARD] == -7.25e300).all()) and bool((obuf[-GUARD:] == -7.25e300).all()), \
                    f"{prob.name}/{variant}/{recon}: a guard band of out was written"
                for b, _ in bufs:
                    assert bool(torch.isnan(b[:GUARD]).all()) and bool(torch.isnan(b[-GUARD:]).all())
        finally:
            grx.set_variant("auto")


def test_repeated_launches_bitwise_under_load(grx):
    """Race evidence without a sanitizer: the TMA kernel's shared-memory hand-offs (mbarrier-completed TMA planes, two
    CTA barriers per plane, the rim warp's exchange slots) are exercised 40 times on a ragged multi-tile batch while a
    second stream keeps the SMs busy with another launch, so that CTAs are scheduled in changing company; every result
    must be bit-identical to the first."""
    import torch
    prob = inputs.general_metric_box(n=(70, 30, 21), seed=17, nbox=3)
    prim, met, K = _to_dev(prob)
    big = inputs.sweep_boxes(64, 4)
    bdev = _to_dev(big)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    grx.set_variant("tma")
    try:
        for recon in ("weno5", "minmod"):
            first = None
            for it in range(40):
                if it % 2 == 0:
                    grx.valencia_rhs(*bdev, big.dx, big.nghost, recon, big.gamma, stream=s2)
                out = grx.valencia_rhs(prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, stream=s1)
                s1.synchronize()
                if first is None:
                    first = out
                else:
                    assert torch.equal(out[prob.interior], first[prob.interior]), f"{recon}: launch {it} differs"
            s2.synchronize()
    finally:
        grx.set_variant("auto")


def test_uniform_state_constant_metric_exact_zero(grx):
    """Pin P5 on the GPU: a uniform state on any constant metric has an exactly vanishing right-hand side
    in the flux part and rounding-level sources (the derivative stencil gives exact zeros)."""
    import torch
    n, g = (20, 9, 6), 3
    shape = (1, 1, n[2] + 2 * g, n[1] + 2 * g, n[0] + 2 * g)
    pv = [0.7, 0.2, -0.1, 0.3, 1.3, 0.4, -0.2, 0.1]
    mv = [0.9, 0.02, -0.03, 0.01, 1.2, 0.1, -0.05, 1.1, 0.07, 0.95]
    kv = [0.0] * 6
    mk = lambda vals: torch.cat([torch.full(shape, v, dtype=torch.float64, device="cuda") for v in vals], dim=1).contiguous()
    prim, met, K = mk(pv), mk(mv), mk(kv)
    for recon in ("minmod", "mc", "weno5"):
        out = grx.valencia_rhs(prim, met, K, (0.1, 0.2, 0.3), g, recon, 1.4)
        torch.cuda.synchronize()
        assert float(out[:, :, g:-g, g:-g, g:-g].abs().max()) == 0.0


def test_prim2con_parity(grx, oracle):
    import torch
    prob = inputs.general_metric_box(n=(20, 12, 9), seed=7)
    prim, met, _ = _to_dev(prob)
    got = grx.prim2con(prim, met, prob.nghost, prob.gamma).cpu().numpy()
    ref = oracle.prim2con(prob.prim, prob.metric, prob.nghost, prob.gamma)
    assert relerr_per_component(got, ref).max() < 1e-14


def test_con2prim_roundtrip(grx):
    import torch
    prob = inputs.general_metric_box(n=(20, 12, 9), seed=8)
    prim, met, _ = _to_dev(prob)
    cons = grx.prim2con(prim, met, prob.nghost, prob.gamma)
    nfail = torch.zeros(1, dtype=torch.int64, device="cuda")
    back = grx.con2prim(cons, met, prob.nghost, prob.gamma, nfail=nfail)
    torch.cuda.synchronize()
    assert int(nfail.item()) == 0
    assert float((back - prim).abs().max()) < 1e-11


def test_balsara1_rk2_20_steps_gpu_vs_oracle(grx, oracle):
    """Config 1, second half: 20 SSP-RK2 steps (R21/R22) with the GPU right-hand side, prim2con, con2prim and
    RK update against the same loop on the oracle; tolerance 1e-10 * max|U| per component."""
    import torch
    from evolve import fill_copy_bc, rk2_evolve
    prob = inputs.balsara1()
    g, gamma = prob.nghost, prob.gamma
    dt = 0.4 * prob.dx[0]

    class OracleBackend:
        def rhs(self, prim):
            return oracle.valencia_rhs(prim, prob.metric, prob.K, prob.dx, g, "minmod", gamma)[0]

        def prim2con(self, prim):
            return oracle.prim2con(prim, prob.metric, g, gamma)

        def con2prim(self, U):
            return oracle.con2prim(U, prob.metric, g, gamma)[0]

    met_d = torch.from_numpy(prob.metric).cuda()
    K_d = torch.from_numpy(prob.K).cuda()

    class GpuBackend:
        def rhs(self, prim):
            p = torch.from_numpy(np.ascontiguousarray(prim)).cuda()
            out = torch.zeros_like(p)
            grx.valencia_rhs(p, met_d, K_d, prob.dx, g, "minmod", gamma, out=out)
            return out.cpu().numpy()

        def prim2con(self, prim):
            return grx.prim2con(torch.from_numpy(np.ascontiguousarray(prim)).cuda(), met_d, g, gamma).cpu().numpy()

        def con2prim(self, U):
            return grx.con2prim(torch.from_numpy(np.ascontiguousarray(U)).cuda(), met_d, g, gamma).cpu().numpy()

    p_ref, U_ref = rk2_evolve(OracleBackend(), prob.prim, g, dt, 20)
    p_gpu, U_gpu = rk2_evolve(GpuBackend(), prob.prim, g, dt, 20)
    ii = prob.interior
    assert relerr_per_component(U_gpu[ii], U_ref[ii]).max() < 1e-10
    # the device-resident RK building block gives the same stage update
    y = torch.from_numpy(U_ref.copy()).cuda()
    x = y.clone()
    rhs = torch.from_numpy(np.nan_to_num(OracleBackend().rhs(p_ref))).cuda()
    grx.rk_axpy(0.5, x, 0.5, dt, rhs, y, g)
    torch.cuda.synchronize()
    expect = 0.5 * U_ref[ii] + 0.5 * (U_ref[ii] + dt * rhs.cpu().numpy()[ii])
    assert np.abs(y.cpu().numpy()[ii] - expect).max() <= 1e-14 * np.abs(expect).max()


@pytest.mark.parametrize("case", ["balsara1-rk2-copy", "balsara1-rk4-copy", "wave-rk4-periodic", "gen-rk2-periodic",
                                  "wave-rk2-periodic-ct", "gen-rk4-periodic-ct", "balsara1-rk2-copy-ct"])
def test_device_resident_steps_vs_oracle_loop(grx, oracle, case):
    """NEXT-1: N method-of-lines steps entirely on the device (grx_step_rk: RHS, stage update fused with con2prim, ghost
    fill; no host round trip) against the same loop of the oracle (oracle_evolve): 1e-10 max|U| per component (R22).
    "-ct": grx_step_rk_ct against oracle_evolve_ct (constrained transport in every stage, NEXT-2)."""
    import torch
    from test_oracle_evolve import _periodic_wave
    if case.startswith("balsara1"):
        prob, recon, nsteps, cfl = inputs.balsara1(), "minmod", 20, 0.4     # config 1: 20 steps, dt = 0.4 dx (R21)
    elif case.startswith("wave"):
        prob, recon, nsteps, cfl = _periodic_wave(24), "weno5", 6, 0.3
    else:
        prob, recon, nsteps, cfl = inputs.general_metric_box(n=(20, 12, 10), seed=9, nbox=2), "weno5", 4, 0.2
    rk = 4 if "rk4" in case else 2
    bc = "periodic" if "periodic" in case else "copy"
    ct = case.endswith("-ct")
    dt = cfl * min(prob.dx)
    prim0 = prob.prim.copy()
    if not case.startswith("wave"):
        # the generated ghosts are analytic: refill them the way the loop will, so that both sides start from the same state
        from evolve import fill_copy_bc
        g = prob.nghost
        if bc == "copy":
            fill_copy_bc(prim0, g)
        else:
            ii = np.arange(-g, prob.n[0] + g) % prob.n[0] + g
            jj = np.arange(-g, prob.n[1] + g) % prob.n[1] + g
            kk = np.arange(-g, prob.n[2] + g) % prob.n[2] + g
            prim0 = np.ascontiguousarray(prim0[:, :, kk][:, :, :, jj][:, :, :, :, ii])
    p_ref, U_ref, nf_ref = oracle.evolve(prim0, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma, dt, nsteps,
                                         rk=rk, bc=bc, ct=ct)
    assert nf_ref == 0
    prim = torch.from_numpy(prim0).cuda()
    met, K = torch.from_numpy(prob.metric).cuda(), torch.from_numpy(prob.K).cuda()
    cons = grx.prim2con(prim, met, prob.nghost, prob.gamma)
    nfail = torch.zeros(1, dtype=torch.int64, device="cuda")
    grx.step_rk(cons, prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, dt, nsteps, rk=rk, bc=bc, nfail=nfail, ct=ct)
    torch.cuda.synchronize()
    assert int(nfail.item()) == 0
    ii = prob.interior
    assert relerr_per_component(cons.cpu().numpy()[ii], U_ref[ii]).max() < 1e-10
    # primitives incl. their ghost zones follow
    assert np.abs(prim.cpu().numpy() - p_ref).max() < 1e-9 * np.abs(p_ref).max()


def test_device_resident_steps_config5_128_full_block(grx, oracle):
    """grx_step_rk at a size of the sweep (C5 128^3 x 1, WENO5, SSP-RK2, copy boundaries): two steps against oracle_evolve on
    every interior cell -- the multi-wave launch geometry of the right-hand side inside the stepping loop, the fused stage /
    con2prim kernel and the ghost fill on a block of several hundred tiles."""
    import torch
    from evolve import fill_copy_bc
    prob = inputs.sweep_boxes(128, 1)
    g = prob.nghost
    prim0 = fill_copy_bc(prob.prim.copy(), g)
    dt = 0.2 * min(prob.dx)
    p_ref, U_ref, nf_ref = oracle.evolve(prim0, prob.metric, prob.K, prob.dx, g, "weno5", prob.gamma, dt, 2, rk=2, bc="copy")
    assert nf_ref == 0
    prim = torch.from_numpy(prim0).cuda()
    met, K = torch.from_numpy(prob.metric).cuda(), torch.from_numpy(prob.K).cuda()
    cons = grx.prim2con(prim, met, g, prob.gamma)
    nfail = torch.zeros(1, dtype=torch.int64, device="cuda")
    grx.step_rk(cons, prim, met, K, prob.dx, g, "weno5", prob.gamma, dt, 2, rk=2, bc="copy", nfail=nfail)
    torch.cuda.synchronize()
    assert int(nfail.item()) == 0
    ii = prob.interior
    assert relerr_per_component(cons.cpu().numpy()[ii], U_ref[ii]).max() < 1e-10
    assert np.abs(prim.cpu().numpy() - p_ref).max() < 1e-9 * np.abs(p_ref).max()


@pytest.mark.parametrize("test,cfl", [(2, 0.8), (3, 0.4), (4, 0.2), (5, 0.8)])
def test_device_resident_steps_balsara_2_to_5(grx, oracle, test, cfl):
    """NEXT-1 "runs Balsara 1-5 end to end": the Table I states of Balsara 2-5 (minmod + HLLE + RK4,
    copy boundaries l.255, 200 cells, the CFLs at which the oracle's bare loop survives, tests/test_oracle_evolve.py)
    through grx_step_rk against oracle_evolve.  The 10^4 pressure jump of Balsara 3 and the W = 22 collision of Balsara 4 are
    where the warm-started con2prim of the stage kernel has to fall back to its bracketed solve; it must converge in every
    cell (nfail = 0) as the oracle's does."""
    import torch
    from test_oracle_evolve import shocktube
    prob, _ = shocktube(test, 200)
    g = prob.nghost
    dt, nsteps = cfl * prob.dx[0], int(round(8 / cfl))
    p_ref, U_ref, nf_ref = oracle.evolve(prob.prim, prob.metric, prob.K, prob.dx, g, "minmod", prob.gamma, dt, nsteps, rk=4,
                                         bc="copy")
    assert nf_ref == 0
    prim = torch.from_numpy(prob.prim.copy()).cuda()
    met, K = torch.from_numpy(prob.metric).cuda(), torch.from_numpy(prob.K).cuda()
    cons = grx.prim2con(prim, met, g, prob.gamma)
    nfail = torch.zeros(1, dtype=torch.int64, device="cuda")
    grx.step_rk(cons, prim, met, K, prob.dx, g, "minmod", prob.gamma, dt, nsteps, rk=4, bc="copy", nfail=nfail)
    torch.cuda.synchronize()
    assert int(nfail.item()) == 0
    ii = prob.interior
    assert relerr_per_component(cons.cpu().numpy()[ii], U_ref[ii]).max() < 1e-10
    assert np.abs(prim.cpu().numpy() - p_ref).max() < 1e-9 * np.abs(p_ref).max()


def test_steps_with_constrained_transport_keep_the_vertex_divergence(grx):
    """grx_step_rk_ct on a periodic multi-tile block whose field is not solenoidal: the vertex-centred divergence of calB
    after 5 RK2 steps is the initial one to rounding; without CT it is not."""
    import torch
    from test_oracle_ct import _vertex_divergence
    prim_h, met_h, K_h, dx, gamma = inputs._smooth_box((40, 18, 12), 3, inputs.NGHOST)
    g = inputs.NGHOST
    prim = torch.from_numpy(prim_h[None].copy()).cuda()
    met = torch.from_numpy(np.ascontiguousarray(np.broadcast_to(inputs.by_name("c1").metric[:, :, :1, :1, :1], (1, 10) + prim_h.shape[1:]))).cuda()
    K = torch.zeros((1, 6) + prim_h.shape[1:], dtype=torch.float64, device="cuda")
    grx.fill_ghosts(prim, g, "periodic", 7)
    ii = (slice(None), slice(None), slice(g, -g), slice(g, -g), slice(g, -g))
    res = {}
    for ct in (True, False):
        p = prim.clone()
        cons = grx.prim2con(p, met, g, gamma)
        if "U0" not in res:
            res["U0"] = cons[ii].cpu().numpy()
        grx.step_rk(cons, p, met, K, dx, g, "weno5", gamma, 0.2 * min(dx), 5, rk=2, bc="periodic", ct=ct)
        torch.cuda.synchronize()
        res[ct] = cons[ii].cpu().numpy()
    d0 = _vertex_divergence(res["U0"][0, 5:8], dx)
    scale = np.abs(res["U0"][0, 5:8]).max() / min(dx)
    assert np.abs(d0).max() > 1e-2 * scale
    assert np.abs(_vertex_divergence(res[True][0, 5:8], dx) - d0).max() < 1e-12 * scale
    assert np.abs(_vertex_divergence(res[False][0, 5:8], dx) - d0).max() > 1e-6 * scale


def test_selftest_math_accuracy(grx):
    """The MUFU-seeded reciprocal, rsqrt and sqrt helpers are accurate to a few ulp over the range the
    kernels use them on."""
    import torch
    rng = np.random.default_rng(5)
    x = np.concatenate([10.0 ** rng.uniform(-200, 200, 200000), rng.uniform(0.5, 2.0, 200000),
                        1.0 + 10.0 ** rng.uniform(-12, -1, 100000)])
    xd = torch.from_numpy(x).cuda()
    r, rs, s = (t.cpu().numpy() for t in grx.selftest_math(xd))
    xl = x.astype(np.longdouble)
    assert np.max(np.abs(r * xl - 1)) < 4e-16
    assert np.max(np.abs(rs.astype(np.longdouble) ** 2 * xl - 1)) < 8e-16
    assert np.max(np.abs(s.astype(np.longdouble) ** 2 / xl - 1)) < 8e-16


def test_host_entry_point(grx, oracle):
    """grx_valencia_rhs_host: host buffers in, host buffer out, same numbers as the device entry point."""
    import torch
    prob = inputs.sweep_boxes(32, 2)
    hp, hm, hk = (torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (prob.prim, prob.metric, prob.K))
    ho = torch.empty_like(hp).pin_memory()
    ws = torch.empty(grx.host_workspace_bytes(hp.shape, prob.nghost) // 8, dtype=torch.float64, device="cuda")
    grx.valencia_rhs_host(hp, hm, hk, prob.dx, prob.nghost, "weno5", prob.gamma, ho, ws)
    torch.cuda.synchronize()
    dev = gpu_rhs(grx, prob, "weno5")
    ii = prob.interior
    assert np.array_equal(ho.numpy()[ii], dev[ii])


@pytest.mark.parametrize("n,nbox", [((20, 13, 70), 2), ((9, 6, 33), 1), ((12, 12, 96), 1)])
def test_host_entry_point_pipelined(grx, oracle, n, nbox):
    """Blocks with more than 32 planes go through the slab pipeline of grx_valencia_rhs_host (uploads, kernels
    and downloads of 32-plane slabs overlapped on three streams): same bits as the device entry point, parity
    with the oracle, ghost cells of the host `out` untouched."""
    import torch
    prob = inputs.general_metric_box(n=n, seed=17, nbox=nbox)
    hp, hm, hk = (torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (prob.prim, prob.metric, prob.K))
    ws = torch.empty(grx.host_workspace_bytes(hp.shape, prob.nghost) // 8, dtype=torch.float64, device="cuda")
    for recon in ("weno5", "minmod"):
        ho = torch.full(hp.shape, -7.25e300, dtype=torch.float64).pin_memory()
        for _ in range(2):      # twice: the second call reuses the workspace while the first may still be draining
            grx.valencia_rhs_host(hp, hm, hk, prob.dx, prob.nghost, recon, prob.gamma, ho, ws)
        torch.cuda.synchronize()
        got = ho.numpy()
        dev = gpu_rhs(grx, prob, recon)
        ii = prob.interior
        assert np.array_equal(got[ii], dev[ii])
        ref, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
        assert relerr_per_component(got[ii], ref[ii]).max() <= TOL
        g = prob.nghost     # whole interior PLANES come back: the z ghost planes of the host array stay untouched
        assert np.all(got[:, :, :g] == -7.25e300) and np.all(got[:, :, -g:] == -7.25e300)


@pytest.mark.parametrize("n,nbox", [((64, 64, 72), 1), ((32, 32, 100), 1), ((16, 4, 100), 3), ((128, 12, 40), 1),
                                    ((96, 96, 33), 1), ((40, 40, 66), 2), ((33, 20, 41), 1), ((64, 64, 64), 16)])
def test_host_entry_point_has_the_bits_of_the_device_entry_point(grx, n, nbox):
    """The slab pipeline chooses its kernel (and the LDG kernel its row tile) once, on the whole block, as the device entry
    point does: a 32-plane slab on its own would fill the machine differently and could be handed to the other kernel,
    whose rounding differs.  Shapes around the selector's switch-over, small nx / ny with nz > 32, odd Nx, a sweep point."""
    import torch
    prob = inputs.sweep_boxes(n[0], nbox) if n[0] == n[1] == n[2] else inputs.general_metric_box(n=n, seed=5, nbox=nbox)
    hp, hm, hk = (torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (prob.prim, prob.metric, prob.K))
    ws = torch.empty(grx.host_workspace_bytes(hp.shape, prob.nghost) // 8, dtype=torch.float64, device="cuda")
    ii = prob.interior
    for recon in ("weno5", "minmod"):
        ho = torch.zeros(hp.shape, dtype=torch.float64).pin_memory()
        grx.valencia_rhs_host(hp, hm, hk, prob.dx, prob.nghost, recon, prob.gamma, ho, ws)
        torch.cuda.synchronize()
        dev = gpu_rhs(grx, prob, recon)
        assert np.array_equal(ho.numpy()[ii], dev[ii]), (n, nbox, recon)


def test_invalid_arguments_rejected(grx):
    import torch
    prob = inputs.general_metric_box(n=(8, 8, 8), seed=1)
    prim, met, K = _to_dev(prob)
    with pytest.raises(grx.GrxError):
        grx.valencia_rhs(prim, met, K, prob.dx, 2, "weno5", prob.gamma)          # too few ghosts for WENO5
    with pytest.raises(grx.GrxError):
        grx.valencia_rhs(prim, met, K, prob.dx, 3, "weno5", 1.0)                 # gamma <= 1
    with pytest.raises(grx.GrxError):
        grx.valencia_rhs(prim, met, K, (0.1, 0.0, 0.1), 3, "weno5", prob.gamma)  # dx <= 0
    with pytest.raises(grx.GrxError):
        grx.valencia_rhs(prim, met, K, prob.dx, 3, 7, prob.gamma)                # unknown recon
    with pytest.raises(grx.GrxError):
        grx.valencia_rhs(prim, met, K, prob.dx, 3, "weno5", prob.gamma, out=prim.clone()[:, :, :-1].contiguous())
