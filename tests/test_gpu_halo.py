"""NEXT-4 on the GPU (one process, one GPU): the z-range right-hand side composes to the whole-block call bit for bit, the
overlapped slab step equals the device-resident grx_step_rk with periodic ghosts bit for bit (one slab, its own neighbour)
and a two-slab ring emulated in one process equals the undivided domain."""
import numpy as np
import pytest

from paper_2210_17509_b200 import inputs

pytestmark = pytest.mark.gpu


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


@pytest.mark.parametrize("variant", ["auto", "tma", "ldg"])
def test_zrange_pieces_are_the_whole_block_bit_for_bit(grx, variant):
    import torch
    prob = inputs.general_metric_box(n=(34, 20, 40), seed=23)
    prim, met, K = _dev(prob.prim, prob.metric, prob.K)
    g, nz = prob.nghost, prob.n[2]
    grx.set_variant(variant)
    try:
        for recon in ("weno5", "minmod"):
            whole = grx.valencia_rhs(prim, met, K, prob.dx, g, recon, prob.gamma)
            out = torch.full_like(prim, -7.25e300)
            for k0, k1 in ((g, nz - g), (0, g), (nz - g, nz)):
                grx.valencia_rhs_zrange(prim, met, K, prob.dx, g, recon, prob.gamma, out, k0, k1)
            torch.cuda.synchronize()
            ii = prob.interior
            assert torch.equal(out[ii], whole[ii]), f"{variant}/{recon}"
            ghost = torch.ones_like(out, dtype=torch.bool)
            ghost[ii] = False
            assert bool((out[ghost] == -7.25e300).all())
    finally:
        grx.set_variant("auto")
    with pytest.raises(grx.GrxError, match="k_begin"):
        grx.valencia_rhs_zrange(prim, met, K, prob.dx, g, "weno5", prob.gamma, out, 5, nz + 1)


def _periodic_problem(n, seed):
    """Smooth config-5 style fields; ghosts made periodic by the library's own fill."""
    prim, met, K, dx, gamma = inputs._smooth_box(n, seed, inputs.NGHOST)
    return prim[None], met[None], K[None], dx, gamma


@pytest.mark.parametrize("overlap", [True, False])
def test_one_slab_ring_equals_step_rk_periodic(grx, overlap):
    import torch
    from paper_2210_17509_b200 import halo
    g = inputs.NGHOST
    prim_h, met_h, K_h, dx, gamma = _periodic_problem((20, 14, 24), 5)
    # a z-periodic metric, so that the wrapped domain is one consistent problem: take the metric of plane-invariant form
    met_h = np.ascontiguousarray(np.broadcast_to(met_h[:, :, 6:7], met_h.shape))
    K_h = np.ascontiguousarray(np.broadcast_to(K_h[:, :, 6:7], K_h.shape))
    prim, met, K = _dev(prim_h, met_h, K_h)
    grx.fill_ghosts(prim, g, "periodic", 7)
    dt = 0.2 * min(dx)
    consA = grx.prim2con(prim, met, g, gamma)
    primA = prim.clone()
    grx.step_rk(consA, primA, met, K, dx, g, "weno5", gamma, dt, 3, rk=2, bc="periodic")
    consB = grx.prim2con(prim, met, g, gamma)
    primB = prim.clone()
    ex = halo.ZSlabExchange(primB, g)
    work = (torch.empty_like(consB), torch.empty_like(consB))
    halo.step_rk2_zslabs(ex, consB, primB, met, K, dx, g, "weno5", gamma, dt, 3, work, overlap=overlap)
    torch.cuda.synchronize()
    ii = (slice(None), slice(None), slice(g, -g), slice(g, -g), slice(g, -g))
    assert torch.equal(consA[ii], consB[ii])
    assert torch.equal(primA, primB)            # ghosts included
    assert float((consA[ii] - grx.prim2con(prim, met, g, gamma)[ii]).abs().max()) > 1e-6      # it did move


@pytest.mark.parametrize("transport", ["pull", "pack"])
def test_two_slab_ring_in_one_process_equals_the_undivided_domain(grx, oracle, transport):
    """Two z slabs exchanging ghost planes (peer-memory pull kernel, or pack / copy / unpack) against (a) grx_step_rk on the
    undivided periodic domain, bit for bit, and (b) the oracle's method-of-lines loop on the undivided domain
    (oracle_evolve, periodic ghosts filled here with numpy), 1e-10 max|U| per component."""
    import torch
    from paper_2210_17509_b200 import halo
    g = inputs.NGHOST
    nz = 16
    prim_h, met_h, K_h, dx, gamma = _periodic_problem((18, 10, 2 * nz), 9)
    met_h = np.ascontiguousarray(np.broadcast_to(met_h[:, :, 6:7], met_h.shape))
    K_h = np.ascontiguousarray(np.broadcast_to(K_h[:, :, 6:7], K_h.shape))
    # periodic ghosts on the host (no library call on the oracle's input)
    prim_h = np.ascontiguousarray(np.pad(prim_h[:, :, g:-g, g:-g, g:-g], ((0, 0), (0, 0), (g, g), (g, g), (g, g)), mode="wrap"))
    prim, met, K = _dev(prim_h, met_h, K_h)
    filled = prim.clone()
    grx.fill_ghosts(filled, g, "periodic", 7)
    assert torch.equal(filled, prim)            # the library's periodic fill is this wrap
    dt = 0.2 * min(dx)
    cons = grx.prim2con(prim, met, g, gamma)
    whole_p = prim.clone()
    grx.step_rk(cons, whole_p, met, K, dx, g, "weno5", gamma, dt, 2, rk=2, bc="periodic")
    # two slabs: planes [0, nz) and [nz, 2 nz) with their ghost planes cut out of the periodic array
    def cut(a, r):
        return a[:, :, r * nz:(r + 1) * nz + 2 * g].contiguous()
    slabs = []
    for r in range(2):
        p, m, k = cut(prim, r), cut(met, r), cut(K, r)
        slabs.append(dict(prim=p, met=m, K=k, cons=grx.prim2con(p, m, g, gamma), U0=torch.empty_like(p), L=torch.empty_like(p)))
    if transport == "pull":
        exs = [halo.ZSlabExchange(s["prim"], g) for s in slabs]
    else:   # the packing kernels, launched on the exchange's own stream (torch's current stream inside start / finish)
        exs = [halo.ZSlabExchange(s["prim"], g, pack=lambda p, gg, side, buf: grx.halo_z(p, gg, side, False, buf),
                                  unpack=lambda p, gg, side, buf: grx.halo_z(p, gg, side, True, buf)) for s in slabs]
    halo.ZSlabExchange.link_ring(exs)

    def rhs_all():
        for s, ex in zip(slabs, exs):
            ex.start(s["prim"])
        for s in slabs:
            grx.valencia_rhs_zrange(s["prim"], s["met"], s["K"], dx, g, "weno5", gamma, s["L"], g, nz - g)
        for s, ex in zip(slabs, exs):
            ex.finish(s["prim"])
        for s in slabs:
            grx.valencia_rhs_zrange(s["prim"], s["met"], s["K"], dx, g, "weno5", gamma, s["L"], 0, g)
            grx.valencia_rhs_zrange(s["prim"], s["met"], s["K"], dx, g, "weno5", gamma, s["L"], nz - g, nz)

    for _ in range(2):
        for s in slabs:
            s["U0"].copy_(s["cons"])
        rhs_all()
        for s in slabs:
            grx.rk_stage(g, 0.0, s["U0"], 1.0, s["U0"], dt, s["L"], s["cons"], s["met"], gamma, s["prim"])
            grx.fill_ghosts(s["prim"], g, "periodic", 3)
        rhs_all()
        for s in slabs:
            grx.rk_stage(g, 0.5, s["U0"], 0.5, s["cons"], dt, s["L"], s["cons"], s["met"], gamma, s["prim"])
            grx.fill_ghosts(s["prim"], g, "periodic", 3)
    torch.cuda.synchronize()
    for r, s in enumerate(slabs):
        a = s["cons"][:, :, g:-g, g:-g, g:-g]
        b = cons[:, :, g + r * nz:g + (r + 1) * nz, g:-g, g:-g]
        assert torch.equal(a, b), f"slab {r}"
    # against the oracle on the undivided domain
    _, U_ref, nfail = oracle.evolve(prim_h, met_h, K_h, dx, g, "weno5", gamma, dt, 2, rk=2, bc="periodic")
    assert nfail == 0
    ring = np.concatenate([s["cons"][:, :, g:-g, g:-g, g:-g].cpu().numpy() for s in slabs], axis=2)
    ref = U_ref[:, :, g:-g, g:-g, g:-g]
    for c in range(8):
        assert np.abs(ring[:, c] - ref[:, c]).max() <= 1e-10 * np.abs(ref[:, c]).max(), c


def test_halo_pack_unpack_roundtrip(grx):
    import torch
    g = 3
    prim = torch.arange(1 * 8 * 14 * 9 * 10, dtype=torch.float64, device="cuda").reshape(1, 8, 14, 9, 10).contiguous()
    nz = 14 - 2 * g
    buf = torch.empty(grx.halo_z_bytes(prim.shape, g) // 8, dtype=torch.float64, device="cuda")
    for side, k_int, k_ghost in ((0, g, nz + g), (1, nz, 0)):
        grx.halo_z(prim, g, side, False, buf)
        assert torch.equal(buf.view(1, 8, g, 9, 10), prim[:, :, k_int:k_int + g])
        q = prim.clone()
        grx.halo_z(q, g, 1 - side, True, buf)          # what my neighbour does with it
        assert torch.equal(q[:, :, k_ghost:k_ghost + g], prim[:, :, k_int:k_int + g])
        mask = torch.ones_like(q, dtype=torch.bool)
        mask[:, :, k_ghost:k_ghost + g] = False
        assert torch.equal(q[mask], prim[mask])


def test_halo_pull_matches_pack_and_unpack(grx):
    """The peer-memory transport (grx_halo_z_pull) fills the ghost planes with the bits of pack / copy / unpack, touches
    nothing else, and a slab that is its own neighbour wraps around."""
    import torch
    g = 3
    shape = (1, 8, 15, 9, 10)
    slabs = [torch.randn(shape, dtype=torch.float64, device="cuda") for _ in range(3)]
    nz = shape[2] - 2 * g
    for me in range(3):
        below, above = slabs[(me - 1) % 3], slabs[(me + 1) % 3]
        got = slabs[me].clone()
        grx.halo_z_pull(got, g, below, above)
        exp = slabs[me].clone()
        exp[:, :, :g] = below[:, :, nz:nz + g]
        exp[:, :, nz + g:] = above[:, :, g:2 * g]
        assert torch.equal(got, exp)
    own = slabs[0].clone()
    grx.halo_z_pull(own, g, own, own)
    assert torch.equal(own[:, :, :g], slabs[0][:, :, nz:nz + g]) and torch.equal(own[:, :, nz + g:], slabs[0][:, :, g:2 * g])
