"""NEXT-4 host logic on CPU: the z-slab ghost exchange of paper_2210_17509_b200/halo.py over gloo, world sizes 2 and 3
(127.0.0.1), and the single-rank self-exchange.  Packing / unpacking are slicing functions here (the library's kernels need
a GPU); what is tested is which planes go to which neighbour, the ring wrap, tags and ordering: after the exchange the z
ghost planes of every rank hold the planes of the periodic global array, x and y ghost cells included."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
G, NZ, NY, NX = 3, 5, 4, 6


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _pack(prim, g, side, buf):
    nz = prim.shape[2] - 2 * g
    k0 = g if side == 0 else nz
    buf.copy_(prim[:, :, k0:k0 + g])


def _unpack(prim, g, side, buf):
    nz = prim.shape[2] - 2 * g
    k0 = 0 if side == 0 else nz + g
    prim[:, :, k0:k0 + g].copy_(buf)


def _global(world):
    """Periodic global array [1, 8, world * NZ, NY + 2G, NX + 2G] of distinct values."""
    n = 8 * world * NZ * (NY + 2 * G) * (NX + 2 * G)
    return np.arange(n, dtype=np.float64).reshape(1, 8, world * NZ, NY + 2 * G, NX + 2 * G) + 0.5


def _slab(glob, rank, world):
    import torch
    a = np.full((1, 8, NZ + 2 * G, NY + 2 * G, NX + 2 * G), np.nan)
    a[:, :, G:G + NZ] = glob[:, :, rank * NZ:(rank + 1) * NZ]
    return torch.from_numpy(a)


def _expected(glob, rank, world):
    ks = [(rank * NZ + k) % (world * NZ) for k in range(-G, NZ + G)]
    return glob[:, :, ks]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2210_17509_b200.halo import ZSlabExchange
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        glob = _global(world)
        prim = _slab(glob, rank, world)
        ex = ZSlabExchange(prim, G, pack=_pack, unpack=_unpack)
        for rep in range(2):                       # twice: buffers and tags are reusable
            ex.start(prim)
            ex.finish(prim)
        np.save(os.path.join(out, f"halo{rank}.npy"), prim.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_z_slab_exchange_ring(tmp_path, world):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    glob = _global(world)
    for r in range(world):
        got = np.load(tmp_path / f"halo{r}.npy")
        assert np.array_equal(got, _expected(glob, r, world)), f"rank {r} of {world}"


def test_single_rank_is_its_own_neighbour():
    sys.path.insert(0, ROOT)
    from paper_2210_17509_b200.halo import ZSlabExchange
    glob = _global(1)
    prim = _slab(glob, 0, 1)
    ex = ZSlabExchange(prim, G, pack=_pack, unpack=_unpack)
    assert ex.world == 1 and ex.bytes_per_exchange == 2 * 8 * G * (NY + 2 * G) * (NX + 2 * G) * 8
    ex.start(prim)
    ex.finish(prim)
    assert np.array_equal(prim.numpy(), _expected(glob, 0, 1))


def test_exchange_rejects_batches_and_thin_slabs():
    import torch
    sys.path.insert(0, ROOT)
    from paper_2210_17509_b200.halo import ZSlabExchange
    with pytest.raises(ValueError):
        ZSlabExchange(torch.zeros(2, 8, 12, 8, 8, dtype=torch.float64), 3, pack=_pack, unpack=_unpack)
    with pytest.raises(ValueError):
        ZSlabExchange(torch.zeros(1, 8, 8, 8, 8, dtype=torch.float64), 3, pack=_pack, unpack=_unpack)
