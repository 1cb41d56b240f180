"""NEXT-4: ghost-zone exchange of a slab decomposition along z, overlapped with the interior update.

PAPER.md l.222-230: every block is surrounded by ghost zones "filled by copying from other MPI processes"; l.371: the
paper's weak-scaling ceiling (40-50 %) is the bandwidth of that exchange, and its proposed fix is to "start the
computations of those cells of the next kernel which do not need ghost cells while ghost cells from previous kernel are
getting filled, and then compute the remaining cells thereafter".  This module is that scheme for one process per GPU:

    ZSlabExchange.start(prim)   pack the nghost lowest / highest interior planes (grx_halo_z) on a communication stream and
                                post the point-to-point transfers to the two z neighbours of the ring;
    interior planes             grx_valencia_rhs_zrange(nghost, nz - nghost) on the compute stream -- reads no z ghost plane;
    ZSlabExchange.finish(prim)  wait for the transfers, unpack into the z ghost planes, make the compute stream wait;
    boundary planes             grx_valencia_rhs_zrange(0, nghost) and (nz - nghost, nz).

The domain is periodic along z over the ring of ranks (l.329); x and y ghosts are filled per rank (grx_fill_ghosts, dirs = 3)
BEFORE the exchange, so that whole planes travel and edge / corner ghost cells come along.  Transfers are
torch.distributed point-to-point operations (NCCL over NVLink between GPUs; gloo in the CPU tests); a rank whose neighbour
is itself (world size 1) copies buffer to buffer.  The arithmetic is all in libgrx.so: this file moves buffers and orders
streams.  Only the packing / unpacking can be swapped (the CPU tests pass slicing functions, as there is no CUDA-free
library path).
"""


class ZSlabExchange:
    """Ghost planes of one z slab per rank; ranks form a periodic ring in rank order (slab r sits below slab r + 1)."""

    def __init__(self, prim, nghost, group=None, pack=None, unpack=None):
        import torch
        import torch.distributed as dist
        self.g = int(nghost)
        self.group = group
        self.dist = dist if (dist.is_available() and dist.is_initialized()) else None
        self.world = self.dist.get_world_size(group) if self.dist else 1
        self.rank = self.dist.get_rank(group) if self.dist else 0
        nbox, nf, Nz, Ny, Nx = prim.shape
        if nf != 8 or nbox != 1:
            raise ValueError("ZSlabExchange expects prim[1, 8, Nz, Ny, Nx]: one box per rank")
        if Nz - 2 * self.g < self.g:
            raise ValueError("a slab needs at least nghost interior planes")
        shape = (nbox, 8, self.g, Ny, Nx)
        mk = lambda: torch.empty(shape, dtype=prim.dtype, device=prim.device)   # noqa: E731
        self.send = [mk(), mk()]          # [0]: my lowest interior planes (go down), [1]: my highest (go up)
        self.recv = [mk(), mk()]          # [0]: fills my low ghosts (comes from below), [1]: my high ghosts (from above)
        self.cuda = prim.is_cuda
        self.stream = torch.cuda.Stream(device=prim.device) if self.cuda else None
        self._pack, self._unpack = pack, unpack
        self._reqs = []
        self._ring = None          # in-process ring (link_ring): the slabs of several "ranks" live in this process
        self._packed = None
        self._cs = None            # compute stream of the exchange in flight (pull transport: the neighbours order on it)
        self._prim = None
        self.bytes_per_exchange = 2 * self.send[0].numel() * self.send[0].element_size()

    @staticmethod
    def link_ring(exchanges):
        """A ring of slabs inside ONE process (one GPU holding every slab, or one process driving several GPUs with peer
        access): exchanges[r] is slab r's object.  On CUDA the transport is the peer-memory pull kernel grx_halo_z_pull
        (no pack buffers, one kernel per slab).  Protocol: start() on every slab, then finish() on every slab."""
        for r, ex in enumerate(exchanges):
            ex._ring = (exchanges, r)

    # -- packing: the library's kernels on the GPU; injectable for the CPU tests
    def _do_pack(self, prim, side, buf):
        if self._pack is not None:
            return self._pack(prim, self.g, side, buf)
        from . import grx
        grx.halo_z(prim, self.g, side, False, buf, stream=self.stream)

    def _do_unpack(self, prim, side, buf):
        if self._unpack is not None:
            return self._unpack(prim, self.g, side, buf)
        from . import grx
        grx.halo_z(prim, self.g, side, True, buf, stream=self.stream)

    def start(self, prim, compute_stream=None):
        """Posts the exchange of the z ghost planes of `prim` (whose x / y ghosts are filled).  Returns immediately."""
        import torch
        if self.cuda:
            cs = compute_stream or torch.cuda.current_stream()
            self._cs = cs
            self.stream.wait_stream(cs)          # prim is final on the compute stream
            ctx = torch.cuda.stream(self.stream)
        else:
            import contextlib
            ctx = contextlib.nullcontext()
        self._pull = self._ring is not None and self.cuda and self._pack is None and self._unpack is None
        if self._pull:
            # peer-memory transport (grx_halo_z_pull): nothing to pack; the neighbours read this array directly once the
            # compute stream has produced it
            self._prim = prim
            self._packed = torch.cuda.Event()
            self._packed.record(self.stream)
            self._reqs = []
            return
        with ctx:
            self._do_pack(prim, 0, self.send[0])
            self._do_pack(prim, 1, self.send[1])
            if self._ring is not None:
                if self.cuda:
                    import torch as _t
                    self._packed = _t.cuda.Event()
                    self._packed.record(self.stream)
                self._reqs = []
            elif self.world == 1:
                # my own neighbour on both sides: low ghosts <- my highest planes, high ghosts <- my lowest
                self.recv[0].copy_(self.send[1], non_blocking=True)
                self.recv[1].copy_(self.send[0], non_blocking=True)
                self._reqs = []
            else:
                d = self.dist
                below, above = (self.rank - 1) % self.world, (self.rank + 1) % self.world
                to_g = (lambda r: d.get_global_rank(self.group, r)) if self.group is not None else (lambda r: r)
                ops = [d.P2POp(d.isend, self.send[0], to_g(below), self.group, tag=0),
                       d.P2POp(d.isend, self.send[1], to_g(above), self.group, tag=1),
                       d.P2POp(d.irecv, self.recv[1], to_g(above), self.group, tag=0),   # its lowest planes
                       d.P2POp(d.irecv, self.recv[0], to_g(below), self.group, tag=1)]   # its highest planes
                self._reqs = d.batch_isend_irecv(ops)

    def finish(self, prim, compute_stream=None):
        """Completes the exchange: the z ghost planes of `prim` are filled for later work on the compute stream."""
        import torch
        if self._reqs:
            # Work.wait() of the NCCL backend does not block the host: it makes the CURRENT stream wait for the transfer.
            # The unpack kernels run on self.stream, so that is the stream that has to be current here (gloo blocks the
            # host instead, where any stream will do).
            if self.cuda:
                with torch.cuda.stream(self.stream):
                    for r in self._reqs:
                        r.wait()
            else:
                for r in self._reqs:
                    r.wait()
        self._reqs = []
        if self._ring is not None and getattr(self, "_pull", False):
            from . import grx
            ring, me = self._ring
            below, above = ring[(me - 1) % len(ring)], ring[(me + 1) % len(ring)]
            self.stream.wait_event(below._packed)
            self.stream.wait_event(above._packed)
            grx.halo_z_pull(prim, self.g, below._prim, above._prim, stream=self.stream)
            # the pull read the neighbours' arrays: whatever their compute streams enqueue from now on (the next stage
            # writes prim) is ordered after it.  The protocol (every start() before any finish(), the next writes after
            # every finish()) makes "from now on" early enough.
            pulled = torch.cuda.Event()
            pulled.record(self.stream)
            for nb in (below, above):
                if nb is not self and nb._cs is not None:
                    nb._cs.wait_event(pulled)
            # self._prim stays set: the neighbours' finish() calls, which come later, read it
            (compute_stream or torch.cuda.current_stream()).wait_stream(self.stream)
            return
        if self._ring is not None:
            ring, me = self._ring
            below, above = ring[(me - 1) % len(ring)], ring[(me + 1) % len(ring)]
            if self.cuda:
                self.stream.wait_event(below._packed)
                self.stream.wait_event(above._packed)
                ctx = torch.cuda.stream(self.stream)
            else:
                import contextlib
                ctx = contextlib.nullcontext()
            with ctx:
                self.recv[0].copy_(below.send[1], non_blocking=True)
                self.recv[1].copy_(above.send[0], non_blocking=True)
        if self.cuda:
            with torch.cuda.stream(self.stream):
                self._do_unpack(prim, 0, self.recv[0])
                self._do_unpack(prim, 1, self.recv[1])
            (compute_stream or torch.cuda.current_stream()).wait_stream(self.stream)
        else:
            self._do_unpack(prim, 0, self.recv[0])
            self._do_unpack(prim, 1, self.recv[1])


def rhs_overlapped(exch, prim, metric, K, dx, nghost, recon, gamma, out, overlap=True, stream=None):
    """One right-hand-side evaluation of this rank's slab with the z ghost exchange of `prim` in flight: interior planes
    while the planes travel, boundary planes after they have arrived (l.371).  overlap = False: exchange first, then one
    whole-block call (what the paper's current scheme does; the measurement's comparison arm).  Same bits either way."""
    from . import grx
    nz = prim.shape[2] - 2 * nghost
    if not overlap or nz < 3 * nghost:
        exch.start(prim, stream)
        exch.finish(prim, stream)
        return grx.valencia_rhs_zrange(prim, metric, K, dx, nghost, recon, gamma, out, 0, nz, stream=stream)
    exch.start(prim, stream)
    grx.valencia_rhs_zrange(prim, metric, K, dx, nghost, recon, gamma, out, nghost, nz - nghost, stream=stream)
    exch.finish(prim, stream)
    grx.valencia_rhs_zrange(prim, metric, K, dx, nghost, recon, gamma, out, 0, nghost, stream=stream)
    grx.valencia_rhs_zrange(prim, metric, K, dx, nghost, recon, gamma, out, nz - nghost, nz, stream=stream)
    return out


def step_rk2_zslabs(exch, cons, prim, metric, K, dx, nghost, recon, gamma, dt, nsteps, work, overlap=True, nfail=None,
                    stream=None):
    """`nsteps` SSP-RK2 steps (R21) of this rank's slab of a domain that is periodic in x, y (per rank) and z (over the
    ring): per stage  L = rhs_overlapped(prim);  U <- a U0 + b (U + dt L) fused with con2prim (grx_rk_stage);  x / y ghost
    fill (grx_fill_ghosts, dirs = 3).  `prim` must come with filled x / y ghosts; its z ghosts are exchanged here.
    work: two arrays shaped like cons (U1 and L)."""
    from . import grx
    if stream is not None and cons.is_cuda:
        import torch
        if stream != torch.cuda.current_stream(cons.device):
            # any torch operation a caller's pack / unpack hooks issue goes to torch's current stream: make `stream` that one
            with torch.cuda.stream(stream):
                return step_rk2_zslabs(exch, cons, prim, metric, K, dx, nghost, recon, gamma, dt, nsteps, work, overlap,
                                       nfail, stream)
    U1, L = work
    for _ in range(nsteps):
        # cons keeps U^n until the second stage overwrites it; U1 goes to the first work array (no copy of cons per step)
        rhs_overlapped(exch, prim, metric, K, dx, nghost, recon, gamma, L, overlap, stream)
        grx.rk_stage(nghost, 0.0, cons, 1.0, cons, dt, L, U1, metric, gamma, prim, nfail=nfail, stream=stream)
        grx.fill_ghosts(prim, nghost, "periodic", 3, stream=stream)
        rhs_overlapped(exch, prim, metric, K, dx, nghost, recon, gamma, L, overlap, stream)
        grx.rk_stage(nghost, 0.5, cons, 0.5, U1, dt, L, cons, metric, gamma, prim, nfail=nfail, stream=stream)
        grx.fill_ghosts(prim, nghost, "periodic", 3, stream=stream)
    # leave prim with consistent z ghosts
    exch.start(prim, stream)
    exch.finish(prim, stream)
    return cons, prim
