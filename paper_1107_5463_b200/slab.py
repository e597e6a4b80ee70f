"""Slab decomposition of one lattice over several handles / GPUs.

The lattice is cut along its slowest axis (z for d = 3, y for d = 2) into equal slabs of an even number of planes; every
slab is one libspin handle created with `slab_global` / `slab_offset` (include/spin.h).  Before the half-sweep of
colour c each slab needs its two neighbours' boundary planes of colour 1 - c: ONE exchange step per half-sweep, the
only data-path communication of the method.  Random numbers are keyed by global site indices, so the slabs together
reproduce the unsharded lattice bit for bit, for any number of slabs.

This module holds the plumbing only (who sends which face to whom); every arithmetic step runs in the library.
  LocalRing  all slabs on ONE device (tests, and the way to check the decomposition on a single GPU)
  DistRing   one slab per rank, faces exchanged with torch.distributed point-to-point calls (NCCL over NVLink on a
             multi-GPU node; the same code runs on gloo with CPU tensors in the CPU test)
"""
import numpy as np


def slab_axis(dims):
    dims = tuple(dims) + (1,) * (3 - len(dims))
    return 2 if dims[2] > 1 else 1


def plan(global_dims, n_slabs):
    """[(local_dims, offset)] for n_slabs equal slabs; the extent along the slab axis must divide into even slabs."""
    dims = [int(v) for v in global_dims] + [1] * (3 - len(global_dims))
    ax = slab_axis(dims)
    L = dims[ax]
    if n_slabs < 1 or L % (2 * n_slabs) != 0:
        raise ValueError("extent %d along the slab axis does not split into %d slabs of an even thickness" % (L, n_slabs))
    own = L // n_slabs
    out = []
    for k in range(n_slabs):
        local = list(dims)
        local[ax] = own
        out.append((tuple(local), k * own))
    return out


def ring_neighbours(rank, world):
    """(rank that owns the planes below mine, rank that owns the planes above mine), periodic"""
    return (rank - 1) % world, (rank + 1) % world


class LocalRing:
    """All slabs of one lattice as separate handles on one device; halos move by peer stores (spin_halo_push: every slab
    writes its boundary planes straight into its neighbours' ghost planes, one kernel per slab) or, with
    peer_stores=False, through the packed message buffers DistRing sends (one pack and one unpack kernel per slab and
    exchange); a single slab wraps onto itself with one kernel."""

    def __init__(self, system_cls, global_dims, n_slabs, peer_stores=True, **kw):
        import torch

        self.dims = tuple(int(v) for v in global_dims) + (1,) * (3 - len(global_dims))
        self.axis = slab_axis(self.dims)
        self.parts = plan(self.dims, n_slabs)
        self.systems = [system_cls(local, slab_global=self.dims[self.axis], slab_offset=off, **kw)
                        for local, off in self.parts]
        s0 = self.systems[0]
        self.peer_stores = bool(peer_stores) and hasattr(s0, "halo_push")
        self.n, self.R = s0.n, s0.R
        self.N = self.dims[0] * self.dims[1] * self.dims[2]
        self.hb = s0.halo_bytes()
        self.send = [torch.empty(2 * self.hb, dtype=torch.uint8, device=s0.device) for _ in self.systems]
        self.recv = [torch.empty(2 * self.hb, dtype=torch.uint8, device=s0.device) for _ in self.systems]
        self.exchange(0)
        self.exchange(1)

    def exchange(self, colour):
        G, hb = len(self.systems), self.hb
        if G == 1:
            self.systems[0].halo_wrap(colour)
            return
        if self.peer_stores:
            # every slab stores its boundary planes straight into its neighbours' ghost planes (one kernel per slab; all
            # slabs share the stream here, which orders the pushes before the half-sweeps that read the ghosts)
            ptrs = [s.colour_array(colour)[0] for s in self.systems]
            for k, s in enumerate(self.systems):
                below, above = ring_neighbours(k, G)
                s.halo_push(colour, ptrs[below], ptrs[above])
            return
        for k, s in enumerate(self.systems):
            s.halo_pack(colour, self.send[k])                  # [my lowest owned plane][my highest]
        for k, s in enumerate(self.systems):
            below, above = ring_neighbours(k, G)
            self.recv[k][:hb].copy_(self.send[below][hb:])     # ghost below me = highest plane of the slab below
            self.recv[k][hb:].copy_(self.send[above][:hb])     # ghost above me = lowest plane of the slab above
            s.halo_unpack(colour, self.recv[k])

    def sweep(self, beta, n_sweeps=1):
        for _ in range(int(n_sweeps)):
            for c in (0, 1):
                for s in self.systems:
                    s.halfsweep(beta, c)
                self.exchange(c)

    def measure(self):
        E, M = None, None
        for s in self.systems:
            e, m = s.measure()
            E, M = (e, m) if E is None else (E + e, M + m)
        return E, M

    def get_spins(self):
        ax = self.axis
        shp = lambda d: (self.R, d[2], d[1], d[0]) + ((self.n,) if self.n > 1 else ())
        parts = [s.get_spins().reshape(shp(local)) for s, (local, _) in zip(self.systems, self.parts)]
        full = np.concatenate(parts, axis=1 if ax == 2 else 2)
        return full.reshape((self.R, self.N) + ((self.n,) if self.n > 1 else ()))

    def set_spins(self, spins):
        ax = self.axis
        d = self.dims
        full = np.asarray(spins).reshape((self.R, d[2], d[1], d[0]) + ((self.n,) if self.n > 1 else ()))
        for s, (local, off) in zip(self.systems, self.parts):
            sl = [slice(None)] * full.ndim
            sl[1 if ax == 2 else 2] = slice(off, off + local[ax])
            s.set_spins(np.ascontiguousarray(full[tuple(sl)]).reshape(self.R, -1, *(() if self.n == 1 else (self.n,))))
        self.exchange(0)
        self.exchange(1)

    def close(self):
        for s in self.systems:
            s.close()


def exchange_packed(send, recv, dist, rank, world):
    """One halo exchange for the slab of this rank.  send = [my lowest owned plane][my highest] (two halves of one
    contiguous tensor), recv = [ghost below me][ghost above me]: my lowest plane goes to the rank below (as its upper
    ghost), my highest plane to the rank above (as its lower ghost).  The only data-path communication of the method:
    point-to-point, ring neighbours, 2 x halo_bytes each way per half-sweep."""
    hb = send.numel() // 2
    low, high = send[:hb], send[hb:]
    from_below, from_above = recv[:hb], recv[hb:]
    if world == 1:
        from_below.copy_(high)
        from_above.copy_(low)
        return
    below, above = ring_neighbours(rank, world)
    if world == 2:
        # both neighbours are the same rank: two messages each way, told apart by their tags
        ops = [dist.P2POp(dist.isend, low, below, tag=0), dist.P2POp(dist.isend, high, above, tag=1),
               dist.P2POp(dist.irecv, from_above, above, tag=0), dist.P2POp(dist.irecv, from_below, below, tag=1)]
    else:
        ops = [dist.P2POp(dist.isend, low, below), dist.P2POp(dist.isend, high, above),
               dist.P2POp(dist.irecv, from_above, above), dist.P2POp(dist.irecv, from_below, below)]
    for w in dist.batch_isend_irecv(ops):
        w.wait()


def exchange_faces(get_face, put_face, colour, dist, rank, world):
    """The same exchange through per-face callbacks (get_face(colour, side) -> tensor, put_face(colour, side, tensor))."""
    import torch

    low, high = get_face(colour, 0), get_face(colour, 1)
    send = torch.cat([low.reshape(-1), high.reshape(-1)])
    recv = torch.empty_like(send)
    exchange_packed(send, recv, dist, rank, world)
    hb = low.numel()
    put_face(colour, 1, recv[hb:].reshape(low.shape))     # the lowest plane of the slab above me is my upper ghost
    put_face(colour, 0, recv[:hb].reshape(high.shape))


class DistRing:
    """One slab per rank (one process per GPU); the N ranks together hold ONE lattice (strong scaling).

    Per half-sweep of colour c: the two boundary planes of the slab are updated first and packed; their exchange runs on
    a side stream while the interior planes are updated on the main stream; the ghosts are unpacked when both are done
    ("overlap by updating boundary planes first").  `system` may be any object with the slab calls of
    binding.SpinSystem (the CPU test drives the ring with an oracle-backed stand-in over gloo)."""

    def __init__(self, system_cls, global_dims, dist, device, overlap=True, **kw):
        import torch

        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.dims = tuple(int(v) for v in global_dims) + (1,) * (3 - len(global_dims))
        local, off = plan(self.dims, self.world)[self.rank]
        self.own = local[slab_axis(self.dims)]
        self.system = system_cls(local, slab_global=self.dims[slab_axis(self.dims)], slab_offset=off, device=device, **kw)
        self.hb = self.system.halo_bytes()
        self.device = torch.device(device)
        self.cuda = self.device.type == "cuda"
        self.send = torch.empty(2 * self.hb, dtype=torch.uint8, device=device)
        self.recv = torch.empty(2 * self.hb, dtype=torch.uint8, device=device)
        self.overlap = bool(overlap) and self.own >= 4
        self.side = torch.cuda.Stream(device=self.device) if self.cuda else None
        self.comm_bytes = 0          # bytes this rank has sent
        self.exchange(0)
        self.exchange(1)

    def _communicate(self):
        """send -> neighbours -> recv, on the side stream when there is one"""
        import torch

        if self.side is None:
            exchange_packed(self.send, self.recv, self.dist, self.rank, self.world)
        else:
            main = torch.cuda.current_stream(self.device)
            self.side.wait_stream(main)                    # the pack kernel has been enqueued on the main stream
            with torch.cuda.stream(self.side):
                exchange_packed(self.send, self.recv, self.dist, self.rank, self.world)
            main.wait_stream(self.side)
        self.comm_bytes += 2 * self.hb

    def exchange(self, colour):
        if self.world == 1 and hasattr(self.system, "halo_wrap"):
            self.system.halo_wrap(colour)
            return
        self.system.halo_pack(colour, self.send)
        self._communicate()
        self.system.halo_unpack(colour, self.recv)

    def halfsweep(self, beta, colour):
        import torch

        s = self.system
        if not self.overlap or self.world == 1:
            s.halfsweep(beta, colour)
            self.exchange(colour)
            return
        s.halfsweep_range(beta, colour, 0, 1, False)                   # lowest owned plane
        s.halfsweep_range(beta, colour, self.own - 1, 1, False)        # highest owned plane
        s.halo_pack(colour, self.send)
        if self.side is None:
            exchange_packed(self.send, self.recv, self.dist, self.rank, self.world)
            s.halfsweep_range(beta, colour, 1, self.own - 2, True)
        else:
            main = torch.cuda.current_stream(self.device)
            self.side.wait_stream(main)
            with torch.cuda.stream(self.side):
                exchange_packed(self.send, self.recv, self.dist, self.rank, self.world)
            s.halfsweep_range(beta, colour, 1, self.own - 2, True)      # interior, while the messages are in flight
            main.wait_stream(self.side)
        self.comm_bytes += 2 * self.hb
        s.halo_unpack(colour, self.recv)

    def sweep(self, beta, n_sweeps=1):
        for _ in range(int(n_sweeps)):
            for c in (0, 1):
                self.halfsweep(beta, c)

    def measure(self):
        """E and M of the whole lattice (sum over ranks)."""
        import torch

        E, M = self.system.measure()
        t = torch.from_numpy(np.concatenate([E.ravel(), M.ravel()])).to(self.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        v = t.cpu().numpy()
        return v[: E.size].reshape(E.shape), v[E.size:].reshape(M.shape)
