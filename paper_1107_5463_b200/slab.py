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
    """All slabs of one lattice as separate handles on one device; halos move by device-to-device copies."""

    def __init__(self, system_cls, global_dims, n_slabs, **kw):
        import torch

        self.dims = tuple(int(v) for v in global_dims) + (1,) * (3 - len(global_dims))
        self.axis = slab_axis(self.dims)
        self.parts = plan(self.dims, n_slabs)
        self.systems = [system_cls(local, slab_global=self.dims[self.axis], slab_offset=off, **kw)
                        for local, off in self.parts]
        s0 = self.systems[0]
        self.n, self.R = s0.n, s0.R
        self.N = self.dims[0] * self.dims[1] * self.dims[2]
        self.buf = torch.empty(s0.halo_bytes(), dtype=torch.uint8, device=s0.device)
        self.exchange(0)
        self.exchange(1)

    def exchange(self, colour):
        G = len(self.systems)
        for k, s in enumerate(self.systems):
            below, above = ring_neighbours(k, G)
            s.halo_get(colour, 0, self.buf)                   # my lowest owned plane ...
            self.systems[below].halo_put(colour, 1, self.buf)  # ... is the ghost above the slab below me
            s.halo_get(colour, 1, self.buf)
            self.systems[above].halo_put(colour, 0, self.buf)

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


def exchange_faces(get_face, put_face, colour, dist, rank, world):
    """One halo exchange of colour `colour` for the slab of this rank.  get_face(colour, side) -> contiguous tensor with my
    boundary plane; put_face(colour, side, tensor) stores a neighbour's plane as my ghost.  My lowest plane goes to the
    rank below (as its upper ghost), my highest plane to the rank above (as its lower ghost)."""
    import torch

    low, high = get_face(colour, 0), get_face(colour, 1)
    if world == 1:
        put_face(colour, 1, low)
        put_face(colour, 0, high)
        return
    below, above = ring_neighbours(rank, world)
    from_above, from_below = torch.empty_like(low), torch.empty_like(high)
    if world == 2:
        # both neighbours are the same rank: two messages each way, told apart by their tags
        ops = [dist.P2POp(dist.isend, low, below, tag=0), dist.P2POp(dist.isend, high, above, tag=1),
               dist.P2POp(dist.irecv, from_above, above, tag=0), dist.P2POp(dist.irecv, from_below, below, tag=1)]
    else:
        ops = [dist.P2POp(dist.isend, low, below), dist.P2POp(dist.isend, high, above),
               dist.P2POp(dist.irecv, from_above, above), dist.P2POp(dist.irecv, from_below, below)]
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    put_face(colour, 1, from_above)    # the lowest plane of the slab above me is my upper ghost
    put_face(colour, 0, from_below)


class DistRing:
    """One slab per rank (one process per GPU); the N ranks together hold ONE lattice (strong scaling)."""

    def __init__(self, system_cls, global_dims, dist, device, **kw):
        import torch

        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.dims = tuple(int(v) for v in global_dims) + (1,) * (3 - len(global_dims))
        local, off = plan(self.dims, self.world)[self.rank]
        self.system = system_cls(local, slab_global=self.dims[slab_axis(self.dims)], slab_offset=off, device=device, **kw)
        nbytes = self.system.halo_bytes()
        self._bufs = [torch.empty(nbytes, dtype=torch.uint8, device=device) for _ in range(2)]
        self.exchange(0)
        self.exchange(1)

    def _get(self, colour, side):
        self.system.halo_get(colour, side, self._bufs[side])
        return self._bufs[side]

    def _put(self, colour, side, t):
        self.system.halo_put(colour, side, t)

    def exchange(self, colour):
        exchange_faces(self._get, self._put, colour, self.dist, self.rank, self.world)

    def sweep(self, beta, n_sweeps=1):
        for _ in range(int(n_sweeps)):
            for c in (0, 1):
                self.system.halfsweep(beta, c)
                self.exchange(c)

    def measure(self):
        """E and M of the whole lattice (sum over ranks)."""
        import torch

        E, M = self.system.measure()
        t = torch.from_numpy(np.concatenate([E.ravel(), M.ravel()])).to(self._bufs[0].device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        v = t.cpu().numpy()
        return v[: E.size].reshape(E.shape), v[E.size:].reshape(M.shape)
