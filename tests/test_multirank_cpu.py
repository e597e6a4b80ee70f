"""The N > 1 host logic of bench.py (paper_1107_5463_b200/ranks.py) under a real world_size-2 process group on CPU
(gloo): per-rank seeds give independent lattices, the timed region is the slowest rank's, the metric sums the updates
of all ranks.  There is no data-path collective to test: the path shards by independent lattices.
The lattices themselves are driven here by the oracle, standing in for the GPU handle (no GPU in this test)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist

    import oracle
    from paper_1107_5463_b200 import ranks, workloads

    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        seed = ranks.rank_seed(workloads.SEED, rank)
        S = oracle.System((16, 16, 1), seed=seed)
        S.sweep(0.4406868, 3)
        E, M = S.measure()
        spins = S.get_spins()
        # pretend rank r needed (10 + 5 r) ms for 1e6 updates
        value, ms = ranks.whole_job_flips_per_ns(1e6, 10.0 + 5.0 * rank, dist)
        mx = ranks.max_over_ranks(float(rank), dist)
        out.put((rank, seed, float(E[0]), spins.tobytes(), value, ms, mx))
    finally:
        dist.destroy_process_group()


def test_world_size_two_gloo():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, e0, sp0, v0, ms0, mx0), (r1, s1, e1, sp1, v1, ms1, mx1) = res
    assert (r0, r1) == (0, 1) and s1 == s0 + 1
    assert sp0 != sp1, "ranks must simulate different lattices"
    # slowest rank defines the time; both ranks' updates count
    assert ms0 == ms1 == 15.0 and mx0 == mx1 == 1.0
    assert v0 == v1 == pytest.approx(2e6 / (15.0 * 1e6))


def test_single_process_defaults():
    sys.path.insert(0, ROOT)
    from paper_1107_5463_b200 import ranks

    assert ranks.max_over_ranks(3.5) == 3.5
    v, ms = ranks.whole_job_flips_per_ns(4e6, 2.0)
    assert ms == 2.0 and v == pytest.approx(2.0)
    assert ranks.rank_seed(7, 3) == 10


# --------------------------------------------------------------------------- slab decomposition: who sends what to whom
def _slab_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    from paper_1107_5463_b200 import slab

    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        # a fake slab: owned planes hold 10 * rank + plane index, ghosts start at -1
        own = 4
        planes = {c: torch.full((own + 4, 3), -1.0) for c in (0, 1)}
        for c in (0, 1):
            for p in range(own):
                planes[c][2 + p] = 100.0 * c + 10.0 * rank + p

        def get_face(colour, side):
            return planes[colour][2 if side == 0 else own + 1].clone()

        def put_face(colour, side, t):
            planes[colour][1 if side == 0 else own + 2] = t

        for c in (0, 1):
            slab.exchange_faces(get_face, put_face, c, dist, rank, world)
        out.put((rank, {c: (planes[c][1, 0].item(), planes[c][own + 2, 0].item()) for c in (0, 1)}))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_slab_halo_exchange_ring_gloo(world):
    """exchange_faces over a real process group: my lower ghost = highest plane of the rank below, my upper ghost =
    lowest plane of the rank above (periodic), for both colours; world 2 (both neighbours are the same rank) and 3."""
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_slab_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    own = 4
    for r in range(world):
        below, above = (r - 1) % world, (r + 1) % world
        for c in (0, 1):
            low_ghost, high_ghost = res[r][c]
            assert low_ghost == 100.0 * c + 10.0 * below + (own - 1)
            assert high_ghost == 100.0 * c + 10.0 * above + 0


def test_slab_plan():
    sys.path.insert(0, ROOT)
    from paper_1107_5463_b200 import slab

    assert slab.plan((512, 512, 512), 8) == [((512, 512, 64), 64 * k) for k in range(8)]
    assert slab.plan((16384, 16384), 4)[3] == ((16384, 4096, 1), 12288)
    assert slab.ring_neighbours(0, 4) == (3, 1) and slab.ring_neighbours(3, 4) == (2, 0)
    with pytest.raises(ValueError):
        slab.plan((64, 64, 6), 2)


class _OracleSlab:
    """A slab handle on the CPU with the slab calls of binding.SpinSystem (halfsweep, halfsweep_range, halo_pack / unpack,
    halo_bytes, measure, get_spins), standing in for the GPU handle so that DistRing runs end to end under gloo.  2D Ising,
    J = +1, cut along y; rows are kept in the canonical layout with two ghost rows on either side, and every decision is the
    oracle's own (oracle.ising_uniform / oracle.threshold on GLOBAL site indices), one site at a time."""

    def __init__(self, local_dims, slab_global=0, slab_offset=0, device="cpu", seed=0, full_hot_start=None):
        import oracle

        self.o = oracle
        self.Lx, self.own, self.Ly, self.off, self.seed = local_dims[0], local_dims[1], slab_global, slab_offset, seed
        self.n, self.R, self.t, self.next = 1, 1, 0, 0
        full = oracle.System((self.Lx, self.Ly, 1), seed=seed).get_spins()[0].reshape(self.Ly, self.Lx)
        self.rows = np.zeros((self.own + 4, self.Lx), dtype=np.int8)            # local row p = global row off - 2 + p
        self.rows[2:2 + self.own] = full[self.off:self.off + self.own]

    def halo_bytes(self):
        return self.Lx

    def halo_pack(self, colour, buf):
        import torch

        buf.copy_(torch.from_numpy(np.concatenate([self.rows[2], self.rows[1 + self.own]]).view(np.uint8)))

    def halo_unpack(self, colour, buf):
        v = buf.numpy().view(np.int8)
        self.rows[1] = v[:self.Lx]                  # from the slab below: its highest row
        self.rows[2 + self.own] = v[self.Lx:]       # from the slab above: its lowest row

    def halfsweep_range(self, beta, colour, plane0, n_planes, last):
        assert colour == self.next
        Lx = self.Lx
        T = {dE: self.o.threshold(beta, dE) for dE in (4, 8)}
        for p in range(2 + plane0, 2 + plane0 + n_planes):
            y = (self.off - 2 + p) % self.Ly
            for x in range(Lx):
                if (x + y) & 1 != colour:
                    continue
                s = int(self.rows[p, x])
                h = int(self.rows[p, (x - 1) % Lx]) + int(self.rows[p, (x + 1) % Lx]) + int(self.rows[p - 1, x]) + int(self.rows[p + 1, x])
                dE = 2 * s * h
                j = (x >> 1) + (Lx // 2) * y
                if dE <= 0 or self.o.ising_uniform(self.seed, j, 0, self.t, colour) < T[dE]:
                    self.rows[p, x] = -s
        if last:
            self.next = 1 - colour
            self.t += colour

    def halfsweep(self, beta, colour):
        self.halfsweep_range(beta, colour, 0, self.own, True)

    def measure(self):
        own = self.rows[2:2 + self.own].astype(np.int64)
        up = self.rows[3:3 + self.own].astype(np.int64)                         # row y + 1 (the last one is the ghost above)
        E = -float((own * np.roll(own, -1, axis=1)).sum() + (own * up).sum())
        return np.array([E]), np.array([[float(own.sum())]])

    def get_spins(self):
        return self.rows[2:2 + self.own].copy()


def _dist_ring_worker(rank, world, port, overlap, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist

    from paper_1107_5463_b200 import slab

    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        ring = slab.DistRing(_OracleSlab, (16, 24, 1), dist, "cpu", overlap=overlap, seed=77)
        ring.sweep(0.4406868, 3)
        E, M = ring.measure()
        out.put((rank, ring.system.get_spins().tobytes(), float(E[0]), float(M[0, 0]), ring.comm_bytes))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,overlap", [(2, True), (3, True), (2, False)])
def test_dist_ring_end_to_end_gloo(world, overlap):
    """slab.DistRing over a real process group with the oracle standing in for the handle: boundary planes first, packed
    exchange with the ring neighbours, interior, unpack -- the slabs together must equal the unsharded oracle lattice bit
    for bit after every rank's three sweeps, E and M (all-reduced) must be the lattice's, and every rank sends two faces
    each way per half-sweep."""
    import torch.multiprocessing as mp

    sys.path.insert(0, ROOT)
    import oracle

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_dist_ring_worker, args=(r, world, port, overlap, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = {r[0]: r[1:] for r in (q.get(timeout=180) for _ in procs)}
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    O = oracle.System((16, 24, 1), seed=77)
    O.sweep(0.4406868, 3)
    want = O.get_spins()[0].reshape(24, 16)
    own = 24 // world
    got = np.concatenate([np.frombuffer(res[r][0], dtype=np.int8).reshape(own, 16) for r in range(world)])
    assert np.array_equal(got, want)
    E, M = O.measure()
    for r in range(world):
        assert res[r][1] == E[0] and res[r][2] == M[0, 0]
        assert res[r][3] == (2 + 2 * 3) * 2 * 16, "two initial exchanges + one per half-sweep, two faces of 16 bytes each"
