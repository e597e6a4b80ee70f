"""Slab decomposition on ONE GPU: the slabs of a lattice as separate libspin handles that
exchange boundary planes between half-sweeps (paper_1107_5463_b200/slab.py LocalRing) must reproduce the unsharded
lattice: bit for bit against the oracle for n = 1, bit for bit against the single-handle run for n >= 2."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1107_5463_b200 as pkg

    pkg.lib()
    return pkg


ISING = [
    # dims, storage, J, R, streams, rule, slab counts
    ((64, 16, 1), "int8", 1.0, 1, 0, "metropolis", (1, 2, 4)),      # int8 strip kernel, y slabs
    ((128, 24, 1), "bitpack", 1.0, 2, 1, "metropolis", (2, 3, 6)),  # bit-packed, y slabs, own stream per replica
    ((64, 6, 8), "int8", -1.0, 1, 0, "metropolis", (2, 4)),         # 3D z slabs, antiferromagnet
    ((64, 4, 12), "bitpack", 1.0, 3, 0, "heatbath", (2, 3)),        # shared stream, heat bath
    ((10, 8, 1), "int8", 1.0, 1, 0, "metropolis", (2, 4)),          # generic kernel (Lx % 64 != 0), slabs of 2 rows
    ((6, 4, 8), "int8", 1.0, 2, 1, "heatbath", (2,)),
]


@pytest.mark.parametrize("dims,storage,J,R,streams,rule,counts", ISING)
def test_ising_slabs_reproduce_the_whole_lattice(P, oracle, dims, storage, J, R, streams, rule, counts):
    from paper_1107_5463_b200 import slab

    beta = 0.4406868 if dims[2] == 1 else 0.2216546
    O = oracle.System(dims, J=(J, J, J), n_replicas=R, replica_streams=streams, seed=77,
                      rule=oracle.RULE_HEATBATH if rule == "heatbath" else oracle.RULE_METROPOLIS)
    want0 = O.get_spins()
    O.sweep(beta, 4)
    want, (Eo, Mo) = O.get_spins(), O.measure()
    for G in counts:
        ring = slab.LocalRing(P.SpinSystem, dims, G, storage=storage, J=(J, J, J), replicas=R, replica_streams=streams,
                              seed=77, rule=rule)
        assert np.array_equal(ring.get_spins(), want0), ("hot start", G)
        ring.sweep(beta, 4)
        assert np.array_equal(ring.get_spins(), want), ("spins", G)
        E, M = ring.measure()
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo), (G, E, Eo)
        # set_spins on slabs + continue: same as the oracle continuing
        ring.set_spins(want)
        ring.sweep(beta, 1)
        O2 = oracle.System(dims, J=(J, J, J), n_replicas=R, replica_streams=streams, seed=77,
                           rule=oracle.RULE_HEATBATH if rule == "heatbath" else oracle.RULE_METROPOLIS)
        O2.set_spins(want)
        O2.sweep_counter = 4
        O2.sweep(beta, 1)
        assert np.array_equal(ring.get_spins(), O2.get_spins()), ("after set_spins", G)
        ring.close()


@pytest.mark.parametrize("n,dims,rule,counts", [(3, (16, 8, 8), "metropolis", (2, 4)), (2, (16, 12, 1), "metropolis", (2, 3)),
                                                (3, (8, 4, 4), "heatbath", (2,)), (3, (6, 4, 8), "metropolis", (2,))])
def test_vector_slabs_match_the_single_handle_bitwise(P, oracle, n, dims, rule, counts):
    from paper_1107_5463_b200 import slab

    beta = 0.693
    ref = P.SpinSystem(dims, n=n, storage="fp32", seed=5, rule=rule)
    ref.sweep(beta, 3)
    want = ref.get_spins()
    Er, Mr = ref.measure()
    for G in counts:
        ring = slab.LocalRing(P.SpinSystem, dims, G, n=n, storage="fp32", seed=5, rule=rule)
        ring.sweep(beta, 3)
        assert np.array_equal(ring.get_spins().view(np.uint32), want.view(np.uint32)), G
        E, M = ring.measure()
        assert np.allclose(E, Er, rtol=1e-12, atol=1e-9) and np.allclose(M, Mr, rtol=1e-12, atol=1e-9)
        ring.close()


def test_slab_handles_refuse_whole_sweeps_and_bad_plans(P):
    from paper_1107_5463_b200 import slab

    S = P.SpinSystem((64, 8, 1), slab_global=16, slab_offset=8)
    with pytest.raises(P.SpinError):
        S.sweep(0.4, 1)
    S.halfsweep(0.4, 0)
    with pytest.raises(P.SpinError):
        S.halfsweep(0.4, 0)          # colours alternate
    S.halfsweep(0.4, 1)
    assert S.sweep_counter == 1
    assert S.halo_bytes() == 32      # one row of one colour: 32 int8 sites
    with pytest.raises(P.SpinError):
        P.SpinSystem((64, 8, 1), slab_global=16, slab_offset=3)
    with pytest.raises(P.SpinError):
        P.SpinSystem((64, 8, 1), slab_global=12, slab_offset=8)
    with pytest.raises(ValueError):
        slab.plan((64, 12, 1), 4)    # slabs of 3 rows are not even
    U = P.SpinSystem((64, 8, 1))
    with pytest.raises(P.SpinError):
        U.halo_bytes()


@pytest.mark.parametrize("kw,dims", [
    (dict(n=1, storage="int8"), (128, 24, 1)), (dict(n=1, storage="bitpack"), (128, 20, 1)),
    (dict(n=1, storage="int8"), (64, 6, 10)), (dict(n=1, storage="bitpack", rule="heatbath"), (64, 6, 8)),
    (dict(n=1, storage="int8"), (10, 12, 1)), (dict(n=3, storage="fp32"), (16, 8, 10)), (dict(n=2, storage="fp32"), (16, 14, 1)),
    (dict(n=3, storage="fp32"), (6, 6, 8)),
])
def test_half_sweeps_in_pieces_equal_whole_half_sweeps(P, kw, dims):
    """spin_halfsweep_range: sites of one colour do not interact, so a half-sweep issued as boundary planes first and the
    interior afterwards (the order the overlapped halo exchange needs) leaves the bits of the whole half-sweep -- for the
    strip kernels (ragged strips inside the range), the word kernels and the one-thread-per-site kernels."""
    beta = 0.5
    A, B = P.SpinSystem(dims, seed=21, **kw), P.SpinSystem(dims, seed=21, **kw)
    planes = dims[2] if dims[2] > 1 else dims[1]
    for t in range(3):
        for c in (0, 1):
            A.halfsweep(beta, c)
            B.halfsweep_range(beta, c, 0, 1, False)
            B.halfsweep_range(beta, c, planes - 1, 1, False)
            B.halfsweep_range(beta, c, 1, 3, False)
            B.halfsweep_range(beta, c, 4, planes - 5, True)
    assert A.sweep_counter == B.sweep_counter == 3
    assert np.array_equal(A.get_spins().view(np.uint8), B.get_spins().view(np.uint8))
    with pytest.raises(P.SpinError):
        B.halfsweep_range(beta, 0, planes - 1, 2, True)


@pytest.mark.parametrize("dims,storage,overlap", [((128, 32, 1), "int8", True), ((64, 8, 12), "bitpack", True),
                                                  ((128, 32, 1), "bitpack", False)])
def test_dist_ring_single_rank_on_the_gpu(P, dims, storage, overlap):
    """slab.DistRing with the real handle and a one-rank NCCL group: the slab is its own neighbour (spin_halo_wrap), and
    with two pseudo-neighbours forced through the packed path (world 1 copies its faces) it still equals the oracle."""
    import torch
    import torch.distributed as dist

    import oracle
    from paper_1107_5463_b200 import slab

    created = False
    if not dist.is_initialized():
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:29533", rank=0, world_size=1,
                                device_id=torch.device("cuda:0"))
        created = True
    try:
        ring = slab.DistRing(P.SpinSystem, dims, dist, "cuda:0", overlap=overlap, n=1, storage=storage, seed=5)
        O = oracle.System(dims, n=1, seed=5)
        ring.sweep(0.44, 4)
        O.sweep(0.44, 4)
        assert np.array_equal(ring.system.get_spins(), O.get_spins())
        E, M = ring.measure()
        Eo, Mo = O.measure()
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
        # the packed path as a rank with neighbours would run it: boundary planes, pack, exchange, interior, unpack
        s = ring.system
        for c in (0, 1):
            s.halfsweep_range(0.44, c, 0, 1, False)
            s.halfsweep_range(0.44, c, ring.own - 1, 1, False)
            s.halo_pack(c, ring.send)
            slab.exchange_packed(ring.send, ring.recv, dist, 0, 1)
            s.halfsweep_range(0.44, c, 1, ring.own - 2, True)
            s.halo_unpack(c, ring.recv)
        O.sweep(0.44, 1)
        assert np.array_equal(s.get_spins(), O.get_spins())
    finally:
        if created:
            dist.destroy_process_group()


def test_exchange_cost_of_a_self_exchanging_slab(P):
    """SURVEY 8(e) / VERDICT item 10: the halo exchange costs one small kernel per half-sweep (it was four strided copies
    driven from Python, 16 us).  2D L = 16384 int8 as ONE slab that is its own neighbour against the plain handle."""
    import torch

    from paper_1107_5463_b200 import slab

    dims, beta, sweeps = (16384, 16384, 1), 0.4406868, 10
    A = P.SpinSystem(dims, n=1, storage="int8", seed=1)
    A.set_option(P.OPT_TEMPORAL_BLOCKING, 0)
    ring = slab.LocalRing(P.SpinSystem, dims, 1, n=1, storage="int8", seed=1)

    def timed(fn):
        fn(2)
        best = 1e30
        for _ in range(3):                       # best of three: the assertion below is about cost, not about noise
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn(sweeps)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, 1e3 * e0.elapsed_time(e1) / (2 * sweeps))
        return best

    plain = timed(lambda k: A.sweep(beta, k))
    slabbed = timed(lambda k: ring.sweep(beta, k))
    print("half-sweep %.1f us, with self-exchange %.1f us" % (plain, slabbed))
    assert slabbed - plain <= 5.0, (plain, slabbed)
    assert A.sweep_counter == ring.systems[0].sweep_counter
    assert np.array_equal(A.get_spins(), ring.get_spins())


@pytest.mark.parametrize("dims,kw,G", [((128, 24, 1), dict(n=1, storage="int8"), 3), ((64, 6, 12), dict(n=1, storage="bitpack", replicas=2, replica_streams=1), 2),
                                       ((16, 8, 12), dict(n=3, storage="fp32"), 3), ((10, 12, 1), dict(n=1, storage="int8"), 2)])
def test_peer_stores_and_packed_messages_agree(P, dims, kw, G):
    """The two halo paths -- spin_halo_push (boundary planes stored straight into the neighbours' ghost planes) and the packed
    messages DistRing sends (spin_halo_pack / copy / spin_halo_unpack) -- leave identical slabs, equal to the single handle."""
    from paper_1107_5463_b200 import slab

    beta = 0.5
    A = slab.LocalRing(P.SpinSystem, dims, G, peer_stores=True, seed=8, **kw)
    B = slab.LocalRing(P.SpinSystem, dims, G, peer_stores=False, seed=8, **kw)
    W = P.SpinSystem(dims, seed=8, **kw)
    assert A.peer_stores and not B.peer_stores
    for S in (A, B, W):
        S.sweep(beta, 5)
    a, b, w = A.get_spins(), B.get_spins(), W.get_spins()
    assert np.array_equal(a.view(np.uint8), w.view(np.uint8)) and np.array_equal(b.view(np.uint8), w.view(np.uint8))
    A.close()
    B.close()
