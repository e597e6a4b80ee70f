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
