"""The deferred digit comparison (DESIGN R-16; bit-packed / int8 strip kernels, own-stream +-J kernel): a thread makes two
unconditional Philox calls per word and pushes a word with undecided lanes onto a per-warp queue in shared memory; a full
queue (about once in 10^6 warps at the default capacity of 32) makes the thread finish the word itself.  SPIN_OPT_DEFER_CAP
shrinks the queue so that this overflow path runs for most words: the spins must stay EXACTLY the oracle's, whatever the
capacity (0 = everything inline, 1 and 5 = a mix of queued and inline words in every warp, 32 = default)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SEED = 11075463


@pytest.fixture(scope="module")
def P():
    import paper_1107_5463_b200 as pkg
    pkg.lib()
    return pkg


@pytest.fixture(scope="module")
def oracle():
    import oracle as o
    return o


def _equal(G, O, tag):
    bad = int(np.count_nonzero(G.get_spins() != O.get_spins()))
    assert bad == 0, "%s: %d spins differ" % (tag, bad)
    Eg, Mg = G.measure()
    Eo, Mo = O.measure()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo), (tag, Eg, Eo)


CASES = [
    # dims, storage, coupling, R, rule, beta
    ((512, 24, 1), "bitpack", "uniform", 2, "metropolis", 0.4406868),    # bit-packed strip kernel, 2D
    ((512, 24, 1), "bitpack", "uniform", 2, "heatbath", 0.4406868),
    ((256, 10, 6), "bitpack", "uniform", 1, "metropolis", 0.2216544),    # 3D, ragged strips
    ((256, 10, 6), "bitpack", "uniform", 2, "heatbath", 0.2216544),
    ((512, 22, 1), "int8", "uniform", 1, "heatbath", 0.4406868),         # int8 strip kernel (heat bath defers, Metropolis does not)
    ((128, 6, 6), "int8", "uniform", 2, "heatbath", 0.2216544),
    ((512, 22, 1), "int8", "uniform", 1, "metropolis", 0.4406868),
    ((256, 8, 4), "bitpack", "bond_pm1", 3, "metropolis", 0.9),          # own-stream +-J quad kernel
]


@pytest.mark.parametrize("cap", [0, 1, 5, 32])
@pytest.mark.parametrize("dims,storage,coupling,R,rule,beta", CASES)
def test_queue_capacity_does_not_change_results(P, oracle, dims, storage, coupling, R, rule, beta, cap):
    G = P.SpinSystem(dims, n=1, storage=storage, coupling=coupling, replicas=R, replica_streams=1, seed=SEED, rule=rule)
    G.set_option(P.OPT_DEFER_CAP, cap)
    kind = {"uniform": oracle.J_UNIFORM, "bond_pm1": oracle.J_BOND_PM1}[coupling]
    O = oracle.System(dims, n=1, coupling_kind=kind, n_replicas=R, replica_streams=1, seed=SEED,
                      rule=oracle.RULE_HEATBATH if rule == "heatbath" else oracle.RULE_METROPOLIS)
    for t in range(3):
        G.sweep(beta, 1)
        O.sweep(beta, 1)
        _equal(G, O, "cap %d sweep %d" % (cap, t))
    G.sweep(beta, 30)          # CUDA-graph replay: the captured argument block carries the capacity
    O.sweep(beta, 30)
    _equal(G, O, "cap %d after 33 sweeps" % cap)


def test_queue_capacity_changed_between_sweeps(P, oracle):
    """changing the capacity drops the captured graph; results stay the oracle's across the change"""
    dims, beta = (512, 16, 1), 0.4406868
    G = P.SpinSystem(dims, n=1, storage="bitpack", replicas=2, replica_streams=1, seed=SEED, rule="heatbath")
    O = oracle.System(dims, n=1, n_replicas=2, replica_streams=1, seed=SEED, rule=oracle.RULE_HEATBATH)
    for cap in (32, 2, 0, 7, 32):
        G.set_option(P.OPT_DEFER_CAP, cap)
        G.sweep(beta, 20)
        O.sweep(beta, 20)
        _equal(G, O, "cap %d" % cap)


def test_queue_capacity_range(P):
    G = P.SpinSystem((64, 4, 1), n=1, storage="bitpack", seed=SEED)
    for bad in (-1, 33):
        with pytest.raises(P.SpinError):
            G.set_option(P.OPT_DEFER_CAP, bad)
