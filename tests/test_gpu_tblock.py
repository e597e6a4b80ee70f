"""Exact temporal blocking ("k updates per tile load", made results-neutral): spin_sweep with
SPIN_OPT_TEMPORAL_BLOCKING runs two sweeps per pass over the lattice and must leave EXACTLY the spins of plain sweeps.
Bit-exact against the oracle after every pair of sweeps and after odd counts (the odd sweep goes through the plain
kernel), for ragged and wrapping stripes, several replicas, the antiferromagnet, beta = 0 and a large beta."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SEED = 11075463
BETA_C = 0.4406868


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
    gs, os_ = G.get_spins(), O.get_spins()
    bad = int(np.count_nonzero(gs != os_))
    assert bad == 0, "%s: %d spins differ" % (tag, bad)
    Eg, Mg = G.measure()
    Eo, Mo = O.measure()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo), (tag, Eg, Eo)


@pytest.mark.parametrize("dims,rows,R,beta", [((2048, 40, 1), 0, 1, BETA_C), ((2048, 26, 1), 5, 2, 0.3), ((4096, 12, 1), 3, 1, 0.0)])
def test_temporal_blocking_heat_bath(P, oracle, dims, rows, R, beta):
    """the same kernel with the heat-bath rule: bit-exact against the oracle after pairs and odd counts"""
    G = P.SpinSystem(dims, n=1, storage="int8", replicas=R, replica_streams=1, seed=SEED, rule="heatbath")
    G.set_option(P.OPT_TEMPORAL_BLOCKING, 1)
    G.set_option(P.OPT_TBLOCK_ROWS, rows)
    O = oracle.System(dims, n=1, n_replicas=R, replica_streams=1, seed=SEED, rule=oracle.RULE_HEATBATH)
    for n in (2, 3, 4):
        l0 = G.launch_count
        G.sweep(beta, n)
        assert G.launch_count - l0 == n // 2 + 2 * (n % 2)
        O.sweep(beta, n)
        _equal(G, O, "after %d sweeps" % n)


@pytest.mark.parametrize("dims,storage,rows,J,R,beta", [
    ((2048, 40, 1), "int8", 0, 1.0, 1, BETA_C),       # automatic stripe height
    ((2048, 38, 1), "int8", 7, 1.0, 1, BETA_C),       # ragged last stripe
    ((2048, 38, 1), "int8", 5, -1.0, 2, BETA_C),   # antiferromagnet, two replicas with their own streams
    ((2048, 6, 1), "int8", 2, 1.0, 1, BETA_C),        # halo wraps around the whole lattice
    ((2048, 2, 1), "int8", 1, 1.0, 1, BETA_C),     # two rows: every neighbour row is the other row
    ((4096, 24, 1), "int8", 9, 1.0, 3, 0.3),          # two warps per row
    ((2048, 30, 1), "int8", 30, 1.0, 1, 0.0),         # beta = 0: every spin flips twice per pair
    ((2048, 30, 1), "int8", 11, 1.0, 1, 50.0),     # frozen
    ((16384, 12, 1), "int8", 4, 1.0, 1, BETA_C),      # BASELINE row width (256 threads per CTA)
    ((32768, 10, 1), "int8", 3, 1.0, 1, BETA_C),   # 512 threads per CTA
])
def test_temporal_blocking_is_bit_exact(P, oracle, dims, storage, rows, J, R, beta):
    kw = dict(n=1, storage=storage, J=(J, J, J), replicas=R, replica_streams=1, seed=SEED)
    G = P.SpinSystem(dims, **kw)
    G.set_option(P.OPT_TEMPORAL_BLOCKING, 1)
    G.set_option(P.OPT_TBLOCK_ROWS, rows)
    O = oracle.System(dims, n=1, J=(J, J, J), n_replicas=R, replica_streams=1, seed=SEED)
    l0 = G.launch_count
    G.sweep(beta, 2)
    assert G.launch_count - l0 == 1, "one launch for two sweeps"
    O.sweep(beta, 2)
    _equal(G, O, "after one pair")
    for k, n in enumerate((4, 3, 1, 5)):             # pairs, odd counts (plain kernel for the last sweep), a single sweep
        G.sweep(beta, n)
        O.sweep(beta, n)
        _equal(G, O, "after %d more sweeps (call %d)" % (n, k))
    assert G.sweep_counter == 15


def test_temporal_blocking_equals_plain_sweeps_and_checkpoint(P):
    """The same chain with and without temporal blocking (bitwise), continued from a get_spins / set_spins checkpoint."""
    dims = (2048, 64, 1)
    kw = dict(n=1, storage="int8", seed=7)
    A, B = P.SpinSystem(dims, **kw), P.SpinSystem(dims, **kw)
    A.set_option(P.OPT_TEMPORAL_BLOCKING, 1)
    B.set_option(P.OPT_TEMPORAL_BLOCKING, 0)
    A.sweep(BETA_C, 7)
    B.sweep(BETA_C, 7)
    assert np.array_equal(A.get_spins(), B.get_spins())
    C = P.SpinSystem(dims, **kw)
    C.set_option(P.OPT_TEMPORAL_BLOCKING, 1)
    C.set_spins(A.get_spins())
    C.sweep_counter = A.sweep_counter
    A.sweep(BETA_C, 6)
    C.sweep(BETA_C, 6)
    B.sweep(BETA_C, 6)
    assert np.array_equal(A.get_spins(), C.get_spins()) and np.array_equal(A.get_spins(), B.get_spins())
    dE, dM = A.sweep_record(BETA_C, 3)               # recorded sweeps use the plain kernels on the swapped arrays
    B.sweep(BETA_C, 3)
    E, M = B.measure()
    assert dE[-1, 0].item() == E[0] and dM[-1, 0, 0].item() == M[0, 0]


def test_temporal_blocking_not_offered(P):
    """Shapes outside the offer run the plain kernels whatever the option says (results are the contract, not the kernel)."""
    G = P.SpinSystem((1024, 16, 1), n=1, storage="int8", seed=3)
    G.set_option(P.OPT_TEMPORAL_BLOCKING, 1)
    l0 = G.launch_count
    G.sweep(BETA_C, 2)
    assert G.launch_count - l0 >= 1
    H = P.SpinSystem((1024, 16, 1), n=1, storage="int8", seed=3)
    H.set_option(P.OPT_PLAIN_KERNELS, 1)
    H.sweep(BETA_C, 2)
    assert np.array_equal(G.get_spins(), H.get_spins())


@pytest.mark.parametrize("storage", ["int8"])
def test_full_size_pairs_equal_plain_sweeps(P, storage):
    """BASELINE config 2 at full size, default knobs: five sweeps with temporal blocking (two passes + one plain sweep)
    leave exactly the bytes of five plain sweeps."""
    w = P.workloads.WORKLOADS["ising2d_L16384_" + storage]
    A, B = P.from_workload(w, P.workloads.SEED), P.from_workload(w, P.workloads.SEED)
    B.set_option(P.OPT_TEMPORAL_BLOCKING, 0)
    l0 = A.launch_count
    A.sweep(w["beta"], 5)
    B.sweep(w["beta"], 5)
    assert A.launch_count - l0 == 2 + 2, "two passes of two sweeps and the two half-sweeps of the odd one"
    assert np.array_equal(A.get_spins(), B.get_spins())
