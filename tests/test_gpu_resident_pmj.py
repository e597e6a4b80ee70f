"""Many +-J realisations of a small lattice with a shared update stream (Table 1's many-realisation
workload; R-17): spin_sweep keeps groups of realisations in shared memory for all sweeps of the call
(ising_resident_pmj_kernel.cuh).  Bit-exact against the oracle after every call -- single sweeps, odd counts, counts that
are not a multiple of the masks-ahead round, replica counts that do not fill the last group -- and against the
one-launch-per-half-sweep kernels (SPIN_OPT_KERNEL_VARIANT = 1) at sizes the oracle does not reach in seconds."""
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
    gs, os_ = G.get_spins(), O.get_spins()
    bad = int(np.count_nonzero(gs != os_))
    assert bad == 0, "%s: %d spins differ" % (tag, bad)
    Eg, Mg = G.measure()
    Eo, Mo = O.measure()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo), (tag, Eg[:4], Eo[:4], Mg[:4], Mo[:4])


@pytest.mark.parametrize("rule", ["metropolis", "heatbath"])
@pytest.mark.parametrize("dims,R,beta", [
    ((64, 64, 1), 19, 1.0),          # the bench lattice: 64 words per colour, 8 threads per word position
    ((64, 2, 1), 5, 0.4406868),      # 2 words per colour: a round builds the masks of 256 half-sweeps
    ((64, 16, 1), 300, 0.9),         # more replicas than one group
    ((128, 32, 1), 7, 1.1),          # 128 words per colour, two-word rows
    ((64, 4, 4), 40, 1.0 / 1.1),     # 3D, three thresholds
    ((64, 16, 16), 3, 0.5),          # 256 words per colour: two threads per word position
    ((64, 32, 16), 5, 0.8),          # 512 words per colour: one thread per word position, no masks ahead
    ((64, 8, 2), 33, 0.0),           # a size-2 dimension; beta = 0
    ((64, 8, 1), 2, 50.0),           # frozen
])
def test_resident_pmj_bit_exact_against_the_oracle(P, oracle, dims, R, beta, rule):
    G = P.SpinSystem(dims, n=1, storage="bitpack", coupling="bond_pm1", replicas=R, replica_streams=0, seed=SEED, rule=rule)
    O = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, n_replicas=R, replica_streams=0, seed=SEED,
                      rule=oracle.RULE_HEATBATH if rule == "heatbath" else oracle.RULE_METROPOLIS)
    assert np.array_equal(G.get_bonds(), O.get_bonds())
    _equal(G, O, "hot start")
    done = 0
    for ns in (1, 1, 2, 3, 5, 12):
        l0 = G.launch_count
        G.sweep(beta, ns)
        assert G.launch_count - l0 == 1, "all sweeps of the call in one launch"
        O.sweep(beta, ns)
        done += ns
        assert G.sweep_counter == done
        _equal(G, O, "%s R=%d after %d sweeps" % (dims, R, done))
    G.close()


@pytest.mark.parametrize("rule", ["metropolis", "heatbath"])
@pytest.mark.parametrize("dims,R,sweeps", [((64, 64, 1), 4096, 37), ((64, 64, 1), 1000, 130), ((64, 16, 8), 777, 21)])
def test_resident_pmj_agrees_with_the_per_half_sweep_kernels(P, dims, R, sweeps, rule):
    A = P.SpinSystem(dims, n=1, storage="bitpack", coupling="bond_pm1", replicas=R, replica_streams=0, seed=SEED, rule=rule)
    B = P.SpinSystem(dims, n=1, storage="bitpack", coupling="bond_pm1", replicas=R, replica_streams=0, seed=SEED, rule=rule)
    B.set_option(P.OPT_KERNEL_VARIANT, 1)
    la, lb = A.launch_count, B.launch_count
    A.sweep(1.0, sweeps)
    B.sweep(1.0, sweeps)
    assert A.launch_count - la == 1 and B.launch_count - lb >= 2, "two different paths"
    assert np.array_equal(A.get_spins(), B.get_spins())
    # recorded sweeps (fused E / M) stay on the per-half-sweep kernels and continue the same chain
    Ea, Ma = A.sweep_record(1.0, 3)
    Eb, Mb = B.sweep_record(1.0, 3)
    assert np.array_equal(Ea.cpu().numpy(), Eb.cpu().numpy()) and np.array_equal(Ma.cpu().numpy(), Mb.cpu().numpy())
    assert np.array_equal(A.get_spins(), B.get_spins())
    A.close()
    B.close()
