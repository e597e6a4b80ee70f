"""Replica-per-bit multi-spin coding (SPIN_STORE_MSC; Table 1 row "2D spin glass, Metro. multi-spin" at
PAPER.md:88): 32 disorder realisations of one site per word, one random number per site for all of them.
Bit-exact against the oracle (+-J bonds per realisation, shared update stream) after every sweep, on the paper's own
L = 32 lattice and on shapes the site-packed layout refuses; both update rules; E and M per realisation; canonical
get / set / bonds round trips; and agreement with the site-packed kernels where both are offered."""
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


@pytest.mark.parametrize("dims,R,beta,rule", [
    ((32, 32, 1), 64, 1.0, "metropolis"),        # the paper's lattice
    ((32, 32, 1), 96, 0.4406868, "heatbath"),
    ((16, 8, 1), 32, 0.7, "metropolis"),         # one unit per colour
    ((8, 8, 8), 64, 1.0 / 1.1, "metropolis"),    # 3D
    ((8, 4, 4), 32, 0.5, "heatbath"),
    ((16, 4, 2), 32, 0.9, "metropolis"),         # a size-2 dimension: both bonds to the same neighbour count
    ((64, 16, 1), 160, 0.0, "metropolis"),       # beta = 0
    ((64, 16, 1), 32, 50.0, "metropolis"),       # frozen
])
def test_msc_bit_exact_against_the_oracle(P, oracle, dims, R, beta, rule):
    G = P.SpinSystem(dims, n=1, storage="msc", coupling="bond_pm1", replicas=R, replica_streams=0, seed=SEED, rule=rule)
    O = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, n_replicas=R, replica_streams=0, seed=SEED,
                      rule=oracle.RULE_HEATBATH if rule == "heatbath" else oracle.RULE_METROPOLIS)
    assert np.array_equal(G.get_bonds(), O.get_bonds()), "bonds drawn from the seed"
    _equal(G, O, "hot start")
    for t in range(8):
        G.sweep(beta, 1)
        O.sweep(beta, 1)
        _equal(G, O, "sweep %d" % t)
    G.sweep(beta, 40)      # CUDA-graph replay territory (32 sweeps) + plain sweeps
    O.sweep(beta, 40)
    _equal(G, O, "after 48 sweeps")


def test_msc_user_bonds_set_spins_and_site_packed_agreement(P, oracle):
    """User-supplied bonds and spins through the canonical layouts; the same system in the site-packed layout
    (SPIN_STORE_BITPACK, shared update stream) follows the same trajectory bit for bit; recorded sweeps."""
    dims, R, beta = (64, 32, 1), 64, 0.8
    rng = np.random.default_rng(5)
    N = dims[0] * dims[1]
    bonds = rng.choice(np.array([-1, 1], dtype=np.int8), size=(R, 2, N))
    spins = rng.choice(np.array([-1, 1], dtype=np.int8), size=(R, N))
    A = P.SpinSystem(dims, n=1, storage="msc", coupling="bond_pm1", bonds=bonds, replicas=R, seed=3)
    B = P.SpinSystem(dims, n=1, storage="bitpack", coupling="bond_pm1", bonds=bonds, replicas=R, seed=3)
    O = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, bonds=bonds, n_replicas=R, seed=3)
    assert np.array_equal(A.get_bonds(), bonds)
    for S in (A, B, O):
        S.set_spins(spins)
    assert np.array_equal(A.get_spins(), spins)
    dE, dM = A.sweep_record(beta, 5)
    B.sweep(beta, 5)
    O.sweep(beta, 5)
    assert np.array_equal(A.get_spins(), B.get_spins()) and np.array_equal(A.get_spins(), O.get_spins())
    Eo, Mo = O.measure()
    assert np.array_equal(dE[-1].cpu().numpy(), Eo) and np.array_equal(dM[-1, :, 0].cpu().numpy(), Mo[:, 0])


def test_msc_argument_checks(P):
    bad = [dict(replicas=48), dict(replica_streams=1), dict(coupling="uniform"), dict(dims=(6, 6, 1))]
    for kw in bad:
        args = dict(dims=(32, 32, 1), n=1, storage="msc", coupling="bond_pm1", replicas=32, replica_streams=0, seed=1)
        args.update(kw)
        with pytest.raises(P.SpinError):
            P.SpinSystem(**args)
