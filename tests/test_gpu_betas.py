"""Temperature axis (spin_sweep_betas): replica r swept at betas[r] must follow exactly the
chain it follows in a handle (or an oracle system) swept at betas[r] throughout -- bit-exact against the oracle for n = 1
in every kernel family that offers it, bitwise against the single-beta handle for n = 2, 3."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SEED = 424242


@pytest.fixture(scope="module")
def P():
    import paper_1107_5463_b200 as pkg
    pkg.lib()
    return pkg


@pytest.mark.parametrize("dims,storage,coupling,rule", [
    ((128, 12, 1), "int8", "uniform", "metropolis"),        # int8 strip kernel
    ((128, 10, 4), "bitpack", "uniform", "heatbath"),       # bit-packed strip kernel, 3D
    ((10, 8, 1), "int8", "uniform", "metropolis"),          # generic kernel
    ((12, 6, 4), "int8", "bond_pm1", "metropolis"),         # generic kernel, per-bond couplings: spin-glass tempering
    ((64, 64, 1), "int8", "uniform", "metropolis"),         # resident-kernel territory: plain launches here
])
def test_temperature_axis_ising_against_the_oracle(P, dims, storage, coupling, rule):
    import oracle

    R, betas = 4, [0.0, 0.3, 0.4406868, 0.9]
    G = P.SpinSystem(dims, n=1, storage=storage, coupling=coupling, replicas=R, replica_streams=1, seed=SEED, rule=rule)
    kind = oracle.J_BOND_PM1 if coupling == "bond_pm1" else oracle.J_UNIFORM
    orule = oracle.RULE_HEATBATH if rule == "heatbath" else oracle.RULE_METROPOLIS
    Os = [oracle.System(dims, n=1, coupling_kind=kind, n_replicas=R, replica_streams=1, seed=SEED, rule=orule) for _ in range(R)]
    for n in (1, 3, 2):
        G.sweep_betas(betas, n)
        g = G.get_spins()
        Eg, Mg = G.measure()
        for r in range(R):
            Os[r].sweep(betas[r], n)
            assert np.array_equal(g[r], Os[r].get_spins()[r]), (n, r)
            Eo, Mo = Os[r].measure()
            assert Eg[r] == Eo[r] and Mg[r, 0] == Mo[r, 0]
    assert G.sweep_counter == 6
    G.sweep(betas[1], 2)                 # back to one beta for all: replica 1 simply continues its chain
    Os[1].sweep(betas[1], 2)
    assert np.array_equal(G.get_spins()[1], Os[1].get_spins()[1])


@pytest.mark.parametrize("n,dims", [(3, (16, 8, 8)), (2, (16, 12, 1)), (3, (6, 6, 4))])
def test_temperature_axis_vector_models_bitwise(P, n, dims):
    R, betas = 3, [0.2, 0.693, 1.5]
    kw = dict(n=n, storage="fp32", replicas=R, replica_streams=1, seed=SEED)
    G = P.SpinSystem(dims, **kw)
    G.sweep_betas(betas, 6)
    g = G.get_spins().view(np.uint32)
    for r in range(R):
        H = P.SpinSystem(dims, **kw)
        H.sweep(betas[r], 6)
        assert np.array_equal(g[r], H.get_spins().view(np.uint32)[r]), r


def test_temperature_axis_argument_checks(P):
    S = P.SpinSystem((128, 8, 1), n=1, storage="bitpack", coupling="bond_pm1", replicas=2, replica_streams=1, seed=1)
    with pytest.raises(P.SpinError):
        S.sweep_betas([0.1, 0.2], 1)                       # bit-packed per-bond couplings: not offered
    T = P.SpinSystem((128, 8, 1), n=1, storage="int8", replicas=2, replica_streams=0, seed=1)
    with pytest.raises(P.SpinError):
        T.sweep_betas([0.1, 0.2], 1)                       # shared update stream
    U = P.SpinSystem((128, 8, 1), n=1, storage="int8", replicas=2, replica_streams=1, seed=1)
    with pytest.raises(P.SpinError):
        U.sweep_betas([0.1, -0.2], 1)
    with pytest.raises(ValueError):
        U.sweep_betas([0.1], 1)
