"""Deterministic pins of the oracle's sweep: an independent vectorised restatement of one sweep, limits (P6),
gauge invariance (P12), bookkeeping.  PAPER.md:31-38 (model, Eq. (2)), PAPER.md:42 (checkerboard order)."""
import numpy as np
import pytest

import exact_results as X

BETA_C = 0.4406868


def _coords(dims):
    Lx, Ly, Lz = dims
    i = np.arange(Lx * Ly * Lz)
    return i % Lx, (i // Lx) % Ly, i // (Lx * Ly)


def numpy_ising_sweep(oracle, spins, dims, beta, seed, t, rho=0, bonds=None):
    """One sweep written a second, different way: whole-colour array operations with np.roll instead of a site
    loop.  Uses only the oracle's per-site uniform and threshold (pinned separately)."""
    Lx, Ly, Lz = dims
    d = 2 if Lz == 1 else 3
    x, y, z = _coords(dims)
    j = (x >> 1) + (Lx // 2) * (y + Ly * z)
    s = spins.astype(np.int64).reshape(Lz, Ly, Lx).copy()
    Jf = [np.ones((Lz, Ly, Lx), dtype=np.int64) if bonds is None else bonds[mu].reshape(Lz, Ly, Lx).astype(np.int64)
          for mu in range(d)]
    T = {dE: oracle.threshold(beta, dE) for dE in range(2, 13, 2)}
    for colour in (0, 1):
        U = np.array([oracle.ising_uniform(seed, int(jj), rho, t, colour) for jj in j], dtype=np.uint64).reshape(Lz, Ly, Lx)
        h = np.zeros_like(s)
        for mu in range(d):
            ax = 2 - mu
            h += Jf[mu] * np.roll(s, -1, axis=ax)                      # +mu neighbour through our forward bond
            h += np.roll(Jf[mu], 1, axis=ax) * np.roll(s, 1, axis=ax)  # -mu neighbour through its forward bond
        dE = 2 * s * h
        thr = np.zeros_like(U)
        for k, v in T.items():
            thr[dE == k] = v
        flip = (dE <= 0) | (U < thr)
        mask = ((x + y + z) % 2 == colour).reshape(Lz, Ly, Lx)
        s = np.where(mask & flip, -s, s)
    return s.reshape(-1).astype(np.int8)


@pytest.mark.parametrize("dims", [(4, 4, 1), (8, 6, 1), (64, 4, 1), (66, 2, 1), (4, 2, 2), (6, 4, 8), (2, 2, 2)])
def test_ising_sweep_equals_vectorised_restatement(oracle, dims):
    seed = 11075463
    S = oracle.System(dims, n=1, seed=seed)
    ref = S.get_spins()[0].copy()
    for t in range(3):
        ref = numpy_ising_sweep(oracle, ref, dims, BETA_C, seed, t)
        S.sweep(BETA_C, 1)
        assert np.array_equal(S.get_spins()[0], ref), (dims, t)


def test_pmj_sweep_equals_vectorised_restatement_and_replica_streams(oracle):
    dims, seed, R = (6, 4, 4), 99, 3
    for streams in (0, 1):
        S = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, n_replicas=R, replica_streams=streams, seed=seed)
        bonds = S.get_bonds()
        assert set(np.unique(bonds)) == {-1, 1}
        ref = S.get_spins().copy()
        for t in range(2):
            S.sweep(0.9, 1)
            got = S.get_spins()
            for r in range(R):
                ref[r] = numpy_ising_sweep(oracle, ref[r], dims, 0.9, seed, t, rho=(r if streams else 0), bonds=bonds[r])
                assert np.array_equal(got[r], ref[r]), (streams, t, r)


def test_hot_start_and_bonds_follow_the_contract(oracle):
    seed = 4242
    dims = (8, 6, 4)
    N = 8 * 6 * 4
    S = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, n_replicas=2, seed=seed)
    sp, bo = S.get_spins(), S.get_bonds()
    for r in range(2):
        for i in range(N):
            w = oracle.rand(seed, i >> 7, r, 0, 16 * 1)
            assert sp[r, i] == (-1 if (w[(i >> 5) & 3] >> (i & 31)) & 1 else 1)
            w = oracle.rand(seed, i >> 5, r, 0, 16 * 2)
            for mu in range(3):
                assert bo[r, mu, i] == (-1 if (w[mu] >> (i & 31)) & 1 else 1)
    # roughly half the spins and bonds are -1
    big = oracle.System((64, 64, 1), n=1, coupling_kind=oracle.J_BOND_PM1, seed=seed)
    assert abs(big.get_spins().mean()) < 4 / 64
    assert abs(big.get_bonds().mean()) < 4 / 90


def test_beta_zero_flips_every_spin(oracle):
    """P6: dE <= 0 accepts, and T = 2^32 at beta = 0 accepts the rest: every spin flips once per sweep."""
    for dims in [(8, 8, 1), (4, 6, 8)]:
        S = oracle.System(dims, n=1, seed=5)
        s0 = S.get_spins().copy()
        E0, M0 = S.measure()
        acc = S.sweep_count(0.0, 1)
        assert acc[0] == S.N
        assert np.array_equal(S.get_spins(), -s0)
        E1, M1 = S.measure()
        assert E1[0] == E0[0] and M1[0, 0] == -M0[0, 0]


def test_cold_start_frozen_at_large_beta_and_ground_state_energy(oracle):
    for dims, d in [((8, 8, 1), 2), ((4, 6, 8), 3)]:
        S = oracle.System(dims, n=1, init=oracle.INIT_COLD, seed=5)
        E, M = S.measure()
        assert E[0] == -d * S.N and M[0, 0] == S.N
        assert S.sweep_count(50.0, 3).sum() == 0
        assert np.all(S.get_spins() == 1)


def test_zero_coupling_accepts_everything(oracle):
    S = oracle.System((8, 8, 1), n=1, coupling_kind=oracle.J_PER_DIRECTION, J=(0.0, 0.0, 0.0), seed=5)
    assert S.sweep_count(2.0, 2).tolist() == [64, 64]
    E, _ = S.measure()
    assert E[0] == 0


def test_antiferromagnet_is_the_staggered_ferromagnet(oracle):
    """J = -1 on a bipartite lattice: s_i -> (-1)^(x+y+z) s_i maps it onto J = +1 with identical dE and random numbers."""
    dims, seed = (8, 6, 4), 31
    F = oracle.System(dims, n=1, J=(1.0, 1.0, 1.0), seed=seed)
    A = oracle.System(dims, n=1, J=(-1.0, -1.0, -1.0), seed=seed)
    x, y, z = _coords(dims)
    stag = (1 - 2 * ((x + y + z) & 1)).astype(np.int8)
    A.set_spins(F.get_spins() * stag)
    for _ in range(4):
        F.sweep(0.3, 1)
        A.sweep(0.3, 1)
        assert np.array_equal(A.get_spins()[0] * stag, F.get_spins()[0])
    assert A.measure()[0][0] == F.measure()[0][0]


@pytest.mark.parametrize("dims", [(8, 8, 1), (6, 4, 4), (4, 2, 2)])
def test_mattis_gauge_invariance(oracle, dims):
    """P12: J_ij = sigma_i sigma_j with s = sigma s0 evolves as sigma x (ferromagnet from s0), bit for bit."""
    seed = 777
    rng = np.random.default_rng(1)
    Lx, Ly, Lz = dims
    d = 2 if Lz == 1 else 3
    N = Lx * Ly * Lz
    sigma = (1 - 2 * rng.integers(0, 2, N)).astype(np.int8)
    sg = sigma.reshape(Lz, Ly, Lx)
    bonds = np.stack([(sg * np.roll(sg, -1, axis=2 - mu)).reshape(-1) for mu in range(d)]).astype(np.int8)
    F = oracle.System(dims, n=1, seed=seed)
    G = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, bonds=bonds[None], seed=seed)
    G.set_spins(F.get_spins() * sigma)
    assert G.measure()[0][0] == F.measure()[0][0]
    for _ in range(5):
        F.sweep(0.35, 1)
        G.sweep(0.35, 1)
        assert np.array_equal(G.get_spins()[0] * sigma, F.get_spins()[0])
        assert G.measure()[0][0] == F.measure()[0][0]


def test_measure_matches_numpy_energy(oracle):
    for dims in [(8, 6, 1), (6, 4, 4), (2, 2, 2), (4, 2, 2)]:
        S = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, seed=3)
        sp, bo = S.get_spins()[0], S.get_bonds()[0]
        E, M = S.measure()
        assert E[0] == X.lattice_energy(sp, dims, bo)
        assert M[0, 0] == sp.astype(np.int64).sum()
        S2 = oracle.System(dims, n=1, seed=3)
        assert S2.measure()[0][0] == X.lattice_energy(S2.get_spins()[0], dims)


def test_sweep_counter_composition_and_resume(oracle):
    """sweep(a); sweep(b) == sweep(a + b); state + counter resumes bit-exactly (no generator state)."""
    dims = (8, 8, 1)
    A = oracle.System(dims, seed=9)
    B = oracle.System(dims, seed=9)
    A.sweep(BETA_C, 7)
    B.sweep(BETA_C, 3)
    B.sweep(BETA_C, 4)
    assert A.sweep_counter == B.sweep_counter == 7
    assert np.array_equal(A.get_spins(), B.get_spins())
    C_ = oracle.System(dims, seed=9, init=oracle.INIT_COLD)
    C_.set_spins(A.get_spins())
    C_.sweep_counter = 7
    A.sweep(BETA_C, 5)
    C_.sweep(BETA_C, 5)
    assert np.array_equal(A.get_spins(), C_.get_spins())


def test_energy_change_equals_sum_of_accepted_dE_vector_models(oracle):
    """P14 (bookkeeping part): over one sweep the energy of Eq. (1), re-measured from the spins, changes
    by exactly the sum of the dE of the accepted moves as the sweep computed them from its local field (fp32 there, so
    equal up to rounding).  A wrong neighbour, sign or coupling in any of the six field terms breaks the balance."""
    for n in (2, 3):
        S = oracle.System((8, 6, 4), n=n, seed=12)
        s = S.get_spins()[0].astype(np.float64)
        assert np.allclose((s ** 2).sum(axis=1), 1.0, atol=4e-7)
        for beta in (0.7, 0.7, 2.5, 0.0):
            E0, _ = S.measure()
            acc = S.sweep_count(beta, 1)
            E1, M = S.measure()
            assert 0 < acc[0] <= S.N
            dE = S.last_sweep_dE()
            assert abs((E1[0] - E0[0]) - dE) <= 1e-6 * S.N, (n, beta, E1[0] - E0[0], dE)
            assert abs(E1[0] - E0[0]) > 1e-3        # the balance is not 0 = 0
        s = S.get_spins()[0].astype(np.float64)
        assert np.allclose((s ** 2).sum(axis=1), 1.0, atol=4e-7)
        g = s.reshape(4, 6, 8, n)
        e = -sum((g * np.roll(g, -1, axis=2 - mu)).sum() for mu in range(3))
        assert E1[0] == pytest.approx(e, rel=1e-12)
        assert np.allclose(M[0], s.sum(axis=0), rtol=1e-12)


def test_energy_change_equals_sum_of_accepted_dE_ising(oracle):
    """The same balance for n = 1, exact in integers: uniform, per-direction and +-J couplings, 2D and 3D."""
    cases = [dict(dims=(8, 6, 4)), dict(dims=(8, 6, 1)), dict(dims=(6, 4, 2), coupling_kind=oracle.J_PER_DIRECTION, J=(1.0, -1.0, 0.0)),
             dict(dims=(8, 6, 4), coupling_kind=oracle.J_BOND_PM1, n_replicas=2)]
    for kw in cases:
        S = oracle.System(kw.pop("dims"), n=1, seed=5, **kw)
        for beta in (0.3, 0.3, 1.0, 0.0):
            E0, _ = S.measure()
            S.sweep(beta, 1)
            E1, _ = S.measure()
            assert (E1 - E0).sum() == S.last_sweep_dE()


def test_invalid_arguments_are_rejected(oracle):
    for dims in [(3, 4, 1), (4, 5, 1), (4, 4, 3), (0, 4, 1)]:
        with pytest.raises(ValueError):
            oracle.System(dims)
    with pytest.raises(ValueError):
        oracle.System((4, 4, 1), n=4)
    with pytest.raises(ValueError):
        oracle.System((4, 4, 1), n=1, J=(0.5, 0.5, 0.5))
    with pytest.raises(ValueError):
        oracle.System((4, 4, 1), n_replicas=0)
