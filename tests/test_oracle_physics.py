"""Statistical / exact-distribution pins of the oracle.

The Metropolis sweep is pinned by what its stationary distribution must be: exact
enumeration of tiny lattices, Kaufman's finite-lattice energy, Onsager/Yang, 1D-chain closed forms and the 3D
high-temperature series.  Seeds are fixed, so each 3-sigma statement is decided once.
"""
import numpy as np
import pytest

import exact_results as X

BETA_C2 = 0.4406868
BETA_C3 = 0.2216546
G = X.golden_values()


# --------------------------------------------------------------------------- helpers
def energy_histogram(oracle, dims, beta, n_chains, therm, n_samples, gap, seed, bonds=None):
    kw = dict(n=1, n_replicas=n_chains, replica_streams=1, seed=seed)
    if bonds is not None:
        kw.update(coupling_kind=oracle.J_BOND_PM1, bonds=np.broadcast_to(bonds, (n_chains,) + bonds.shape))
    S = oracle.System(dims, **kw)
    S.sweep(beta, therm)
    Es, Ms = [], []
    for k in range(n_samples):
        if k:
            S.sweep(beta, gap)
        E, M = S.measure()
        Es.append(E.copy())
        Ms.append(M[:, 0].copy())
    return np.concatenate(Es), np.concatenate(Ms)


def check_histogram(E, PE, min_p=3e-4, nsig=3.0):
    """every bin with P > min_p within nsig sigma of the multinomial expectation (rest pooled); returns chi2/dof."""
    n = E.size
    vals, counts = np.unique(E.astype(np.int64), return_counts=True)
    got = dict(zip(vals.tolist(), counts.tolist()))
    assert set(got) <= set(PE), "sampled an energy that does not exist"
    worst, chi2, dof = 0.0, 0.0, 0
    pooled_p, pooled_c = 0.0, 0
    for Ev, p in PE.items():
        c = got.get(Ev, 0)
        if p > min_p:
            sig = np.sqrt(n * p * (1 - p))
            zscore = (c - n * p) / sig
            worst = max(worst, abs(zscore))
            chi2 += zscore ** 2 * (1 - p)
            dof += 1
        else:
            pooled_p += p
            pooled_c += c
    if pooled_p > 0:
        sig = np.sqrt(n * pooled_p * (1 - pooled_p))
        worst = max(worst, abs(pooled_c - n * pooled_p) / max(sig, 1.0))
    return worst, chi2 / max(dof - 1, 1)


# --------------------------------------------------------------------------- P3 / P4: exact enumeration
def test_ising_4x4_energy_histogram_matches_boltzmann(oracle):
    dims = (4, 4, 1)
    e, absm, m2, PE = X.boltzmann_moments(dims, BETA_C2)
    E, M = energy_histogram(oracle, dims, BETA_C2, n_chains=40000, therm=60, n_samples=1, gap=0, seed=11075463)
    worst, chi2 = check_histogram(E, PE)
    assert worst < 3.0, worst
    assert chi2 < 2.5
    n = E.size
    assert abs(E.mean() / 16 - e) < 3 * E.std() / 16 / np.sqrt(n)
    assert abs(np.abs(M).mean() / 16 - absm) < 3 * np.abs(M).std() / 16 / np.sqrt(n)
    assert abs((M ** 2).mean() / 256 - m2) < 3 * (M ** 2).std() / 256 / np.sqrt(n)


def test_ising_4x4_histogram_test_has_resolving_power(oracle):
    """negative control: a chain run at 1.02 beta must FAIL the same test."""
    dims = (4, 4, 1)
    PE = X.boltzmann_moments(dims, BETA_C2)[3]
    E, _ = energy_histogram(oracle, dims, 1.02 * BETA_C2, n_chains=40000, therm=60, n_samples=1, gap=0, seed=11075463)
    worst, _ = check_histogram(E, PE)
    assert worst > 5.0


@pytest.mark.parametrize("dims,beta", [((2, 2, 2), BETA_C3), ((4, 2, 2), BETA_C3), ((4, 2, 2), 0.1)])
def test_ising_small_3d_histograms(oracle, dims, beta):
    e, absm, _, PE = X.boltzmann_moments(dims, beta)
    N = dims[0] * dims[1] * dims[2]
    E, M = energy_histogram(oracle, dims, beta, n_chains=30000, therm=50, n_samples=1, gap=0, seed=2024)
    worst, chi2 = check_histogram(E, PE)
    assert worst < 3.0, worst
    assert chi2 < 2.5
    assert abs(E.mean() / N - e) < 3 * E.std() / N / np.sqrt(E.size)
    assert abs(np.abs(M).mean() / N - absm) < 3 * np.abs(M).std() / N / np.sqrt(E.size)


@pytest.mark.parametrize("dims", [(4, 4, 1), (4, 2, 2)])
def test_pmj_fixed_sample_histogram(oracle, dims):
    """P13: a fixed +-J sample; stationary distribution by brute force over all 2^16 states."""
    N = dims[0] * dims[1] * dims[2]
    d = 2 if dims[2] == 1 else 3
    rng = np.random.default_rng(20110728)
    bonds = (1 - 2 * rng.integers(0, 2, (d, N))).astype(np.int8)
    beta = 0.7
    e, _, _, PE = X.boltzmann_moments(dims, beta, bonds)
    E, _ = energy_histogram(oracle, dims, beta, n_chains=30000, therm=80, n_samples=1, gap=0, seed=5, bonds=bonds)
    worst, chi2 = check_histogram(E, PE)
    assert worst < 3.0, worst
    assert chi2 < 2.5
    assert abs(E.mean() / N - e) < 3 * E.std() / N / np.sqrt(E.size)


# --------------------------------------------------------------------------- P5: stationarity of each half-sweep
@pytest.mark.parametrize("beta", [BETA_C2, 0.2, 1.0])
def test_half_sweep_operator_leaves_boltzmann_distribution_invariant(oracle, beta):
    """Build the colour-c half-sweep transition operator on the 4x4 lattice from the oracle's own thresholds
    (p = T / 2^32) and check sum_s pi(s) P_c(s -> s') = pi(s') for all 65536 s'."""
    dims = (4, 4, 1)
    N = 16
    st = X.all_states(N).astype(np.int64)           # (65536, 16); bit k of the index set <=> spin k = -1
    E = X.lattice_energy(st, dims)
    w = np.exp(-beta * (E - E.min()).astype(np.float64))
    pi = w / w.sum()
    g = st.reshape(-1, 4, 4)
    h = np.roll(g, 1, 1) + np.roll(g, -1, 1) + np.roll(g, 1, 2) + np.roll(g, -1, 2)
    dE = (2 * g * h).reshape(-1, N)
    p_table = {k: (1.0 if k <= 0 else oracle.threshold(beta, k) / 2.0 ** 32) for k in range(-8, 9, 4)}
    acc = np.vectorize(p_table.get)(dE).astype(np.float64)  # acceptance probability of every site in every state
    idx = np.arange(1 << N)
    xs, ys = np.arange(N) % 4, np.arange(N) // 4
    for colour in (0, 1):
        sites = [k for k in range(N) if (xs[k] + ys[k]) % 2 == colour]
        out = np.zeros(1 << N)
        for subset in range(1 << len(sites)):
            prob = pi.copy()
            flipmask = 0
            for b, k in enumerate(sites):
                if (subset >> b) & 1:
                    prob = prob * acc[:, k]
                    flipmask |= 1 << k
                else:
                    prob = prob * (1.0 - acc[:, k])
            np.add.at(out, idx ^ flipmask, prob)
        # exact up to the 2^-32 quantisation of the tabulated factors, relative to the smallest of them
        tol = 16 * 2.0 ** -32 / min(v for v in p_table.values() if v > 0)
        assert np.max(np.abs(out - pi) / pi) < tol, (colour, tol)


# --------------------------------------------------------------------------- P7 / P8: 2D Ising exact results
def _replica_means(oracle, dims, beta, R, therm, sweeps, seed, init=None, **kw):
    S = oracle.System(dims, n_replicas=R, replica_streams=1, seed=seed,
                      init=(oracle.INIT_HOT if init is None else init), **kw)
    S.sweep(beta, therm)
    e_acc = np.zeros(R)
    m_acc = np.zeros(R)
    for _ in range(sweeps):
        S.sweep(beta, 1)
        E, M = S.measure()
        e_acc += E
        m_acc += np.sqrt((M ** 2).sum(axis=1))
    return e_acc / sweeps / S.N, m_acc / sweeps / S.N


def _mean_and_error(x):
    return x.mean(), x.std(ddof=1) / np.sqrt(x.size)


def test_2d_ising_critical_energy_is_kaufmans_finite_lattice_value(oracle):
    """north_star's "-sqrt(2)" check, at the finite-L value it really takes."""
    L = 16
    exact = X.kaufman_energy_per_spin(L, BETA_C2)
    assert exact == pytest.approx(G["kaufman_e_L16_b0.4406868"], abs=2e-10)
    e, _ = _replica_means(oracle, (L, L, 1), BETA_C2, R=16, therm=400, sweeps=9000, seed=11075463)
    mean, err = _mean_and_error(e)
    assert err < 2.5e-3
    assert abs(mean - exact) < 3 * err, (mean, err, exact)
    assert abs(mean + np.sqrt(2.0)) > 5 * err  # the infinite-lattice value is NOT what a 16x16 torus gives
    # resolving power: 2 % off in beta is a many-sigma effect
    assert abs(X.kaufman_energy_per_spin(L, 1.02 * BETA_C2) - exact) > 10 * err


def test_2d_ising_critical_energy_kaufman_L32(oracle):
    """SURVEY.md P7 asks for L = 16 and 32: the same pin on the 32 x 32 torus (16 chains x 30 000 sweeps)."""
    L = 32
    exact = X.kaufman_energy_per_spin(L, BETA_C2)
    e, _ = _replica_means(oracle, (L, L, 1), BETA_C2, R=16, therm=1500, sweeps=30000, seed=1107)
    mean, err = _mean_and_error(e)
    assert err < 3.5e-3
    assert abs(mean - exact) < 3 * err, (mean, err, exact)
    assert abs(mean + np.sqrt(2.0)) > 4 * err
    assert abs(exact - X.kaufman_energy_per_spin(16, BETA_C2)) > 4 * err   # L = 32 is told apart from L = 16


def test_2d_ising_ordered_phase_matches_onsager_yang(oracle):
    """P8: beta = 0.5, cold start, L = 32: <|m|> = (1 - sinh^-4 2beta)^(1/8), <e> = Onsager."""
    L = 32
    e, m = _replica_means(oracle, (L, L, 1), 0.5, R=8, therm=200, sweeps=3500, seed=8, init=oracle.INIT_COLD)
    em, ee = _mean_and_error(e)
    mm, me = _mean_and_error(m)
    assert ee < 1.5e-3 and me < 1.5e-3
    assert abs(em - X.kaufman_energy_per_spin(L, 0.5)) < 3 * ee, (em, ee)
    assert abs(mm - X.yang_magnetisation(0.5)) < 3 * me + 2e-4, (mm, me)


# --------------------------------------------------------------------------- P9: 1D chains, all n
@pytest.mark.parametrize("n,K,R,sweeps", [(2, 1.0, 16, 1300), (3, 1.0, 16, 1300), (3, 2.0, 16, 1300)])
def test_reduction_to_independent_chains(oracle, n, K, R, sweeps):
    """couplings (1, 0, 0): Ly independent periodic chains of length 64; pins proposal, acceptance and E for n = 2, 3."""
    dims = (64, 16, 1)
    e, _ = _replica_means(oracle, dims, K, R=R, therm=300, sweeps=sweeps, seed=1234 + n,
                          n=n, coupling_kind=oracle.J_PER_DIRECTION, J=(1.0, 0.0, 0.0))
    mean, err = _mean_and_error(-e)
    exact = X.chain_bond_average(n, K, 64)
    assert err < 3e-3
    assert abs(mean - exact) < 3 * err, (n, K, mean, err, exact)


def test_ising_chain_conserves_its_domain_wall_charge(oracle):
    """n = 1 cannot use the 1D closed form: with dE = 0 always accepted (Eq. (2)) and the two colours
    updated in turn, a domain wall whose left site has colour 0 moves left two sites per sweep, one
    whose left site has colour 1 moves right, pairs are created and annihilated as one of each: the difference of the
    two counts is conserved in every chain, so the chain is not ergodic in 1D.  That conservation law is itself a
    sharp deterministic pin of the acceptance rule and the colour order (finding F-1)."""
    dims = (64, 16, 1)
    S = oracle.System(dims, n=1, coupling_kind=oracle.J_PER_DIRECTION, J=(1.0, 0.0, 0.0), seed=3)
    x, y = np.arange(64)[None, :], np.arange(16)[:, None]

    def charge(sp):
        g = sp.reshape(16, 64)
        wall = g != np.roll(g, -1, axis=1)
        left_colour = (x + y) % 2
        return (wall & (left_colour == 0)).sum(axis=1) - (wall & (left_colour == 1)).sum(axis=1)

    q0 = charge(S.get_spins()[0])
    assert np.abs(q0).max() > 0
    for _ in range(6):
        S.sweep(1.0, 5)
        assert np.array_equal(charge(S.get_spins()[0]), q0)


def test_3d_code_path_reduces_to_2d_layers(oracle):
    """P10: couplings (1, 1, 0) make an L x L x Lz lattice Lz independent tori, driven through the 3D neighbour code."""
    L = 8
    exact = X.kaufman_energy_per_spin(L, BETA_C2)
    e, _ = _replica_means(oracle, (L, L, 4), BETA_C2, R=8, therm=300, sweeps=5000, seed=77,
                          coupling_kind=oracle.J_PER_DIRECTION, J=(1.0, 1.0, 0.0))
    mean, err = _mean_and_error(e)
    assert abs(mean - exact) < 3 * err, (mean, err, exact)


# --------------------------------------------------------------------------- P11: genuinely 3D coupling
def test_3d_ising_high_temperature_series(oracle):
    K = 0.1
    minus_e, omitted = X.sc_ising_series_minus_e(K)
    e, _ = _replica_means(oracle, (8, 8, 8), K, R=8, therm=100, sweeps=7000, seed=3)
    mean, err = _mean_and_error(-e)
    assert err < 6e-4
    assert abs(mean - minus_e) < 3 * err + 2 * omitted, (mean, err, minus_e)


@pytest.mark.parametrize("n", [2, 3])
def test_3d_vector_models_high_temperature_series(oracle, n):
    """The genuinely three-dimensional n >= 2 path (all six neighbour terms of sweep_vector): 8^3 at
    K = 0.05 against -e = 3 t + 12 n t^3 t' (exact_results.sc_on_series_minus_e, derived from the definition).  A dropped
    or doubled y / z term in the local field moves -e by a third of its value, a missing lattice term by 0.25 %."""
    K = 0.05
    minus_e, omitted = X.sc_on_series_minus_e(n, K)
    e, _ = _replica_means(oracle, (8, 8, 8), K, R=16, therm=50, sweeps=1500, seed=40 + n, n=n)
    mean, err = _mean_and_error(-e)
    assert err < 6e-4
    assert abs(mean - minus_e) < 3 * err + 2 * omitted, (n, mean, err, minus_e)
    assert abs(2.0 / 3.0 * minus_e - mean) > 10 * err     # resolving power: one missing direction is a many-sigma effect


# --------------------------------------------------------------------------- P14: continuous spins
def test_direction_maps(oracle):
    rng = np.random.default_rng(7)
    for _ in range(200):
        a, b = (int(v) for v in rng.integers(0, 2 ** 32, 2))
        v = oracle.direction3(a, b).astype(np.float64)
        assert abs((v ** 2).sum() - 1.0) < 4e-7
        assert v[2] == 2.0 * ((a >> 8) / 2.0 ** 24) - 1.0
        phi = np.pi * 2.0 * ((b >> 8) / 2.0 ** 24)
        rho = np.sqrt(max(0.0, 1.0 - v[2] ** 2))
        assert abs(v[0] - rho * np.cos(phi)) < 2e-7 and abs(v[1] - rho * np.sin(phi)) < 2e-7
        w = oracle.direction2(a).astype(np.float64)
        th = np.pi * 2.0 * ((a >> 8) / 2.0 ** 24)
        assert abs(w[0] - np.cos(th)) < 1e-7 and abs(w[1] - np.sin(th)) < 1e-7
    # exact special angles
    assert oracle.direction2(0).tolist() == [1.0, 0.0]
    assert oracle.direction2(1 << 30).tolist() == [0.0, 1.0]
    assert oracle.direction2(1 << 31).tolist() == [-1.0, 0.0]
    assert oracle.direction3(1 << 31, 0).tolist() == [1.0, 0.0, 0.0]
    assert oracle.u24(0xFFFFFFFF) == 1.0 - 2.0 ** -24 and oracle.u24(0xFF) == 0.0


def test_vector_accept_rule(oracle):
    import mpmath as mp
    rng = np.random.default_rng(8)
    for _ in range(300):
        beta = float(rng.uniform(0.1, 3.0))
        dE = float(np.float32(rng.uniform(-2, 8)))
        w = int(rng.integers(0, 2 ** 32))
        u = (w >> 8) / 2.0 ** 24
        p = float(mp.exp(-mp.mpf(float(np.float32(beta))) * mp.mpf(dE)))
        want = 1 if (dE <= 0 or u < p) else 0
        if dE > 0 and abs(u - p) < 1e-6 * p:
            continue  # within fp32 rounding of the boundary
        assert oracle.vector_accept(beta, dE, w) == want


@pytest.mark.parametrize("n", [2, 3])
def test_beta_zero_gives_iid_uniform_directions(oracle, n):
    dims = (16, 16, 16)
    S = oracle.System(dims, n=n, init=oracle.INIT_COLD, seed=21)
    acc = S.sweep_count(0.0, 1)
    assert acc[0] == S.N                      # every proposal accepted
    s = S.get_spins()[0].astype(np.float64)
    N = S.N
    assert np.allclose((s ** 2).sum(axis=1), 1.0, atol=4e-7)
    for a in range(n):
        assert abs(s[:, a].mean()) < 4 * np.sqrt(1.0 / n / N)
        assert abs((s[:, a] ** 2).mean() - 1.0 / n) < 4 * np.sqrt((3.0 / (n * (n + 2)) - 1.0 / n ** 2) / N)
    assert abs((s[:, 0] * s[:, 1]).mean()) < 4 / n / np.sqrt(N)
    E, M = S.measure()
    assert abs(E[0]) < 4 * np.sqrt(3 * N / n)  # <E> = 0, Var E = d N / n
    # hot start is the same distribution
    H = oracle.System(dims, n=n, seed=22)
    sh = H.get_spins()[0].astype(np.float64)
    for a in range(n):
        assert abs(sh[:, a].mean()) < 4 * np.sqrt(1.0 / n / N)
        assert abs((sh[:, a] ** 2).mean() - 1.0 / n) < 4 * np.sqrt((3.0 / (n * (n + 2)) - 1.0 / n ** 2) / N)
