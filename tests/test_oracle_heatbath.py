"""Pins of the oracle's heat-bath rule.

The heat-bath update draws the new spin from its conditional Boltzmann distribution in the local field, so the
same exact results that pin the Metropolis sweep pin it: exact enumeration of tiny lattices (P3, P4, P13), the
invariance of the Boltzmann distribution under each half-sweep operator (P5), Kaufman's finite-lattice energy (P7)
and the 1D-chain closed forms (P9) -- the n = 1 chain included, because heat bath has no deterministic dE = 0 flips.
"""
import numpy as np
import pytest

import exact_results as X
from test_oracle_physics import _mean_and_error, check_histogram

BETA_C2 = 0.4406868
BETA_C3 = 0.2216546


def _hist(oracle, dims, beta, n_chains, therm, seed, bonds=None):
    kw = dict(n=1, n_replicas=n_chains, replica_streams=1, seed=seed, rule=oracle.RULE_HEATBATH)
    if bonds is not None:
        kw.update(coupling_kind=oracle.J_BOND_PM1, bonds=np.broadcast_to(bonds, (n_chains,) + bonds.shape))
    S = oracle.System(dims, **kw)
    S.sweep(beta, therm)
    E, M = S.measure()
    return E, M[:, 0]


# --------------------------------------------------------------------------- the tabulated probabilities
@pytest.mark.parametrize("beta", [0.0, 0.1, BETA_C3, BETA_C2, 1.0 / 1.1, 3.0])
def test_heatbath_thresholds(oracle, beta):
    """T_hb(h) = floor(2^32 / (1 + exp(-2 beta h))) against 50-digit arithmetic; h = 0 is exactly one half."""
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 50
    assert oracle.heatbath_threshold(beta, 0) == 1 << 31
    for h in range(-6, 7):
        T = oracle.heatbath_threshold(beta, h)
        exact = mp.mpf(2) ** 32 / (1 + mp.exp(-2 * mp.mpf(beta) * h))
        assert abs(T - int(mp.floor(exact))) <= 1, (beta, h, T)   # last digit may depend on libm's exp
        assert 0 <= T <= 1 << 32
        # p(h) + p(-h) = 1 up to the two floors
        assert (1 << 32) - 1 <= T + oracle.heatbath_threshold(beta, -h) <= (1 << 32)
    assert oracle.heatbath_threshold(50.0, 4) == 1 << 32 and oracle.heatbath_threshold(50.0, -4) == 0


# --------------------------------------------------------------------------- P3 / P4 / P13: exact enumeration
def test_heatbath_4x4_histogram_matches_boltzmann_and_has_resolving_power(oracle):
    dims = (4, 4, 1)
    e, absm, m2, PE = X.boltzmann_moments(dims, BETA_C2)
    E, M = _hist(oracle, dims, BETA_C2, 40000, 60, seed=71)
    worst, chi2 = check_histogram(E, PE)
    assert worst < 3.0 and chi2 < 2.5, (worst, chi2)
    n = E.size
    assert abs(E.mean() / 16 - e) < 3 * E.std() / 16 / np.sqrt(n)
    assert abs(np.abs(M).mean() / 16 - absm) < 3 * np.abs(M).std() / 16 / np.sqrt(n)
    Ebad, _ = _hist(oracle, dims, 1.02 * BETA_C2, 40000, 60, seed=71)
    assert check_histogram(Ebad, PE)[0] > 5.0


@pytest.mark.parametrize("dims,beta", [((2, 2, 2), BETA_C3), ((4, 2, 2), BETA_C3)])
def test_heatbath_small_3d_histograms(oracle, dims, beta):
    PE = X.boltzmann_moments(dims, beta)[3]
    E, _ = _hist(oracle, dims, beta, 30000, 60, seed=5)
    worst, chi2 = check_histogram(E, PE)
    assert worst < 3.0 and chi2 < 2.5, (worst, chi2)


def test_heatbath_pmj_fixed_sample_histogram(oracle):
    dims = (4, 4, 1)
    rng = np.random.default_rng(3)
    bonds = rng.choice(np.array([-1, 1], dtype=np.int8), size=(2, 16))
    PE = X.boltzmann_moments(dims, 0.6, bonds=bonds)[3]
    E, _ = _hist(oracle, dims, 0.6, 30000, 80, seed=9, bonds=bonds)
    worst, chi2 = check_histogram(E, PE)
    assert worst < 3.0 and chi2 < 2.5, (worst, chi2)


# --------------------------------------------------------------------------- P5: stationarity of each half-sweep
@pytest.mark.parametrize("beta", [BETA_C2, 1.0])
def test_heatbath_half_sweep_operator_leaves_boltzmann_invariant(oracle, beta):
    dims, N = (4, 4, 1), 16
    st = X.all_states(N).astype(np.int64)
    E = X.lattice_energy(st, dims)
    w = np.exp(-beta * (E - E.min()).astype(np.float64))
    pi = w / w.sum()
    g = st.reshape(-1, 4, 4)
    h = (np.roll(g, 1, 1) + np.roll(g, -1, 1) + np.roll(g, 1, 2) + np.roll(g, -1, 2)).reshape(-1, N)
    p_up = {k: oracle.heatbath_threshold(beta, k) / 2.0 ** 32 for k in range(-4, 5, 2)}
    pu = np.vectorize(p_up.get)(h).astype(np.float64)
    # probability that site k ends up FLIPPED relative to the current state
    pflip = np.where(st > 0, 1.0 - pu, pu)
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
                    prob = prob * pflip[:, k]
                    flipmask |= 1 << k
                else:
                    prob = prob * (1.0 - pflip[:, k])
            np.add.at(out, idx ^ flipmask, prob)
        tol = 16 * 2.0 ** -32 / min(p_up.values())
        assert np.max(np.abs(out - pi) / pi) < tol, (colour, tol)


# --------------------------------------------------------------------------- P7, P9: exact energies
def _means(oracle, dims, beta, R, therm, sweeps, seed, **kw):
    S = oracle.System(dims, n_replicas=R, replica_streams=1, seed=seed, rule=oracle.RULE_HEATBATH, **kw)
    S.sweep(beta, therm)
    e_acc = np.zeros(R)
    for _ in range(sweeps):
        S.sweep(beta, 1)
        E, _ = S.measure()
        e_acc += E
    return e_acc / sweeps / S.N


def test_heatbath_2d_critical_energy_is_kaufmans(oracle):
    L = 16
    e = _means(oracle, (L, L, 1), BETA_C2, R=16, therm=400, sweeps=6000, seed=21)
    mean, err = _mean_and_error(e)
    exact = X.kaufman_energy_per_spin(L, BETA_C2)
    assert err < 3e-3
    assert abs(mean - exact) < 3 * err, (mean, err, exact)


@pytest.mark.parametrize("n,K", [(1, 0.5), (1, 1.0), (3, 1.0), (3, 2.0)])
def test_heatbath_reduction_to_independent_chains(oracle, n, K):
    """couplings (1, 0, 0): independent periodic chains of length 64: tanh-formula (n = 1), coth K - 1/K (n = 3)."""
    e = _means(oracle, (64, 16, 1), K, R=16, therm=300, sweeps=900, seed=100 + n, n=n,
               coupling_kind=oracle.J_PER_DIRECTION, J=(1.0, 0.0, 0.0))
    mean, err = _mean_and_error(-e)
    exact = X.chain_bond_average(n, K, 64)
    assert err < 3e-3
    assert abs(mean - exact) < 3 * err, (n, K, mean, err, exact)


# --------------------------------------------------------------------------- n = 3: the single-site law
def test_heatbath3_single_site_law(oracle):
    """|s'| = 1; s'.hhat has mean coth H - 1/H and second moment 1 - 2 (coth H - 1/H) / H; the part of s'
    perpendicular to h averages to zero (uniform azimuth); beta |h| = 0 falls back to the uniform direction."""
    rng = np.random.default_rng(17)
    beta, h = 0.7, np.array([1.5, -2.0, 0.75], dtype=np.float32)
    hn = float(np.linalg.norm(h.astype(np.float64)))
    hhat = h.astype(np.float64) / hn
    H = beta * hn
    n = 40000
    W = rng.integers(0, 1 << 32, size=(n, 2), dtype=np.uint64)
    S = np.array([oracle.heatbath3(beta, h, int(a), int(b)) for a, b in W], dtype=np.float64)
    assert np.max(np.abs(np.linalg.norm(S, axis=1) - 1.0)) < 1e-6
    c = S @ hhat
    L1 = 1.0 / np.tanh(H) - 1.0 / H
    assert abs(c.mean() - L1) < 3 * c.std() / np.sqrt(n)
    assert abs((c ** 2).mean() - (1.0 - 2.0 * L1 / H)) < 3 * (c ** 2).std() / np.sqrt(n)
    perp = S - np.outer(c, hhat)
    assert np.all(np.abs(perp.mean(axis=0)) < 3.5 * perp.std(axis=0) / np.sqrt(n))
    # negative z component of h exercises the other branch of the frame construction
    S2 = np.array([oracle.heatbath3(beta, -h, int(a), int(b)) for a, b in W[:2000]], dtype=np.float64)
    assert np.max(np.abs(np.linalg.norm(S2, axis=1) - 1.0)) < 1e-6
    assert abs((S2 @ -hhat).mean() - L1) < 4 * c.std() / np.sqrt(2000)
    for a, b in W[:20]:
        assert np.array_equal(oracle.heatbath3(0.0, h, int(a), int(b)), oracle.direction3(int(a), int(b)))
        assert np.array_equal(oracle.heatbath3(beta, np.zeros(3), int(a), int(b)), oracle.direction3(int(a), int(b)))


def test_heatbath_and_metropolis_agree_on_a_3d_heisenberg_lattice(oracle):
    """Two different Markov chains, one stationary distribution: <e> on 4^3 at beta = 0.693 within 3 sigma."""
    res = []
    for rule, seed in ((oracle.RULE_METROPOLIS, 1), (oracle.RULE_HEATBATH, 2)):
        S = oracle.System((4, 4, 4), n=3, n_replicas=24, replica_streams=1, seed=seed, rule=rule)
        S.sweep(0.693, 200)
        acc = np.zeros(24)
        for _ in range(700):
            S.sweep(0.693, 1)
            acc += S.measure()[0]
        res.append(_mean_and_error(acc / 700 / 64))
    (m1, e1), (m2, e2) = res
    assert abs(m1 - m2) < 3 * np.hypot(e1, e2), res


def test_heatbath_is_refused_for_xy(oracle):
    with pytest.raises(ValueError):
        oracle.System((4, 4, 1), n=2, rule=oracle.RULE_HEATBATH)
