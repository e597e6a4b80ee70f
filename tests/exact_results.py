"""Closed forms and brute-force enumerations the oracle is pinned against.

Nothing here touches oracle/ or the CUDA path: these are the textbook results
SURVEY.md section 8(c) names (pins P3, P4, P7, P8, P9, P11), written from their
definitions.  PAPER.md:76 uses the same idea (exact 2D Ising results as ground
truth); PAPER.md:31-35 defines the Hamiltonian they refer to.
"""
import itertools
import os

import mpmath as mp
import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden_values():
    out = {}
    with open(os.path.join(GOLDEN, "exact_values.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split()
            out[k] = float(v)
    return out


# ----------------------------------------------------------------- enumeration
def all_states(N):
    """(2^N, N) int8 array of +-1; bit k of the state index set <=> spin k = -1."""
    idx = np.arange(1 << N, dtype=np.int64)
    bits = (idx[:, None] >> np.arange(N)[None, :]) & 1
    return (1 - 2 * bits).astype(np.int8)


def lattice_energy(spins, dims, bonds=None):
    """H = -sum_<ij> J_ij s_i s_j for an array (..., N) of +-1 spins on a
    periodic lattice dims = (Lx, Ly, Lz); every site owns its +x, +y, +z bond, so a
    direction of size 2 contributes its bond twice.  bonds: (d, N) of +-1 or None (J = 1)."""
    Lx, Ly, Lz = dims
    d = 2 if Lz == 1 else 3
    s = spins.reshape(spins.shape[:-1] + (Lz, Ly, Lx)).astype(np.int64)
    E = np.zeros(spins.shape[:-1], dtype=np.int64)
    for mu in range(d):
        axis = s.ndim - 1 - mu
        sp = np.roll(s, -1, axis=axis)
        prod = s * sp
        if bonds is not None:
            prod = prod * bonds[mu].reshape(Lz, Ly, Lx).astype(np.int64)
        E -= prod.reshape(spins.shape[:-1] + (-1,)).sum(axis=-1)
    return E


def density_of_states(dims):
    N = dims[0] * dims[1] * dims[2]
    E = lattice_energy(all_states(N), dims)
    vals, counts = np.unique(E, return_counts=True)
    return dict(zip(vals.tolist(), counts.tolist()))


def boltzmann_moments(dims, beta, bonds=None):
    """exact <e>, <|m|>, <m^2> and P(E) by enumeration."""
    N = dims[0] * dims[1] * dims[2]
    st = all_states(N)
    E = lattice_energy(st, dims, bonds)
    M = st.astype(np.int64).sum(axis=1)
    w = np.exp(-beta * (E - E.min()).astype(np.float64))
    Z = w.sum()
    p = w / Z
    e = float((p * E).sum() / N)
    absm = float((p * np.abs(M)).sum() / N)
    m2 = float((p * M.astype(np.float64) ** 2).sum() / N ** 2)
    vals = np.unique(E)
    PE = {int(v): float(p[E == v].sum()) for v in vals}
    return e, absm, m2, PE


# ----------------------------------------------------------------- 2D Ising exact
def kaufman_lnZ(L, beta, M=None):
    """ln Z of the L x M periodic square-lattice Ising model, J = 1 (Kaufman 1949)."""
    M = L if M is None else M
    K = mp.mpf(beta)
    n, m = L, M  # n columns enter the gammas, m is the other length

    def gamma(l):
        if l == 0:
            return 2 * K + mp.log(mp.tanh(K))
        c = mp.cosh(2 * K) * mp.coth(2 * K) - mp.cos(mp.pi * l / n)
        return mp.acosh(c)

    p1 = mp.mpf(1)
    p2 = mp.mpf(1)
    p3 = mp.mpf(1)
    p4 = mp.mpf(1)
    for r in range(n):
        g_odd = gamma(2 * r + 1)
        g_even = gamma(2 * r)
        p1 *= 2 * mp.cosh(m * g_odd / 2)
        p2 *= 2 * mp.sinh(m * g_odd / 2)
        p3 *= 2 * mp.cosh(m * g_even / 2)
        p4 *= 2 * mp.sinh(m * g_even / 2)
    Z = mp.mpf(1) / 2 * (2 * mp.sinh(2 * K)) ** (mp.mpf(n * m) / 2) * (p1 + p2 + p3 + p4)
    return mp.log(Z)


def kaufman_energy_per_spin(L, beta):
    mp.mp.dps = 50
    f = lambda b: kaufman_lnZ(L, b)
    return float(-mp.diff(f, mp.mpf(beta)) / (L * L))


def onsager_energy_per_spin(beta):
    """infinite-lattice internal energy per spin (Onsager 1944)."""
    mp.mp.dps = 40
    K = mp.mpf(beta)
    k = 2 * mp.sinh(2 * K) / mp.cosh(2 * K) ** 2
    kp = 2 * mp.tanh(2 * K) ** 2 - 1
    K1 = mp.ellipk(k ** 2)
    return float(-mp.coth(2 * K) * (1 + 2 / mp.pi * kp * K1))


def yang_magnetisation(beta):
    """spontaneous magnetisation (Onsager/Yang), beta > beta_c."""
    return float((1 - mp.sinh(2 * mp.mpf(beta)) ** -4) ** (mp.mpf(1) / 8))


# ----------------------------------------------------------------- 1D chains
def chain_bond_average(n, K, L):
    """<s_i . s_{i+1}> of a periodic O(n) chain of length L at coupling K = beta J."""
    mp.mp.dps = 40
    K = mp.mpf(K)
    if n == 1:
        t = mp.tanh(K)
        return float((t + t ** (L - 1)) / (1 + t ** L))
    if n == 2:
        # transfer-matrix eigenvalues lambda_p = I_p(K); Z = sum_p lambda_p^L
        # (d/dK I_p = (I_{p-1} + I_{p+1}) / 2, I_{-p} = I_p)
        P = 40

        def I(p):
            return mp.besseli(abs(p), K)

        num = sum(I(p) ** (L - 1) * (I(p - 1) + I(p + 1)) / 2 for p in range(-P, P + 1))
        den = sum(I(p) ** L for p in range(-P, P + 1))
        return float(num / den)
    if n == 3:
        # lambda_l = i_l(K) (modified spherical Bessel), degeneracy 2l + 1; d ln Z / dK / L
        P = 40

        def il(l, x):
            return mp.sqrt(mp.pi / (2 * x)) * mp.besseli(l + mp.mpf(1) / 2, x)

        def lnZ(x):
            return mp.log(sum((2 * l + 1) * il(l, x) ** L for l in range(P)))

        return float(mp.diff(lnZ, K) / L)
    raise ValueError(n)


# ----------------------------------------------------------------- 3D high-T series
def sc_ising_series_minus_e(K):
    """-e of the simple-cubic Ising model from ln Z/N = ln 2 + 3 ln cosh K + 3 v^4 + 22 v^6 + 187.5 v^8,
    v = tanh K (standard high-temperature series).  Returns (value, next-term scale)."""
    v = np.tanh(K)
    dv = 1 - v * v
    val = 3 * v + (12 * v ** 3 + 132 * v ** 5 + 1500 * v ** 7) * dv
    return float(val), float(1980 * 10 * v ** 9)  # crude bound on the first omitted term


# ----------------------------------------------------------------- 3D high-T series, O(n)
def on_bond_function(n, K):
    """t(K) = <s.s'> of two O(n) unit spins joined by one bond: tanh K, I_1/I_0, coth K - 1/K (n = 1, 2, 3)."""
    mp.mp.dps = 40
    K = mp.mpf(K)
    if n == 1:
        return mp.tanh(K)
    if n == 2:
        return mp.besseli(1, K) / mp.besseli(0, K)
    if n == 3:
        return mp.coth(K) - 1 / K
    raise ValueError(n)


def sc_on_series_minus_e(n, K):
    """-e of the simple-cubic O(n) model to the first lattice term of the high-temperature expansion, derived from the
    definition (Eq. (1)): integrating out bond by bond, ln Z / N = const + 3 ln lambda_0(K) + 3 n t^4 + O(t^6)
    -- 3 bonds per site, 3 elementary plaquettes per site, a closed loop of four bonds weighs n t^4 (the trace over the n
    components; n = 1 gives the Ising series' 3 v^4) -- and -e = d(ln Z / N)/dK with (ln lambda_0)' = t:
        -e = 3 t + 12 n t^3 t'(K).
    Returns (value, scale of the first omitted term ~ 22 n 6 t^5 t')."""
    t = on_bond_function(n, K)
    dt = 1 - t * t - (n - 1) * t / mp.mpf(K)   # t' of the three bond functions above (Bessel-ratio identity)
    val = 3 * t + 12 * n * t ** 3 * dt
    return float(val), float(132 * n * t ** 5 * dt)
