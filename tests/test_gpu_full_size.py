"""Parity at the FULL BASELINE.json sizes, in the launch configuration bench.py times (default knobs, -m gpu).

The oracle cannot sweep 2.7e8 sites in seconds, so the check is on sampled outputs it computes one by one: for random
sites plus the lattice edges (periodic wrap), the new spin is recomputed from the configuration before the sweep
(neighbours of a colour-1 site: after the colour-0 half-sweep), the site's own random numbers (oracle.ising_uniform /
oracle.rand) and the oracle's decision functions, and compared with what the library wrote.  Size-independent
invariants complete it: E and M from spin_measure equal a numpy evaluation of Eq. (1) on the full
configuration, and the hot start follows the seed contract.
"""
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


def _sample_sites(dims, rng, n_random):
    Lx, Ly, Lz = dims
    N = Lx * Ly * Lz
    idx = [rng.integers(0, N, size=n_random, dtype=np.int64)]
    # edges: first / last rows and columns (periodic wrap in every direction), first / last plane
    xs = np.arange(Lx, dtype=np.int64)
    for y in (0, Ly - 1):
        for z in (0, Lz - 1):
            idx.append(xs + Lx * (y + Ly * z))
    ys = rng.integers(0, Ly, size=256, dtype=np.int64)
    zs = rng.integers(0, Lz, size=256, dtype=np.int64)
    for x in (0, 1, Lx - 2, Lx - 1, 62, 63, 64, 65):
        idx.append(x + Lx * (ys + Ly * zs))
    return np.unique(np.concatenate(idx))


def _coords(idx, dims):
    Lx, Ly, Lz = dims
    x = idx % Lx
    y = (idx // Lx) % Ly
    z = idx // (Lx * Ly)
    return x, y, z


def _neighbours(idx, dims):
    """canonical indices of the 2 d neighbours in the order -x, +x, -y, +y, -z, +z and, for each, the site that owns
    the connecting forward bond and its direction"""
    Lx, Ly, Lz = dims
    d = 2 if Lz == 1 else 3
    x, y, z = _coords(idx, dims)
    L = (Lx, Ly, Lz)
    out = []
    for mu in range(d):
        for sgn in (-1, +1):
            q = [x, y, z]
            q[mu] = (q[mu] + sgn) % L[mu]
            nb = q[0] + Lx * (q[1] + Ly * q[2])
            owner = nb if sgn < 0 else idx
            out.append((nb, owner, mu))
    return out


def _full_energy_ising(s, dims, bonds=None):
    Lx, Ly, Lz = dims
    g = s.reshape(Lz, Ly, Lx)
    E = 0
    for mu, axis in enumerate((2, 1, 0)[: (2 if Lz == 1 else 3)]):
        prod = g * np.roll(g, -1, axis=axis)
        if bonds is not None:
            prod = prod * bonds[mu].reshape(Lz, Ly, Lx)
        E -= int(prod.sum(dtype=np.int64))
    return E


def _check_hot_start(oracle, s0, seed, r, idx):
    for i in idx[:4000].tolist():
        w = oracle.rand(seed, i >> 7, r, 0, 16 * 1)
        want = -1 if (w[(i >> 5) & 3] >> (i & 31)) & 1 else 1
        assert s0[i] == want, ("hot start", i)


def _check_ising_sweep(oracle, dims, seed, beta, t, r, rho, before, after, idx, bonds=None, J=1):
    Lx, Ly, Lz = dims
    x, y, z = _coords(idx, dims)
    colour = (x + y + z) & 1
    j = (x >> 1) + (Lx // 2) * (y + Ly * z)
    h = np.zeros(idx.size, dtype=np.int64)
    for nb, owner, mu in _neighbours(idx, dims):
        s_nb = np.where(colour == 0, before[nb], after[nb]).astype(np.int64)   # colour-1 sites see updated colour 0
        Jb = bonds[mu][owner].astype(np.int64) if bonds is not None else J
        h += Jb * s_nb
    dE = 2 * before[idx].astype(np.int64) * h
    T = {k: oracle.threshold(beta, k) for k in range(0, 13)}
    bad = 0
    for k in range(idx.size):
        U = oracle.ising_uniform(seed, int(j[k]), rho, t, int(colour[k]))
        flip = dE[k] <= 0 or U < T[int(dE[k])]
        want = -before[idx[k]] if flip else before[idx[k]]
        bad += int(want != after[idx[k]])
    assert bad == 0, "%d of %d sampled sites differ from the oracle's decision" % (bad, idx.size)


@pytest.mark.parametrize("name", ["ising2d_L16384_int8", "ising2d_L16384_bitpack", "ising3d_L512_bitpack"])
def test_full_size_ising(P, oracle, name):
    w = P.workloads.WORKLOADS[name]
    seed, dims, beta = P.workloads.SEED, w["dims"], w["beta"]
    N = dims[0] * dims[1] * dims[2]
    rng = np.random.default_rng(1)
    idx = _sample_sites(dims, rng, 12000)
    G = P.from_workload(w, seed)
    s0 = G.get_spins()[0]
    _check_hot_start(oracle, s0, seed, 0, idx)
    G.sweep(beta, 1)
    s1 = G.get_spins()[0]
    _check_ising_sweep(oracle, dims, seed, beta, 0, 0, 0, s0, s1, idx)
    with pytest.raises(AssertionError):      # negative control: the wrong sweep index must not reproduce the spins
        _check_ising_sweep(oracle, dims, seed, beta, 1, 0, 0, s0, s1, idx[:3000])
    del s0
    G.sweep(beta, 3)                         # t = 1, 2, 3
    s4 = G.get_spins()[0]
    G.sweep(beta, 1)                         # t = 4
    s5 = G.get_spins()[0]
    _check_ising_sweep(oracle, dims, seed, beta, 4, 0, 0, s4, s5, idx)
    E, M = G.measure()
    assert M[0, 0] == int(s5.sum(dtype=np.int64))
    assert E[0] == _full_energy_ising(s5, dims)
    assert (N - int(M[0, 0])) % 2 == 0 and abs(E[0]) <= (2 if dims[2] == 1 else 3) * N
    assert G.sweep_counter == 5


def test_full_size_pm_j_spin_glass(P, oracle):
    w = P.workloads.WORKLOADS["ea3d_L256_R16_bitpack"]
    seed, dims, beta = P.workloads.SEED, w["dims"], w["beta"]
    rng = np.random.default_rng(2)
    idx = _sample_sites(dims, rng, 5000)
    G = P.from_workload(w, seed)
    bonds = G.get_bonds()                    # (R, 3, N) int8
    before = G.get_spins()
    G.sweep(beta, 1)
    after = G.get_spins()
    for r in (0, 7, 15):
        # bonds follow the seed contract: bit (i & 31) of word mu of rand(i >> 5, r, 0, BONDS)
        for i in idx[:1500].tolist():
            wds = oracle.rand(seed, i >> 5, r, 0, 16 * 2)
            for mu in range(3):
                assert bonds[r, mu, i] == (-1 if (wds[mu] >> (i & 31)) & 1 else 1)
        _check_hot_start(oracle, before[r], seed, r, idx)
        # all 16 realisations share ONE update stream (replica_streams = 0): rho = 0
        _check_ising_sweep(oracle, dims, seed, beta, 0, r, 0, before[r], after[r], idx, bonds=bonds[r])
    E, M = G.measure()
    for r in (0, 15):
        assert M[r, 0] == int(after[r].sum(dtype=np.int64))
        assert E[r] == _full_energy_ising(after[r], dims, bonds=bonds[r])


@pytest.mark.parametrize("name", ["heisenberg3d_L256_fp32", "xy3d_L256_fp32"])
def test_full_size_vector_models(P, oracle, name):
    w = P.workloads.WORKLOADS[name]
    seed, dims, beta, n = P.workloads.SEED, w["dims"], w["beta"], w["n"]
    Lx, Ly, Lz = dims
    rng = np.random.default_rng(3)
    idx = _sample_sites(dims, rng, 6000)
    G = P.from_workload(w, seed)
    before = G.get_spins()[0]                # (N, n) float32
    G.sweep(beta, 1)
    after = G.get_spins()[0]
    x, y, z = _coords(idx, dims)
    colour = (x + y + z) & 1
    j = (x >> 1) + (Lx // 2) * (y + Ly * z)
    h = np.zeros((idx.size, n), dtype=np.float32)
    for nb, _, _ in _neighbours(idx, dims):
        s_nb = np.where((colour == 0)[:, None], before[nb], after[nb]).astype(np.float32)
        h = (h + np.float32(1.0) * s_nb).astype(np.float32)      # J = 1: every product and sum rounded to fp32
    mismatched = 0
    for k in range(idx.size):
        wds = oracle.vector_site_words(seed, n, int(j[k]), 0, 0, int(colour[k]))
        if n == 3:
            snew, wacc = oracle.direction3(wds[0], wds[1]), wds[2]
        else:
            snew, wacc = oracle.direction2(wds[0]), wds[1]
        so = before[idx[k]]
        acc = np.float32(0)
        for a in range(n):
            prod = np.float32(np.float32(snew[a] - so[a]) * h[k, a])
            acc = prod if a == 0 else np.float32(acc + prod)
        want = snew if oracle.vector_accept(beta, float(-acc), wacc) else so
        if np.max(np.abs(want - after[idx[k]])) > 1e-4:
            mismatched += 1
        else:
            assert np.max(np.abs(want - after[idx[k]])) <= 2e-7 * 4     # sincospi / sqrt within a few ulp
    assert mismatched <= 1e-6 * idx.size + 0, "%d of %d sampled decisions differ" % (mismatched, idx.size)
    # invariants: unit length, E and M against a float64 evaluation of Eq. (1) on the full configuration
    nrm = np.linalg.norm(after.astype(np.float64), axis=1)
    assert np.max(np.abs(nrm - 1.0)) < 1e-6
    E, M = G.measure()
    g = after.astype(np.float64).reshape(Lz, Ly, Lx, n)
    Eref = -sum(float((g * np.roll(g, -1, axis=ax)).sum()) for ax in (2, 1, 0))
    assert abs(E[0] - Eref) <= 1e-9 * abs(Eref) + 1e-6
    assert np.allclose(M[0], g.reshape(-1, n).sum(axis=0), rtol=0, atol=1e-6 * Lx * Ly * Lz * 1e-3 + 1e-3)


@pytest.mark.parametrize("name", ["ising2d_L16384_int8", "ising2d_L16384_bitpack", "ising3d_L512_bitpack",
                                  "ea3d_L256_R16_bitpack", "ea3d_L256_R16_bitpack_ownstreams"])
def test_whole_lattice_two_sweeps_against_the_oracle(P, name):
    """SURVEY 8(c) protocol at full size: every byte of spin_get_spins equals the oracle's configuration after two full
    sweeps of the BASELINE lattice (2.7e8 updates per sweep, about 9 s each for the single-threaded oracle), in the
    launch configuration bench.py times -- for config 2 that is ONE launch of the temporal-blocking kernel (f3)."""
    import oracle

    w = P.workloads.WORKLOADS[name]          # "_ownstreams": config 4 with the replica index in the Philox counter
    kinds = {"uniform": oracle.J_UNIFORM, "per_direction": oracle.J_PER_DIRECTION, "bond_pm1": oracle.J_BOND_PM1}
    G = P.from_workload(w, P.workloads.SEED)
    O = oracle.System(w["dims"], n=1, coupling_kind=kinds[w["coupling"]], J=w["J"], n_replicas=w["replicas"],
                      replica_streams=w["replica_streams"], seed=P.workloads.SEED)
    assert np.array_equal(G.get_spins(), O.get_spins()), "hot start"
    l0 = G.launch_count
    G.sweep(w["beta"], 2)
    if name == "ising2d_L16384_int8":
        assert G.launch_count - l0 == 1, "two sweeps in one pass (temporal blocking is the default for int8 at this size)"
    O.sweep(w["beta"], 2)
    gs, os_ = G.get_spins(), O.get_spins()
    bad = int(np.count_nonzero(gs != os_))
    assert bad == 0, "%d of %d spins differ after two sweeps" % (bad, gs.size)
    Eg, Mg = G.measure()
    Eo, Mo = O.measure()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)


@pytest.mark.parametrize("name", ["heisenberg3d_L256_fp32", "xy3d_L256_fp32"])
def test_full_size_vector_kernels_agree_bitwise(P, name):
    """BASELINE config 5 (and its XY companion) at full size: the tuned strip kernel and the plain one-thread-per-site kernel
    take 6.7e8 accept / reject decisions over 20 sweeps from sums that must round identically (R-14) -- a contracted
    multiply-add in the packed arithmetic shows up here as a handful of differing spins (the small parity lattices have too
    few decisions to meet the 1e-7-wide windows in which the rounding of the sum decides)."""
    w = P.workloads.WORKLOADS[name]
    A, B = P.from_workload(w, P.workloads.SEED), P.from_workload(w, P.workloads.SEED)
    B.set_option(P.OPT_PLAIN_KERNELS, 1)
    A.sweep(w["beta"], 20)
    B.sweep(w["beta"], 20)
    a, b = A.get_spins().view(np.uint32), B.get_spins().view(np.uint32)
    bad = int(np.count_nonzero(a != b))
    assert bad == 0, "%d of %d words differ between the strip and the plain kernel" % (bad, a.size)
    Ea, Ma = A.measure()
    Eb, Mb = B.measure()
    assert Ea[0] == Eb[0] and np.array_equal(Ma, Mb)


@pytest.mark.parametrize("dims,storage", [((32768, 32768, 1), "int8"), ((32768, 65534, 1), "bitpack"), ((1024, 1024, 1022), "bitpack")])
def test_maximum_sizes(P, oracle, dims, storage):
    """The largest lattices the library takes (N R < 2^31; 32768 is also the widest row of the temporal-blocking kernel):
    2^30 int8 sites (the default path at this size is one temporal-blocking launch per two sweeps), 2^31 - 65536 bit-packed
    sites in 2D and 2^30 - 2^21 in 3D.  Index arithmetic near 2^31 is what this covers: the hot start, two sweeps on
    sampled sites against the oracle's decision functions (edges and wrap-around included), E and M against numpy."""
    seed, beta = 5, 0.4406868 if dims[2] == 1 else 0.2216546
    N = dims[0] * dims[1] * dims[2]
    assert N < 2 ** 31
    rng = np.random.default_rng(2)
    idx = _sample_sites(dims, rng, 6000)
    G = P.SpinSystem(dims, n=1, storage=storage, seed=seed)
    s0 = G.get_spins()[0]
    _check_hot_start(oracle, s0, seed, 0, idx)
    G.sweep(beta, 1)                         # one plain sweep ...
    s1 = G.get_spins()[0]
    _check_ising_sweep(oracle, dims, seed, beta, 0, 0, 0, s0, s1, idx)
    del s0
    l0 = G.launch_count
    G.sweep(beta, 2)                         # ... then a pair (int8: the temporal-blocking kernel), checked through its second sweep
    if storage == "int8":
        assert G.launch_count - l0 == 1
    H = P.SpinSystem(dims, n=1, storage=storage, seed=seed)
    H.set_option(P.OPT_TEMPORAL_BLOCKING, 0)
    H.sweep(beta, 2)
    s2 = H.get_spins()[0]
    del H
    s3 = G.get_spins()[0]
    _check_ising_sweep(oracle, dims, seed, beta, 2, 0, 0, s2, s3, idx)
    del s2
    E, M = G.measure()
    assert M[0, 0] == int(s3.sum(dtype=np.int64))
    assert E[0] == _full_energy_ising(s3, dims)
    G.close()


@pytest.mark.parametrize("dims,storage,coupling,R", [((4, 4, 1), "int8", "uniform", 65535), ((64, 2, 1), "bitpack", "bond_pm1", 65535),
                                                     ((8, 8, 1), "msc", "bond_pm1", 32 * 2048)])
def test_maximum_replica_counts(P, dims, storage, coupling, R):
    """The most replicas a handle takes (65535: they map to a grid dimension; MSC storage counts groups of 32), each a tiny
    lattice: bit-exact against the oracle after every sweep, E and M of every replica."""
    import oracle

    streams = 1 if coupling == "uniform" else 0
    G = P.SpinSystem(dims, n=1, storage=storage, coupling=coupling, replicas=R, replica_streams=streams, seed=9)
    O = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1 if coupling == "bond_pm1" else oracle.J_UNIFORM, n_replicas=R,
                      replica_streams=streams, seed=9)
    for t in range(3):
        G.sweep(0.6, 1)
        O.sweep(0.6, 1)
        assert np.array_equal(G.get_spins(), O.get_spins()), t
    Eg, Mg = G.measure()
    Eo, Mo = O.measure()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    with pytest.raises(P.SpinError):
        P.SpinSystem(dims, n=1, storage=storage, coupling=coupling, replicas=(R + 32 if storage == "msc" else R + 1) * (33 if storage == "msc" else 1),
                     replica_streams=streams, seed=9)
