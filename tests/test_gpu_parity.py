"""GPU <-> oracle parity through the C ABI (include/spin.h), run with -m gpu on the B200.

Bar (BASELINE.json north_star): Ising and +-J spins bit-exact after every sweep, E and M equal as integers;
XY / Heisenberg per-sweep energy within 1e-5 relative over the first 10 sweeps, fewer than 1e-6 of the
acceptance decisions differing.  The oracle (oracle/) is the plain CPU restatement of PAPER.md:31-46.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SEED = 11075463
BETA_2D = 0.4406868
BETA_3D = 0.2216546


@pytest.fixture(scope="module")
def P():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1107_5463_b200 as pkg

    pkg.lib()
    return pkg


_PLAIN = False


@pytest.fixture(autouse=True, params=["tuned", "plain"])
def kernels(request):
    """Every test runs twice: with the tuned kernels (strip kernels, the shared-memory-resident small-lattice kernel)
    and with the plain ones (SPIN_OPT_PLAIN_KERNELS: one launch per half-sweep, one thread per site for n >= 2)."""
    global _PLAIN
    _PLAIN = request.param == "plain"
    yield request.param
    _PLAIN = False


def _system(P, *args, **kw):
    G = P.SpinSystem(*args, **kw)
    if _PLAIN:
        G.set_option(P.OPT_PLAIN_KERNELS, 1)
    return G


def _oracle_kind(oracle, coupling):
    return {"uniform": oracle.J_UNIFORM, "per_direction": oracle.J_PER_DIRECTION, "bond_pm1": oracle.J_BOND_PM1}[coupling]


def _pair(P, oracle, dims, n=1, storage="int8", coupling="uniform", J=(1.0, 1.0, 1.0), replicas=1, replica_streams=0,
          seed=SEED, init=0, rule="metropolis"):
    G = _system(P, dims, n=n, storage=storage, coupling=coupling, J=J, replicas=replicas,
                     replica_streams=replica_streams, seed=seed, init=init, rule=rule)
    O = oracle.System(dims, n=n, coupling_kind=_oracle_kind(oracle, coupling), J=J, n_replicas=replicas,
                      replica_streams=replica_streams, seed=seed, init=init,
                      rule=oracle.RULE_HEATBATH if rule == "heatbath" else oracle.RULE_METROPOLIS)
    return G, O


def _assert_ising_equal(G, O, tag):
    gs, os_ = G.get_spins(), O.get_spins()
    assert gs.shape == os_.shape
    bad = int(np.count_nonzero(gs != os_))
    assert bad == 0, "%s: %d spins differ" % (tag, bad)
    Eg, Mg = G.measure()
    Eo, Mo = O.measure()
    assert np.array_equal(Eg, Eo), (tag, Eg, Eo)
    assert np.array_equal(Mg, Mo), (tag, Mg, Mo)


ISING_CASES = [
    # dims, storage, beta, sweeps  -- generic kernel (odd shapes, size-2 dimensions)
    ((4, 4, 1), "int8", BETA_2D, 6),
    ((8, 6, 1), "int8", BETA_2D, 6),
    ((66, 2, 1), "int8", BETA_2D, 6),
    ((4, 2, 2), "int8", BETA_3D, 6),
    ((6, 4, 8), "int8", BETA_3D, 6),
    ((2, 2, 2), "int8", BETA_3D, 6),
    # fast int8 kernel (Lx % 64 == 0): several units per row, ragged grids, 2D and 3D
    ((64, 4, 1), "int8", BETA_2D, 8),
    ((128, 6, 1), "int8", BETA_2D, 8),
    ((192, 10, 1), "int8", BETA_2D, 5),
    ((64, 2, 2), "int8", BETA_3D, 8),
    ((128, 6, 4), "int8", BETA_3D, 6),
    ((192, 10, 6), "int8", BETA_3D, 4),
    # bit-packed multi-spin coding
    ((64, 4, 1), "bitpack", BETA_2D, 8),
    ((128, 6, 1), "bitpack", BETA_2D, 8),
    ((192, 10, 1), "bitpack", BETA_2D, 5),
    ((64, 2, 2), "bitpack", BETA_3D, 8),
    ((128, 6, 4), "bitpack", BETA_3D, 6),
    ((192, 10, 6), "bitpack", BETA_3D, 4),
]


@pytest.mark.parametrize("dims,storage,beta,sweeps", ISING_CASES)
def test_ising_bit_exact_every_sweep(P, oracle, dims, storage, beta, sweeps):
    G, O = _pair(P, oracle, dims, storage=storage)
    _assert_ising_equal(G, O, "initial state %s" % (dims,))
    for t in range(sweeps):
        G.sweep(beta, 1)
        O.sweep(beta, 1)
        _assert_ising_equal(G, O, "%s %s sweep %d" % (dims, storage, t))


@pytest.mark.parametrize("storage", ["int8", "bitpack"])
def test_config1_L64_1000_sweeps_recorded(P, oracle, storage):
    """BASELINE config 1: 64 x 64 at beta_c, 1000 sweeps, E and M after every sweep (bit-exact)."""
    import torch

    G, O = _pair(P, oracle, (64, 64, 1), storage=storage)
    dE, dM = G.sweep_record(BETA_2D, 1000)
    torch.cuda.synchronize()
    Eg, Mg = dE.cpu().numpy()[:, 0], dM.cpu().numpy()[:, 0, 0]
    Eo, Mo = np.zeros(1000), np.zeros(1000)
    for t in range(1000):
        O.sweep(BETA_2D, 1)
        e, m = O.measure()
        Eo[t], Mo[t] = e[0], m[0, 0]
    assert np.array_equal(Eg, Eo)
    assert np.array_equal(Mg, Mo)
    _assert_ising_equal(G, O, "config 1 after 1000 sweeps")
    assert G.sweep_counter == 1000


@pytest.mark.parametrize("dims,storage,R,streams", [((64, 6, 1), "int8", 5, 1), ((64, 64, 1), "bitpack", 3, 1),
                                                     ((64, 4, 4), "int8", 2, 1), ((128, 8, 2), "bitpack", 32, 1),
                                                     ((256, 256, 1), "int8", 1, 0), ((256, 258, 1), "int8", 1, 0)])
def test_recorded_sweeps_replicas_small_lattices(P, oracle, dims, storage, R, streams):
    """spin_sweep_record on lattices around the limit of the shared-memory-resident kernel (1024 words per colour):
    E, M of every replica after every sweep, then the spins, against the oracle; split calls continue the chain."""
    import torch

    beta = BETA_2D if dims[2] == 1 else BETA_3D
    G, O = _pair(P, oracle, dims, storage=storage, replicas=R, replica_streams=streams)
    n1, n2 = 7, 6
    dE1, dM1 = G.sweep_record(beta, n1)
    dE2, dM2 = G.sweep_record(beta, n2)
    torch.cuda.synchronize()
    Eg = np.concatenate([dE1.cpu().numpy(), dE2.cpu().numpy()])
    Mg = np.concatenate([dM1.cpu().numpy(), dM2.cpu().numpy()])[:, :, 0]
    for t in range(n1 + n2):
        O.sweep(beta, 1)
        e, m = O.measure()
        assert np.array_equal(Eg[t], e), (t, Eg[t], e)
        assert np.array_equal(Mg[t], m[:, 0]), (t, Mg[t], m[:, 0])
    _assert_ising_equal(G, O, "after recorded sweeps %s" % (dims,))
    assert G.sweep_counter == n1 + n2


@pytest.mark.parametrize("dims,storage", [((64, 16, 1), "int8"), ((64, 16, 1), "bitpack"), ((64, 8, 4), "bitpack"),
                                          ((12, 8, 1), "int8")])
def test_antiferromagnet(P, oracle, dims, storage):
    G, O = _pair(P, oracle, dims, storage=storage, J=(-1.0, -1.0, -1.0))
    for t in range(5):
        G.sweep(0.5, 1)
        O.sweep(0.5, 1)
        _assert_ising_equal(G, O, "J = -1 %s %s sweep %d" % (dims, storage, t))


@pytest.mark.parametrize("beta", [0.0, 50.0, 0.1, 1.0 / 1.1])
@pytest.mark.parametrize("storage,dims", [("int8", (64, 8, 1)), ("bitpack", (64, 8, 4)), ("int8", (10, 8, 1))])
def test_extreme_betas(P, oracle, beta, storage, dims):
    """beta = 0: T = 2^32 (33 bits) -> every spin flips; beta = 50: T = 0."""
    G, O = _pair(P, oracle, dims, storage=storage)
    for t in range(3):
        G.sweep(beta, 1)
        O.sweep(beta, 1)
        _assert_ising_equal(G, O, "beta %g sweep %d" % (beta, t))


def test_per_direction_couplings_generic(P, oracle):
    for J in [(1.0, 0.0, 0.0), (1.0, -1.0, 0.0), (0.0, 1.0, 1.0)]:
        G, O = _pair(P, oracle, (8, 6, 4), coupling="per_direction", J=J)
        for t in range(4):
            G.sweep(0.7, 1)
            O.sweep(0.7, 1)
            _assert_ising_equal(G, O, "J = %s sweep %d" % (J, t))


@pytest.mark.parametrize("dims,storage,R,streams", [
    ((64, 6, 4), "bitpack", 16, 0),   # config 4 shape: 16 realisations, shared update stream
    ((256, 6, 4), "bitpack", 5, 0),   # Lx = 256: one thread per row of four words (config 4's own kernel)
    ((256, 2, 2), "bitpack", 18, 0),  # the same with size-2 dimensions and replica chunks
    ((512, 4, 4), "bitpack", 3, 0),   # two quads per row: the x-neighbour word comes from the adjacent quad
    ((768, 6, 1), "bitpack", 4, 0),   # d = 2, three quads per row
    ((256, 8, 1), "bitpack", 7, 0),   # d = 2, the row is the quad
    ((128, 4, 6), "bitpack", 3, 1),
    ((64, 8, 1), "bitpack", 5, 0),
    ((64, 8, 1), "bitpack", 2, 1),
    ((8, 6, 4), "int8", 3, 0),        # generic kernel with int8 bonds
    ((64, 4, 1), "int8", 2, 1),
])
def test_pm_j_spin_glass_bit_exact(P, oracle, dims, storage, R, streams):
    G, O = _pair(P, oracle, dims, storage=storage, coupling="bond_pm1", replicas=R, replica_streams=streams)
    assert np.array_equal(G.get_bonds(), O.get_bonds())
    _assert_ising_equal(G, O, "+-J initial")
    beta = 1.0 / 1.1
    for t in range(6):
        G.sweep(beta, 1)
        O.sweep(beta, 1)
        _assert_ising_equal(G, O, "+-J %s %s R=%d sweep %d" % (dims, storage, R, t))


@pytest.mark.parametrize("dims,R,rule", [((64, 8, 1), 80, "metropolis"), ((64, 4, 2), 40, "metropolis"),
                                         ((64, 8, 1), 80, "heatbath"), ((64, 4, 2), 33, "heatbath")])
def test_many_realisations_shared_stream(P, oracle, dims, R, rule):
    """many +-J realisations of a small lattice, one random number per site for all of them
    (PAPER.md:52); the replica axis is then split over gridDim.y chunks."""
    G, O = _pair(P, oracle, dims, storage="bitpack", coupling="bond_pm1", replicas=R, replica_streams=0, rule=rule)
    for t in range(4):
        G.sweep(1.0, 1)
        O.sweep(1.0, 1)
        _assert_ising_equal(G, O, "many realisations %s R=%d sweep %d" % (dims, R, t))


def test_pm_j_user_bonds_and_replica_streams_uniform(P, oracle):
    rng = np.random.default_rng(5)
    dims, R = (64, 4, 2), 4
    N = dims[0] * dims[1] * dims[2]
    bonds = (1 - 2 * rng.integers(0, 2, size=(R, 3, N))).astype(np.int8)
    for storage in ("bitpack", "int8"):
        G = _system(P, dims, storage=storage, coupling="bond_pm1", bonds=bonds, replicas=R, seed=3)
        O = oracle.System(dims, coupling_kind=oracle.J_BOND_PM1, bonds=bonds, n_replicas=R, seed=3)
        assert np.array_equal(G.get_bonds(), bonds)
        for t in range(4):
            G.sweep(0.8, 1)
            O.sweep(0.8, 1)
            _assert_ising_equal(G, O, "user bonds %s sweep %d" % (storage, t))
    # uniform couplings, several replicas with their own streams (int8 fast + bitpack)
    for storage in ("bitpack", "int8"):
        G, O = _pair(P, oracle, (64, 6, 1), storage=storage, replicas=3, replica_streams=1)
        for t in range(4):
            G.sweep(BETA_2D, 1)
            O.sweep(BETA_2D, 1)
            _assert_ising_equal(G, O, "replica streams %s sweep %d" % (storage, t))


@pytest.mark.parametrize("storage,dims", [("int8", (128, 10, 1)), ("bitpack", (128, 10, 6)), ("int8", (10, 6, 4))])
def test_launch_shape_and_call_splitting_do_not_matter(P, oracle, storage, dims):
    beta = 0.3
    A = _system(P, dims, storage=storage, seed=SEED)
    B = _system(P, dims, storage=storage, seed=SEED)
    B.set_launch_shape(64, 1, 37)
    A.sweep(beta, 10)
    for _ in range(10):
        B.sweep(beta, 1)
    assert np.array_equal(A.get_spins(), B.get_spins())
    O = oracle.System(dims, seed=SEED)
    O.sweep(beta, 10)
    assert np.array_equal(A.get_spins(), O.get_spins())
    # checkpoint / resume: state = spins + sweep counter
    C2 = _system(P, dims, storage=storage, seed=SEED, init=P.INIT_COLD)
    C2.set_spins(A.get_spins())
    C2.sweep_counter = A.sweep_counter
    A.sweep(beta, 3)
    C2.sweep(beta, 3)
    assert np.array_equal(A.get_spins(), C2.get_spins())


@pytest.mark.parametrize("dims,J", [((128, 10, 1), 1.0), ((192, 6, 4), 1.0), ((64, 22, 1), -1.0), ((2048, 34, 1), 1.0)])
def test_int8_strip_rows_do_not_matter(P, oracle, dims, J):
    """The int8 kernel's rows-per-thread knob (register-rolled neighbour rows, ragged last strip, warps that
    straddle rows and warps inside one row) never changes a spin: every K against the oracle."""
    beta = BETA_2D if dims[2] == 1 else BETA_3D
    O = oracle.System(dims, J=(J, J, J), seed=SEED)
    O.sweep(beta, 3)
    want = O.get_spins()
    Eo, Mo = O.measure()
    for rows in (1, 2, 4, 8, 16):
        for block in (64, 256):
            G = _system(P, dims, storage="int8", J=(J, J, J), seed=SEED)
            G.set_strip_rows(rows)
            G.set_launch_shape(block, 1, 1)
            G.sweep(beta, 3)
            assert np.array_equal(G.get_spins(), want), (rows, block)
            Eg, Mg = G.measure()
            assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    with pytest.raises(P.SpinError):
        G.set_strip_rows(3)


@pytest.mark.parametrize("n,dims,beta", [(3, (16, 16, 16), 0.693), (2, (16, 16, 16), 0.4542), (3, (32, 32, 1), 0.693),
                                         (2, (32, 32, 1), 1.1), (3, (6, 4, 2), 0.693), (2, (4, 2, 2), 0.5)])
def test_vector_models_within_tolerance(P, oracle, n, dims, beta):
    G, O = _pair(P, oracle, dims, n=n, storage="fp32")
    N = dims[0] * dims[1] * dims[2]
    g0, o0 = G.get_spins(), O.get_spins()
    assert np.max(np.abs(g0 - o0)) <= 2.4e-7, "hot start differs by more than 2 ulp"
    mismatched_sites = 0
    for t in range(10):
        G.sweep(beta, 1)
        O.sweep(beta, 1)
        Eg, Mg = G.measure()
        Eo, Mo = O.measure()
        assert abs(Eg[0] - Eo[0]) <= 1e-5 * abs(Eo[0]), (t, Eg, Eo)
        assert np.max(np.abs(Mg - Mo)) <= 1e-5 * N
        # a differing acceptance decision leaves a spin that differs by O(1), not by rounding
        diff = np.max(np.abs(G.get_spins() - O.get_spins()), axis=2)
        mismatched_sites += int(np.count_nonzero(diff > 1e-4))
    assert mismatched_sites <= max(0, int(1e-6 * 10 * N)), mismatched_sites
    norm = np.linalg.norm(G.get_spins(), axis=2)
    assert np.max(np.abs(norm - 1.0)) < 4e-7


@pytest.mark.parametrize("n,dims,J", [(3, (16, 6, 4), (1.0, 1.0, 1.0)), (2, (24, 10, 1), (1.0, 1.0, 1.0)),
                                      (3, (8, 4, 2), (1.0, -1.0, 0.5)), (2, (8, 2, 6), (-1.0, -1.0, -1.0)),
                                      # couplings whose products J s are inexact: a contracted multiply-add (one rounding) would show
                                      (3, (16, 8, 6), (0.3, 0.7, -1.3)), (2, (16, 12, 1), (1.1, -0.9, 1.0))])
def test_vector_strip_rows_and_plain_kernel_agree_bitwise(P, n, dims, J):
    """n >= 2: the strip kernel (quads of 4 sites, K = 1, 2, 4 rows per thread, several block sizes) and the plain
    one-thread-per-site kernel perform the same fp32 operations in the same order: identical bits."""
    beta = 0.7
    coupling = "uniform" if J[0] == J[1] == J[2] else "per_direction"
    ref = P.SpinSystem(dims, n=n, storage="fp32", coupling=coupling, J=J, seed=5)
    ref.set_option(P.OPT_PLAIN_KERNELS, 1)
    ref.sweep(beta, 4)
    want = ref.get_spins()
    for rows in (0, 1, 2, 4):
        for block in (64, 128):
            G = P.SpinSystem(dims, n=n, storage="fp32", coupling=coupling, J=J, seed=5)
            G.set_option(P.OPT_TMA_KERNELS, 0)   # the strip kernel itself (d = 3 would take the TMA-staged one: test_gpu_tma.py)
            G.set_strip_rows(rows)
            G.set_launch_shape(block, 1, 1)
            G.sweep(beta, 4)
            assert np.array_equal(G.get_spins().view(np.uint32), want.view(np.uint32)), (rows, block)


def test_vector_per_direction_and_replicas(P, oracle):
    G, O = _pair(P, oracle, (16, 8, 4), n=3, storage="fp32", coupling="per_direction", J=(1.0, 0.0, 0.5), replicas=3,
                 replica_streams=1)
    for t in range(5):
        G.sweep(1.0, 1)
        O.sweep(1.0, 1)
        Eg, Mg = G.measure()
        Eo, Mo = O.measure()
        assert np.allclose(Eg, Eo, rtol=1e-5, atol=1e-4)
        assert np.allclose(Mg, Mo, rtol=1e-5, atol=1e-3)


def test_measure_matches_oracle_on_identical_spins(P, oracle):
    """E and M of the SAME configuration (set_spins from the oracle's state): fp64 sums, 1e-12 relative."""
    for n, dims in [(3, (8, 6, 4)), (2, (12, 10, 1))]:
        O = oracle.System(dims, n=n, seed=7)
        O.sweep(0.6, 3)
        G = _system(P, dims, n=n, storage="fp32", seed=1)
        G.set_spins(O.get_spins())
        assert np.array_equal(G.get_spins(), O.get_spins())
        Eg, Mg = G.measure()
        Eo, Mo = O.measure()
        assert np.allclose(Eg, Eo, rtol=1e-12, atol=1e-9)
        assert np.allclose(Mg, Mo, rtol=1e-12, atol=1e-9)


def test_error_paths(P):
    with pytest.raises(P.SpinError) as e:
        P.SpinSystem((64, 64, 1), storage="bitpack", coupling="per_direction", J=(1.0, 0.0, 0.0))
    assert e.value.status == 2
    with pytest.raises(P.SpinError):
        P.SpinSystem((32, 32, 1), storage="bitpack")
    S = P.SpinSystem((64, 4, 1))
    with pytest.raises(P.SpinError):
        S.sweep(-1.0, 1)
    with pytest.raises(P.SpinError):
        S.sweep(float("nan"), 1)
    with pytest.raises(P.SpinError):
        S.set_spins(np.zeros((1, 256), dtype=np.int8))
    S.sweep_counter = 2 ** 32 - 1
    S.sweep(0.4, 1)
    with pytest.raises(P.SpinError) as e:
        S.sweep(0.4, 1)
    assert e.value.status == 5


# --------------------------------------------------------------------------- heat bath
HEATBATH_CASES = [
    # dims, storage, coupling, J, R, streams, beta
    ((8, 6, 1), "int8", "uniform", 1.0, 1, 0, BETA_2D),            # generic kernel
    ((6, 4, 8), "int8", "uniform", 1.0, 2, 1, BETA_3D),
    ((4, 2, 2), "int8", "bond_pm1", 1.0, 3, 1, 0.6),               # size-2 dimensions, per-bond couplings
    ((66, 4, 1), "int8", "per_direction", 1.0, 1, 0, 0.7),         # zero coupling in z / odd local fields
    ((128, 10, 1), "int8", "uniform", 1.0, 1, 0, BETA_2D),         # int8 fast kernel, ragged strips
    ((192, 6, 4), "int8", "uniform", -1.0, 1, 0, BETA_3D),         # antiferromagnet
    ((2048, 34, 1), "int8", "uniform", 1.0, 1, 0, BETA_2D),        # beyond the resident kernel's limit
    ((128, 6, 1), "bitpack", "uniform", 1.0, 1, 0, BETA_2D),
    ((192, 10, 6), "bitpack", "uniform", 1.0, 1, 0, BETA_3D),
    ((64, 130, 4), "bitpack", "uniform", 1.0, 2, 1, BETA_3D),      # one-launch-per-half-sweep bit-packed kernel
    ((64, 6, 4), "bitpack", "bond_pm1", 1.0, 4, 0, 1.0 / 1.1),     # +-J, shared update stream (config 4 shape)
    ((64, 6, 4), "bitpack", "bond_pm1", 1.0, 3, 1, 1.0 / 1.1),
    ((64, 12, 1), "bitpack", "bond_pm1", 1.0, 5, 0, 0.8),
    ((256, 4, 6), "bitpack", "bond_pm1", 1.0, 6, 0, 1.0 / 1.1),    # Lx = 256: the quad kernel, row = quad
    ((512, 6, 1), "bitpack", "bond_pm1", 1.0, 5, 0, 0.8),          # d = 2, two quads per row
]


@pytest.mark.parametrize("dims,storage,coupling,J,R,streams,beta", HEATBATH_CASES)
def test_ising_heatbath_bit_exact_every_sweep(P, oracle, dims, storage, coupling, J, R, streams, beta):
    Jv = (J, J, 0.0) if coupling == "per_direction" else (J, J, J)
    G, O = _pair(P, oracle, dims, storage=storage, coupling=coupling, J=Jv, replicas=R, replica_streams=streams,
                 rule="heatbath")
    for t in range(5):
        G.sweep(beta, 1)
        O.sweep(beta, 1)
        _assert_ising_equal(G, O, "heat bath %s %s sweep %d" % (dims, storage, t))
    # limits: beta = 0 is a fair coin per site (still bit-exact); beta = 50 aligns every spin with its field
    for b in (0.0, 50.0):
        G.sweep(b, 2)
        O.sweep(b, 2)
        _assert_ising_equal(G, O, "heat bath %s beta %g" % (dims, b))


def test_heatbath_recorded_sweeps(P, oracle):
    import torch

    G, O = _pair(P, oracle, (64, 64, 1), storage="int8", replicas=2, replica_streams=1, rule="heatbath")
    dE, dM = G.sweep_record(BETA_2D, 40)
    torch.cuda.synchronize()
    Eg, Mg = dE.cpu().numpy(), dM.cpu().numpy()[:, :, 0]
    for t in range(40):
        O.sweep(BETA_2D, 1)
        e, m = O.measure()
        assert np.array_equal(Eg[t], e) and np.array_equal(Mg[t], m[:, 0]), t
    _assert_ising_equal(G, O, "heat bath recorded")


@pytest.mark.parametrize("dims,J", [((16, 16, 16), (1.0, 1.0, 1.0)), ((32, 32, 1), (1.0, 1.0, 1.0)),
                                    ((8, 6, 4), (1.0, -1.0, 0.5)), ((6, 4, 4), (1.0, 1.0, 1.0))])
def test_heisenberg_heatbath_within_tolerance(P, oracle, dims, J):
    """n = 3 heat bath: per-sweep energy within 1e-5 relative over the first 10 sweeps, spins within 1e-4
    (both sides fp32 in the same order; only expf / logf / sincospif differ from the oracle's once-rounded values)."""
    coupling = "uniform" if J[0] == J[1] == J[2] else "per_direction"
    G, O = _pair(P, oracle, dims, n=3, storage="fp32", coupling=coupling, J=J, rule="heatbath")
    N = dims[0] * dims[1] * dims[2]
    bad = 0
    for t in range(10):
        G.sweep(0.693, 1)
        O.sweep(0.693, 1)
        Eg, Mg = G.measure()
        Eo, Mo = O.measure()
        assert abs(Eg[0] - Eo[0]) <= 1e-5 * abs(Eo[0]), (t, Eg, Eo)
        assert np.max(np.abs(Mg - Mo)) <= 1e-5 * N
        diff = np.max(np.abs(G.get_spins() - O.get_spins()), axis=2)
        bad += int(np.count_nonzero(diff > 1e-4))
        assert np.max(np.abs(np.linalg.norm(G.get_spins()[0].astype(np.float64), axis=1) - 1.0)) < 1e-5
    assert bad <= max(0, int(1e-6 * 10 * N)), bad


def test_heatbath_is_unsupported_for_xy(P):
    with pytest.raises(P.SpinError) as e:
        P.SpinSystem((8, 8, 1), n=2, storage="fp32", rule="heatbath")
    assert e.value.status == 2


# --------------------------------------------------------------------------- CUDA-graph replay (launch-bound sizes)
@pytest.mark.parametrize("dims,storage,rule", [((128, 600, 1), "int8", "metropolis"), ((64, 70, 20), "bitpack", "metropolis"),
                                               ((128, 520, 1), "bitpack", "heatbath")])
def test_graph_replayed_sweeps_ising(P, oracle, dims, storage, rule):
    """spin_sweep with many sweeps on a lattice beyond the resident kernel's limit replays a CUDA graph of 16 sweeps
    whose launches read the sweep counter from device memory: 40 sweeps = 2 graphs + 8 plain sweeps, then another beta
    (graph rebuilt), a changed launch shape, and a counter set by hand -- bit-exact against the oracle throughout."""
    G, O = _pair(P, oracle, dims, storage=storage, rule=rule)
    for beta, n in ((0.4406868, 40), (0.3, 33)):
        G.sweep(beta, n)
        O.sweep(beta, n)
        _assert_ising_equal(G, O, "graph %s beta %g" % (dims, beta))
    G.set_launch_shape(64, 1, 1)
    G.sweep_counter = 1000
    O.sweep_counter = 1000
    G.sweep(0.3, 32)
    O.sweep(0.3, 32)
    _assert_ising_equal(G, O, "graph after counter change")
    assert G.sweep_counter == 1032


@pytest.mark.parametrize("n", [2, 3])
def test_graph_replayed_sweeps_vector(P, n):
    dims = (32, 32, 16)
    A = P.SpinSystem(dims, n=n, storage="fp32", seed=9)
    B = P.SpinSystem(dims, n=n, storage="fp32", seed=9)
    A.sweep(0.6, 37)                 # 2 graphs + 5 plain sweeps
    for _ in range(37):
        B.sweep(0.6, 1)              # never reaches the graph threshold
    assert np.array_equal(A.get_spins().view(np.uint32), B.get_spins().view(np.uint32))
    assert A.sweep_counter == B.sweep_counter == 37


@pytest.mark.parametrize("dims,storage,J,R,rule", [((128, 600, 1), "int8", 1.0, 1, "metropolis"), ((128, 520, 1), "bitpack", -1.0, 2, "metropolis"),
                                                   ((64, 70, 20), "bitpack", 1.0, 1, "heatbath"), ((64, 34, 22), "int8", 1.0, 3, "heatbath"),
                                                   ((192, 300, 1), "int8", -1.0, 1, "metropolis")])
def test_fused_measurement_in_recorded_sweeps(P, oracle, dims, storage, J, R, rule):
    """spin_sweep_record beyond the resident kernel's limit: E and M are accumulated by the colour-1 half-sweep itself
    (every bond joins the two colours) and must equal the oracle's sums after every sweep; warps that
    straddle two replicas, ragged strips, antiferromagnet, both rules."""
    import torch

    beta = BETA_2D if dims[2] == 1 else BETA_3D
    G, O = _pair(P, oracle, dims, storage=storage, J=(J, J, J), replicas=R, replica_streams=1, rule=rule)
    dE, dM = G.sweep_record(beta, 6)
    torch.cuda.synchronize()
    Eg, Mg = dE.cpu().numpy(), dM.cpu().numpy()[:, :, 0]
    for t in range(6):
        O.sweep(beta, 1)
        e, m = O.measure()
        assert np.array_equal(Eg[t], e) and np.array_equal(Mg[t], m[:, 0]), (t, Eg[t], e, Mg[t], m[:, 0])
    _assert_ising_equal(G, O, "after fused recorded sweeps")     # spin_measure (separate pass) agrees as well


@pytest.mark.parametrize("dims,R,streams,rule", [((256, 12, 6), 5, 0, "metropolis"), ((512, 10, 1), 3, 0, "metropolis"),
                                                 ((256, 6, 4), 4, 0, "heatbath"), ((64, 40, 6), 70, 0, "metropolis"),
                                                 ((128, 36, 1), 40, 0, "metropolis"), ((64, 34, 20), 2, 1, "metropolis")])
def test_fused_measurement_in_recorded_sweeps_pm_j(P, oracle, dims, R, streams, rule):
    """The same for the +-J kernels (row a7 for per-bond couplings): the quad kernel (Lx % 256 == 0, both rules), the
    one-thread-per-word kernel with a shared update stream (replica chunks over gridDim.y) and with own streams; E and M
    of every sweep equal the oracle's, and no measurement pass is launched for the Metropolis kernels."""
    import torch

    beta = 1.0 / 1.1
    G, O = _pair(P, oracle, dims, storage="bitpack", coupling="bond_pm1", replicas=R, replica_streams=streams, rule=rule)
    if G.N * R // 64 <= 1024:
        pytest.skip("resident kernel territory")
    l0 = G.launch_count
    dE, dM = G.sweep_record(beta, 5)
    torch.cuda.synchronize()
    if not _PLAIN and (rule == "metropolis" or dims[0] % 256 == 0):
        assert G.launch_count - l0 == 3 * 5, "two half-sweeps and one finalize per recorded sweep"
    Eg, Mg = dE.cpu().numpy(), dM.cpu().numpy()[:, :, 0]
    for t in range(5):
        O.sweep(beta, 1)
        e, m = O.measure()
        assert np.array_equal(Eg[t], e) and np.array_equal(Mg[t], m[:, 0]), (t, Eg[t], e, Mg[t], m[:, 0])
    _assert_ising_equal(G, O, "after fused recorded sweeps (+-J)")


@pytest.mark.parametrize("n", [2, 3])
def test_direction_map_accuracy(P, oracle, n):
    """The kernels' own sincospi (exact integer range reduction + two polynomials) against the oracle's double-precision,
    once-rounded direction map (R-12: at most 2 ulp) on the 2.6e5 hot-start spins of a 64^3 lattice: every component
    within 2 ulp of 1 (2.4e-7); unit length to 3e-7."""
    dims = (64, 64, 64)
    G = P.SpinSystem(dims, n=n, storage="fp32", seed=123)
    O = oracle.System(dims, n=n, seed=123)
    g, o = G.get_spins()[0].astype(np.float64), O.get_spins()[0].astype(np.float64)
    assert np.max(np.abs(g - o)) <= 2.4e-7, np.max(np.abs(g - o))
    assert np.max(np.abs(np.linalg.norm(g, axis=1) - 1.0)) <= 3e-7


def test_stream_aware_get_set_spins(P, oracle):
    """spin_set_spins_async / spin_set_spins_status and the device-canonical calls (caller-owned memory, no device-wide
    synchronisation): same bytes as the blocking calls; a bad Ising value is reported and leaves the arrays untouched."""
    import torch

    for kw, dims in ((dict(n=1, storage="int8"), (128, 16, 1)), (dict(n=1, storage="bitpack"), (64, 6, 4)), (dict(n=3, storage="fp32"), (8, 6, 4))):
        A, B = P.SpinSystem(dims, seed=3, **kw), P.SpinSystem(dims, seed=4, **kw)
        ref = A.get_spins()
        d = A.get_spins_device()
        assert np.array_equal(d.cpu().numpy(), ref)
        host = torch.from_numpy(ref).pin_memory()
        B.set_spins_async(host.numpy())
        B.set_spins_status()
        assert np.array_equal(B.get_spins(), ref)
        C2 = P.SpinSystem(dims, seed=5, **kw)
        flag = C2.set_spins_device(d)
        torch.cuda.synchronize()
        assert (flag is None or int(flag.item()) == 0) and np.array_equal(C2.get_spins(), ref)
        if kw["n"] == 1:
            bad = ref.copy()
            bad[0, 7] = 0
            before = B.get_spins()
            B.set_spins_async(bad)
            with pytest.raises(P.SpinError):
                B.set_spins_status()
            assert np.array_equal(B.get_spins(), before)
            flag = C2.set_spins_device(torch.from_numpy(bad).cuda())
            torch.cuda.synchronize()
            assert int(flag.item()) != 0 and np.array_equal(C2.get_spins(), ref)


@pytest.mark.parametrize("dims,storage,R", [((128, 16, 1), "int8", 2), ((128, 12, 1), "bitpack", 3), ((64, 6, 4), "bitpack", 1),
                                             ((16, 6, 1), "int8", 1), ((64, 6, 4), "int8", 2)])
def test_canonical_bit_arrays(P, dims, storage, R):
    """spin_set_spins_bits_async / spin_get_spins_bits: the canonical configuration as one bit per spin (an eighth of the
    bytes across PCIe) is the same configuration as the int8 canonical array, for every n = 1 layout."""
    import torch

    A = P.SpinSystem(dims, n=1, storage=storage, replicas=R, replica_streams=1, seed=31)
    A.sweep(0.4, 2)
    ref = A.get_spins()
    bits = A.get_spins_bits()
    assert np.array_equal(bits, np.packbits(ref < 0, axis=1, bitorder="little"))
    B = P.SpinSystem(dims, n=1, storage=storage, replicas=R, replica_streams=1, seed=31)
    B.sweep(0.1, 1)                                    # some other configuration, overwritten by the upload
    pinned = torch.from_numpy(bits).pin_memory()
    B.set_spins_bits_async(pinned.numpy())
    torch.cuda.synchronize()
    assert np.array_equal(B.get_spins(), ref)
    B.sweep_counter = A.sweep_counter
    A.sweep(0.4, 3)
    B.sweep(0.4, 3)
    assert np.array_equal(A.get_spins(), B.get_spins())


@pytest.mark.parametrize("dims,R,beta", [((256, 6, 4), 3, 1.0 / 1.1), ((512, 10, 1), 2, 0.7), ((256, 4, 2), 1, 0.9), ((768, 2, 6), 5, 0.0),
                                         ((256, 34, 1), 40, 50.0)])
def test_pm_j_own_streams_quad_kernel(P, oracle, dims, R, beta):
    """+-J couplings with an OWN update stream per replica on rows of whole quads (ising_pmj_quad_own_halfsweep: one thread per
    quad, deferred digit tails finished through the per-warp queue, replica chunks over gridDim.y): bit-exact against the
    oracle after every sweep, also through recorded sweeps (whose colour-1 half runs the fused word kernel) and with the
    one-thread-per-word kernel as A/B partner."""
    import torch

    G, O = _pair(P, oracle, dims, storage="bitpack", coupling="bond_pm1", replicas=R, replica_streams=1)
    H = _system(P, dims, storage="bitpack", coupling="bond_pm1", replicas=R, replica_streams=1, seed=SEED)
    H.set_option(P.OPT_KERNEL_VARIANT, 1)
    for t in range(4):
        G.sweep(beta, 1)
        H.sweep(beta, 1)
        O.sweep(beta, 1)
        _assert_ising_equal(G, O, "sweep %d" % t)
    assert np.array_equal(G.get_spins(), H.get_spins())
    dE, dM = G.sweep_record(beta, 3)
    torch.cuda.synchronize()
    O.sweep(beta, 3)
    Eo, Mo = O.measure()
    assert np.array_equal(dE[-1].cpu().numpy(), Eo) and np.array_equal(dM[-1, :, 0].cpu().numpy(), Mo[:, 0])
    G.sweep(beta, 40)          # CUDA-graph replay for the small ones
    O.sweep(beta, 40)
    _assert_ising_equal(G, O, "after 47 sweeps")
