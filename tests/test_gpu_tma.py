"""The TMA-staged half-sweep of the n >= 2 models (csrc/vector_tma_kernel.cuh; north_star (a), PAPER.md:42 tile + boundary
layer) against the plain one-thread-per-site kernel and the oracle, through the C ABI (-m gpu).

The staged kernel, the strip kernel and the plain kernel perform the same fp32 operations in the same order
(vector_quad_update), so their spins must agree BIT FOR BIT for every tile shape, ring restart pattern (CTAs per replica)
and lattice shape; the plain kernel itself is held to the oracle within north_star's tolerance in test_gpu_parity.py and
here once more with the staged kernel in the loop.  The fused E / M of spin_sweep_record (SURVEY 8(a) row a7,
PAPER.md:44: fp32 terms, fp64 aggregates) is compared with the separate fp64 measurement pass and with the oracle.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SEED = 11075463


@pytest.fixture(scope="module")
def P():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1107_5463_b200 as pkg

    pkg.lib()
    return pkg


# dims, J: full tiles, ragged last row block (Ly % 8 != 0), size-2 dimensions, one tile per plane, rows of 256 sites per
# colour (tile of 4 rows), couplings that are not +1
SHAPES = [
    ((16, 16, 16), (1.0, 1.0, 1.0)),
    ((16, 12, 6), (1.0, 1.0, 1.0)),
    ((8, 6, 4), (1.0, -1.0, 0.5)),
    ((8, 2, 2), (1.0, 1.0, 1.0)),
    ((24, 20, 2), (-1.0, -1.0, -1.0)),
    ((512, 6, 4), (1.0, 1.0, 1.0)),
    ((256, 18, 10), (1.0, 1.0, 1.0)),
]


def _make(P, dims, n, J, tma, replicas=1, replica_streams=0, rule="metropolis", seed=5):
    coupling = "uniform" if J[0] == J[1] == J[2] else "per_direction"
    G = P.SpinSystem(dims, n=n, storage="fp32", coupling=coupling, J=J, seed=seed, replicas=replicas,
                     replica_streams=replica_streams, rule=rule)
    if tma == "plain":
        G.set_option(P.OPT_PLAIN_KERNELS, 1)
    elif tma == "strip":
        G.set_option(P.OPT_TMA_KERNELS, 0)
    else:
        G.set_option(P.OPT_TMA_KERNELS, 1)
    return G


@pytest.mark.parametrize("n", [2, 3])
@pytest.mark.parametrize("dims,J", SHAPES)
def test_tma_kernel_agrees_bitwise_with_plain_and_strip(P, n, dims, J):
    beta = 0.7
    ref = _make(P, dims, n, J, "plain")
    ref.sweep(beta, 4)
    want = ref.get_spins().view(np.uint32)
    strip = _make(P, dims, n, J, "strip")
    strip.sweep(beta, 4)
    assert np.array_equal(strip.get_spins().view(np.uint32), want), "strip kernel"
    # CTAs per replica: all the device takes, then 4, 2 and 1 (one CTA walks every column: ring restarts at each)
    for num, den in ((1, 1), (1, 90), (1, 150), (1, 444), (3, 444 * 2)):
        G = _make(P, dims, n, J, "tma")
        G.set_launch_shape(0, num, den)
        G.sweep(beta, 4)
        assert np.array_equal(G.get_spins().view(np.uint32), want), ("tma", num, den)


@pytest.mark.parametrize("dims,R,streams", [((16, 12, 6), 3, 1), ((8, 6, 4), 5, 0), ((16, 16, 4), 300, 1)])
def test_tma_kernel_replicas_bitwise(P, dims, R, streams):
    for n in (2, 3):
        ref = _make(P, dims, n, (1.0, 1.0, 1.0), "plain", replicas=R, replica_streams=streams)
        G = _make(P, dims, n, (1.0, 1.0, 1.0), "tma", replicas=R, replica_streams=streams)
        for S in (ref, G):
            S.sweep(0.6, 3)
        assert np.array_equal(G.get_spins().view(np.uint32), ref.get_spins().view(np.uint32)), n


def test_tma_heatbath_bitwise(P):
    # the heat-bath spin is arithmetic on the local field, so a contracted multiply-add anywhere (ptxas fuses mul.rn.f32x2 +
    # add.rn.f32x2) shows in the bits; the last case has couplings whose products J s are inexact
    for dims, J in (((16, 12, 6), (1.0, 1.0, 1.0)), ((8, 6, 4), (1.0, 0.5, -1.0)), ((16, 8, 6), (0.3, 0.7, -1.3))):
        ref = _make(P, dims, 3, J, "plain", rule="heatbath")
        G = _make(P, dims, 3, J, "tma", rule="heatbath")
        for S in (ref, G):
            S.sweep(0.9, 3)
        assert np.array_equal(G.get_spins().view(np.uint32), ref.get_spins().view(np.uint32))


@pytest.mark.parametrize("n,beta", [(3, 0.693), (2, 0.4542)])
def test_tma_kernel_against_the_oracle(P, oracle, n, beta):
    """north_star's tolerance with the staged kernel in the loop (32^3: several tiles per plane, several CTAs per column)."""
    dims = (32, 32, 32)
    N = 32 ** 3
    G = P.SpinSystem(dims, n=n, storage="fp32", seed=SEED)
    G.set_option(P.OPT_TMA_KERNELS, 1)
    O = oracle.System(dims, n=n, seed=SEED)
    bad = 0
    for t in range(10):
        G.sweep(beta, 1)
        O.sweep(beta, 1)
        Eg, _ = G.measure()
        Eo, _ = O.measure()
        assert abs(Eg[0] - Eo[0]) <= 1e-5 * abs(Eo[0]), (t, Eg, Eo)
        diff = np.max(np.abs(G.get_spins() - O.get_spins()), axis=2)
        bad += int(np.count_nonzero(diff > 1e-4))
    assert bad <= int(1e-6 * 10 * N), bad


@pytest.mark.parametrize("n,dims,R,J", [(3, (16, 16, 16), 1, (1.0, 1.0, 1.0)), (2, (16, 12, 6), 3, (1.0, 1.0, 1.0)),
                                        (3, (8, 6, 4), 2, (1.0, -1.0, 0.5)), (3, (32, 32, 32), 1, (1.0, 1.0, 1.0))])
@pytest.mark.parametrize("tma", [-1, 1])
def test_fused_measurement_of_recorded_sweeps(P, oracle, n, dims, R, J, tma):
    """spin_sweep_record with the staged kernel: E and M come out of the colour-1 half-sweep (row a7).  Terms are fp32
    (the local field the update has formed), the sums fp64: against the separate fp64 pass on the SAME spins the
    difference is bounded by the fp32 rounding of the N / 2 site terms, |dE| <= 5e-6 N / 2 in the worst case;
    the test holds it to 1e-6 N (1e-6 relative to an energy of order N) and M to 2e-7 N."""
    beta, sweeps = 0.6, 6
    N = dims[0] * dims[1] * dims[2]
    coupling = "uniform" if J[0] == J[1] == J[2] else "per_direction"
    kw = dict(n=n, storage="fp32", coupling=coupling, J=J, seed=9, replicas=R, replica_streams=1)
    A = P.SpinSystem(dims, **kw)
    A.set_option(P.OPT_TMA_KERNELS, tma)
    B = P.SpinSystem(dims, **kw)
    B.set_option(P.OPT_PLAIN_KERNELS, 1)
    O = oracle.System(dims, n=n, coupling_kind=oracle.J_UNIFORM if coupling == "uniform" else oracle.J_PER_DIRECTION, J=J,
                      n_replicas=R, replica_streams=1, seed=9)
    launches0 = A.launch_count
    dE, dM = A.sweep_record(beta, sweeps)
    assert A.launch_count - launches0 == 3 * sweeps, "two half-sweeps and one finalize per recorded sweep: no measurement pass"
    dE, dM = dE.cpu().numpy(), dM.cpu().numpy()
    for t in range(sweeps):
        B.sweep(beta, 1)
        O.sweep(beta, 1)
        Eb, Mb = B.measure()
        assert np.max(np.abs(dE[t] - Eb)) <= 1e-6 * N, (t, dE[t], Eb)
        assert np.max(np.abs(dM[t] - Mb)) <= 2e-7 * N, (t, dM[t], Mb)
        Eo, Mo = O.measure()
        assert np.all(np.abs(dE[t] - Eo) <= 1e-5 * np.abs(Eo)), (t, dE[t], Eo)     # north_star: through the chain
        assert np.max(np.abs(dM[t] - Mo)) <= 1e-5 * N
    assert np.array_equal(A.get_spins().view(np.uint32), B.get_spins().view(np.uint32))
    # recorded and unrecorded sweeps are the same chain
    C = P.SpinSystem(dims, **kw)
    C.sweep(beta, sweeps)
    assert np.array_equal(A.get_spins().view(np.uint32), C.get_spins().view(np.uint32))
