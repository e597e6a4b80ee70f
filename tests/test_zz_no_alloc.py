"""spin_measure_noalloc (include/spin.h): the measurement for callers that may not allocate -- its scratch is a fixed
1 MiB array inside the library instead of cudaMalloc'ed or workspace memory.  Collected last on purpose (the suite runs
with pytest -x).  Checks, on two calls in a row and with another handle's call in between (the array is shared and keeps
the last call's contents): the values equal spin_measure's -- exactly for n = 1 (integers), within the 1e-12 relative
tolerance the tests use for fp64 sums of the same spins for n = 2, 3 -- the free device memory does not change across
the calls, and a system whose scratch would not fit is refused with a clear error."""
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


def _noalloc(S):
    import torch

    d_E = torch.full((S.R,), float("nan"), dtype=torch.float64, device=S.device)
    d_M = torch.full((S.R, S.n), float("nan"), dtype=torch.float64, device=S.device)
    S.measure_noalloc(d_E, d_M)
    torch.cuda.synchronize()
    return d_E.cpu().numpy(), d_M.cpu().numpy()


def test_measure_noalloc_matches_spin_measure_twice_in_a_row(P):
    import torch

    systems = [
        (P.SpinSystem((16, 16, 16), n=3, storage="fp32", replicas=3, replica_streams=1, seed=11), 0.693),
        (P.SpinSystem((128, 24, 1), n=1, storage="int8", replicas=2, replica_streams=1, seed=12), 0.44),
        (P.SpinSystem((32, 20, 1), n=2, storage="fp32", seed=13), 0.9),
        (P.SpinSystem((64, 6, 4), n=1, storage="bitpack", coupling="bond_pm1", replicas=4, seed=14), 0.9),
        (P.SpinSystem((32, 32, 1), n=1, storage="msc", coupling="bond_pm1", replicas=64, seed=15), 1.0),
        (P.SpinSystem((10, 8, 1), n=1, storage="int8", seed=16), 0.3),
    ]
    free0 = None
    for rnd in range(2):                       # two rounds: every handle is measured twice, other handles in between
        for S, beta in systems:
            S.sweep(beta, 2)
            E_ref, M_ref = S.measure()         # the existing path (scratch in the caller's workspace)
            for call in range(2):              # two calls in a row on the shared array
                E, M = _noalloc(S)
                if S.n == 1:
                    assert np.array_equal(E, E_ref) and np.array_equal(M, M_ref), (rnd, call, S.dims, E, E_ref)
                else:
                    assert np.all(np.abs(E - E_ref) <= 1e-12 * np.abs(E_ref)), (rnd, call, S.dims, E, E_ref)
                    assert np.all(np.abs(M - M_ref) <= 1e-12 * S.N), (rnd, call, S.dims, M, M_ref)
            if free0 is None:
                free0 = torch.cuda.mem_get_info()[0]      # after the first calls: module and scratch array are loaded
    # further calls allocate nothing on the device
    S, _ = systems[0]
    d_E = torch.empty((S.R,), dtype=torch.float64, device=S.device)
    d_M = torch.empty((S.R, S.n), dtype=torch.float64, device=S.device)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    for _ in range(20):
        S.measure_noalloc(d_E, d_M)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1
    for S, _ in systems:
        S.close()


def test_measure_noalloc_refuses_what_does_not_fit(P):
    # 56 Heisenberg replicas of a lattice with 592 measurement CTAs: 56 * 592 * 4 * 8 bytes > 1 MiB
    S = P.SpinSystem((64, 64, 76), n=3, storage="fp32", replicas=56, replica_streams=1, seed=2)
    import torch

    d_E = torch.empty((S.R,), dtype=torch.float64, device=S.device)
    d_M = torch.empty((S.R, 3), dtype=torch.float64, device=S.device)
    with pytest.raises(P.SpinError) as err:
        S.measure_noalloc(d_E, d_M)
    assert err.value.status == 2 and "scratch" in str(err.value)       # SPIN_ERR_UNSUPPORTED
    E, M = S.measure()                                                  # the ordinary path still serves it
    assert np.all(np.isfinite(E))
    S.close()
    T = P.SpinSystem((64, 64, 76), n=3, storage="fp32", replicas=55, replica_streams=1, seed=2)   # the largest that fits
    E_ref, M_ref = T.measure()
    E, M = _noalloc(T)
    assert np.all(np.abs(E - E_ref) <= 1e-12 * np.abs(E_ref)) and np.all(np.abs(M - M_ref) <= 1e-12 * T.N)
    T.close()
