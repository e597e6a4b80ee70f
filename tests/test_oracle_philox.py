"""Pin P1: the oracle's Philox-4x32-10 against the published known-answer vectors, plus the derived
random-number maps of DESIGN.md "The contract" (one random number per site, drawn unconditionally)."""
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def _kat():
    rows = []
    with open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(x, 16) for x in line.split()]
            rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answers(oracle):
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert oracle.philox4x32_10(ctr, key) == out


def test_philox_is_a_bijection_of_the_counter_sample(oracle):
    # distinct counters give distinct outputs (a keyed bijection); cheap sanity check on 4096 counters
    seen = set()
    for c in range(4096):
        seen.add(tuple(oracle.philox4x32_10([c, 0, 0, 0], [1, 2])))
    assert len(seen) == 4096


def test_rand_is_philox_with_seed_as_key(oracle):
    seed = 0x299F31D0A4093822
    assert oracle.rand(seed, 0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344) == [0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1]


def test_ising_uniform_bitplane_definition(oracle):
    """digit k (MSB first) of site j's uniform = bit (j & 31) of word k & 3 of call k >> 2 of unit j >> 5 (R-16)."""
    seed, rho, t = 11075463, 3, 17
    for colour in (0, 1):
        for j in (0, 1, 31, 32, 77, 4095, (1 << 27) + 5):
            words = []
            for call in range(8):
                words += oracle.rand(seed, j >> 5, rho, t, colour + 256 * call)
            U = 0
            for k in range(32):
                U = (U << 1) | ((words[k] >> (j & 31)) & 1)
            assert oracle.ising_uniform(seed, j, rho, t, colour) == U


def test_ising_uniform_statistics(oracle):
    """uniforms of different sites / sweeps / colours look uniform and independent (mean, variance, lag-1)."""
    seed = 11075463
    U = np.array([oracle.ising_uniform(seed, j, 0, t, c) for t in range(4) for c in (0, 1) for j in range(2048)],
                 dtype=np.float64) / 2.0 ** 32
    n = U.size
    assert abs(U.mean() - 0.5) < 4 * np.sqrt(1 / 12 / n)
    assert abs(U.var() - 1 / 12) < 4 * np.sqrt(1 / 180 / n)
    c1 = np.mean((U[:-1] - 0.5) * (U[1:] - 0.5))
    assert abs(c1) < 4 * (1 / 12) / np.sqrt(n)
    # every bit position is fair
    Ui = (U * 2.0 ** 32).astype(np.uint64)
    for k in (0, 1, 15, 31):
        frac = ((Ui >> np.uint64(k)) & np.uint64(1)).mean()
        assert abs(frac - 0.5) < 4 * 0.5 / np.sqrt(n)
