"""The closed forms in tests/exact_results.py against the fixture values in tests/golden (SURVEY.md pins
P3, P4, P7, P8, P9, P11) and against each other: Kaufman's finite-lattice formula must reproduce the brute-force
4x4 enumeration, and tend to Onsager's value."""
import os

import numpy as np
import pytest

import exact_results as X

G = X.golden_values()


def _read_dos(fname):
    out = {}
    with open(os.path.join(X.GOLDEN, fname)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            parts = line.split()
            if len(parts) == 2:
                out.setdefault("4x4", {})[int(parts[0])] = int(parts[1])
            else:
                out.setdefault(parts[0], {})[int(parts[1])] = int(parts[2])
    return out


@pytest.mark.parametrize("name,dims,fname", [("4x4", (4, 4, 1), "ising_4x4_dos.txt"),
                                             ("2x2x2", (2, 2, 2), "ising_small3d_dos.txt"),
                                             ("4x2x2", (4, 2, 2), "ising_small3d_dos.txt")])
def test_density_of_states_matches_golden(name, dims, fname):
    gold = _read_dos(fname)[name]
    dos = X.density_of_states(dims)
    assert sum(dos.values()) == 2 ** (dims[0] * dims[1] * dims[2])
    for E, g in dos.items():
        assert gold[-abs(E)] == g  # symmetric in E
    assert set(abs(E) for E in dos) == set(abs(E) for E in gold)


def test_enumeration_moments_match_golden():
    e, absm, m2, _ = X.boltzmann_moments((4, 4, 1), 0.4406868)
    assert e == pytest.approx(G["enum4x4_e_b0.4406868"], abs=1e-11)
    assert absm == pytest.approx(G["enum4x4_absm_b0.4406868"], abs=1e-11)
    assert X.boltzmann_moments((4, 4, 1), 0.5)[0] == pytest.approx(G["enum4x4_e_b0.5"], abs=1e-11)
    assert X.boltzmann_moments((2, 2, 2), 0.2216546)[0] == pytest.approx(G["enum2x2x2_e_b0.2216546"], abs=1e-11)
    assert X.boltzmann_moments((4, 2, 2), 0.2216546)[0] == pytest.approx(G["enum4x2x2_e_b0.2216546"], abs=1e-11)


def test_kaufman_matches_enumeration_and_golden():
    assert X.kaufman_energy_per_spin(4, 0.4406868) == pytest.approx(X.boltzmann_moments((4, 4, 1), 0.4406868)[0], abs=1e-12)
    assert X.kaufman_energy_per_spin(4, 0.3) == pytest.approx(X.boltzmann_moments((4, 4, 1), 0.3)[0], abs=1e-12)
    for L in (4, 8, 16, 32, 64):
        assert X.kaufman_energy_per_spin(L, 0.4406868) == pytest.approx(G["kaufman_e_L%d_b0.4406868" % L], abs=2e-10)


def test_onsager_yang():
    assert X.onsager_energy_per_spin(0.4406868) == pytest.approx(G["onsager_e_inf_b0.4406868"], abs=1e-9)
    assert X.onsager_energy_per_spin(0.4406868) == pytest.approx(-np.sqrt(2.0), abs=1e-6)  # beta literal is 1e-8 off beta_c
    assert X.onsager_energy_per_spin(0.5) == pytest.approx(G["onsager_e_inf_b0.5"], abs=1e-11)
    assert X.yang_magnetisation(0.5) == pytest.approx(G["yang_m_b0.5"], abs=1e-12)
    # finite-size effects at beta = 0.5 are already negligible at L = 32
    assert X.kaufman_energy_per_spin(32, 0.5) == pytest.approx(G["onsager_e_inf_b0.5"], abs=1e-6)


def test_chain_values():
    assert X.chain_bond_average(1, 1.0, 64) == pytest.approx(G["chain_n1_K1_L64"], abs=1e-11)
    assert X.chain_bond_average(1, 1.0, 16) == pytest.approx(G["chain_n1_K1_L16"], abs=1e-11)
    assert X.chain_bond_average(2, 1.0, 64) == pytest.approx(G["chain_n2_K1"], abs=1e-11)
    assert X.chain_bond_average(3, 1.0, 64) == pytest.approx(G["chain_n3_K1"], abs=1e-11)
    assert X.chain_bond_average(2, 2.0, 64) == pytest.approx(G["chain_n2_K2"], abs=2e-10)  # (I1/I0)^64 finite-size term
    assert X.chain_bond_average(3, 2.0, 64) == pytest.approx(G["chain_n3_K2"], abs=2e-10)
    # textbook limits: I1/I0 and coth K - 1/K
    import mpmath as mp
    assert X.chain_bond_average(2, 1.0, 64) == pytest.approx(float(mp.besseli(1, 1) / mp.besseli(0, 1)), abs=1e-10)
    assert X.chain_bond_average(3, 1.0, 64) == pytest.approx(float(mp.coth(1) - 1), abs=1e-10)


def test_series():
    assert X.sc_ising_series_minus_e(0.1)[0] == pytest.approx(G["series3d_K0.1"], abs=1e-7)


def test_on_series_reduces_to_the_ising_series_and_to_its_leading_term():
    """sc_on_series_minus_e: n = 1 must reproduce the first two terms of the Ising series 3 v + 12 v^3 (1 - v^2), and
    for every n the leading behaviour is 3 K / n."""
    import numpy as np
    K = 0.05
    v = np.tanh(K)
    val, omitted = X.sc_on_series_minus_e(1, K)
    assert abs(val - (3 * v + 12 * v ** 3 * (1 - v * v))) < 1e-12
    full, _ = X.sc_ising_series_minus_e(K)
    assert abs(val - full) < 2 * omitted
    for n in (2, 3):
        val, omitted = X.sc_on_series_minus_e(n, K)
        assert abs(val - 3 * K / n) < 3 * K / n * 4 * K * K
        assert omitted < 3e-6
