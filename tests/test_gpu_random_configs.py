"""Randomised GPU <-> oracle parity: seeded random draws over lattice shapes, storage, couplings, replica modes, update
rules, beta and RNG seeds (every kernel family and the ragged / wrap-around cases they dispatch on), a few sweeps each,
spins compared after every sweep.  Deterministic: the draws come from a fixed numpy seed."""
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


def _draw(rng):
    d3 = rng.random() < 0.5
    fast = rng.random() < 0.6
    Lx = int(rng.choice([64, 128, 192, 256])) if fast else int(rng.choice([2, 4, 6, 10, 18, 34, 66, 130]))
    Ly = 2 * int(rng.integers(1, 12))
    Lz = 2 * int(rng.integers(1, 6)) if d3 else 1
    n = int(rng.choice([1, 1, 1, 2, 3]))
    cfg = dict(dims=(Lx, Ly, Lz), n=n, seed=int(rng.integers(0, 2 ** 62)), R=int(rng.choice([1, 1, 2, 3, 4, 5, 8])),
               streams=int(rng.integers(0, 2)), beta=float(rng.choice([0.0, 0.1, 0.2216546, 0.4406868, 0.7, 1.3, 5.0])),
               init=int(rng.integers(0, 2)))
    if n == 1:
        cfg["storage"] = "bitpack" if (fast and rng.random() < 0.5) else "int8"
        kinds = ["uniform", "bond_pm1"] if cfg["storage"] == "bitpack" else ["uniform", "per_direction", "bond_pm1"]
        cfg["coupling"] = str(rng.choice(kinds))
        if cfg["coupling"] == "uniform":
            J = float(rng.choice([1.0, -1.0]))
            cfg["J"] = (J, J, J)
        elif cfg["coupling"] == "per_direction":
            cfg["J"] = tuple(float(v) for v in rng.choice([-1.0, 0.0, 1.0], size=3))
        else:
            cfg["J"] = (1.0, 1.0, 1.0)
        cfg["rule"] = str(rng.choice(["metropolis", "heatbath"]))
    else:
        cfg["storage"] = "fp32"
        cfg["coupling"] = str(rng.choice(["uniform", "per_direction"]))
        cfg["J"] = (1.0, 1.0, 1.0) if cfg["coupling"] == "uniform" else tuple(float(v) for v in rng.choice([-1.0, 0.5, 1.0, 2.0], size=3))
        cfg["rule"] = "heatbath" if (n == 3 and rng.random() < 0.4) else "metropolis"
    return cfg


@pytest.mark.parametrize("case", range(40))
def test_random_configuration_matches_the_oracle(P, oracle, case):
    rng = np.random.default_rng(1107_5463 + case)
    c = _draw(rng)
    kind = {"uniform": oracle.J_UNIFORM, "per_direction": oracle.J_PER_DIRECTION, "bond_pm1": oracle.J_BOND_PM1}[c["coupling"]]
    G = P.SpinSystem(c["dims"], n=c["n"], storage=c["storage"], coupling=c["coupling"], J=c["J"], replicas=c["R"],
                     replica_streams=c["streams"], seed=c["seed"], init=c["init"], rule=c["rule"])
    if rng.random() < 0.3:
        G.set_option(P.OPT_PLAIN_KERNELS, 1)
    if rng.random() < 0.5:
        G.set_launch_shape(int(rng.choice([64, 128, 256])), 1, int(rng.choice([1, 3, 17])))
        G.set_strip_rows(int(rng.choice([1, 2, 4, 8, 16])))
    O = oracle.System(c["dims"], n=c["n"], coupling_kind=kind, J=c["J"], n_replicas=c["R"], replica_streams=c["streams"],
                      seed=c["seed"], init=c["init"],
                      rule=oracle.RULE_HEATBATH if c["rule"] == "heatbath" else oracle.RULE_METROPOLIS)
    N = c["dims"][0] * c["dims"][1] * c["dims"][2]
    for t in range(3):
        G.sweep(c["beta"], 1)
        O.sweep(c["beta"], 1)
        gs, os_ = G.get_spins(), O.get_spins()
        Eg, Mg = G.measure()
        Eo, Mo = O.measure()
        if c["n"] == 1:
            assert np.array_equal(gs, os_), (c, t)
            assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo), (c, t)
        else:
            bad = int(np.count_nonzero(np.max(np.abs(gs - os_), axis=2) > 1e-4))
            assert bad == 0, (c, t, bad)
            scale = max(1.0, float(np.max(np.abs(Eo))))
            assert np.max(np.abs(Eg - Eo)) <= 1e-5 * scale + 1e-6 * N, (c, t, Eg, Eo)
