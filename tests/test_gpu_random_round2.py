"""Seeded random configurations of the round-2 kernels against the oracle (companion of test_gpu_random_configs.py):
temporal blocking (random stripe heights, both rules), replica-per-bit coding, the +-J quad kernels (cooperative and
one-thread-per-quad, every L2-hint setting, recorded sweeps), the resident kernel with masks generated ahead (recorded every
sweep), the temperature axis and the canonical bit arrays.  Every case is bit-exact or the test fails; 150 cases, a few
seconds.  (A 7-minute run of the same generator, 15 000 cases, was clean: profiles/r02_all_kernels.md.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _same(G, O, tag, what):
    g, o = G.get_spins(), O.get_spins()
    assert np.array_equal(g, o), (what, tag, int(np.count_nonzero(g != o)))
    Eg, Mg = G.measure()
    Eo, Mo = O.measure()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo), (what, tag)


def test_random_round2_configurations():
    import torch

    import oracle
    import paper_1107_5463_b200 as P

    P.lib()
    same = _same
    rng = np.random.default_rng(20260211)
    n_ok = {"tblock": 0, "msc": 0, "pmj": 0, "resident": 0, "betas": 0, "bits": 0}
    for case in range(150):
        kind = rng.choice(["tblock", "msc", "pmj", "resident", "betas", "bits"])
        seed = int(rng.integers(1, 2**31)); beta = float(rng.choice([0.0, 0.2, 0.4406868, 0.7, 1.2, 30.0]))
        rule = str(rng.choice(["metropolis", "heatbath"])); orule = oracle.RULE_HEATBATH if rule == "heatbath" else oracle.RULE_METROPOLIS
        if kind == "tblock":
            dims = (int(rng.choice([2048, 4096])), int(2 * rng.integers(1, 24)), 1); R = int(rng.integers(1, 3)); J = float(rng.choice([1.0, -1.0]))
            G = P.SpinSystem(dims, n=1, storage="int8", J=(J, J, J), replicas=R, replica_streams=1, seed=seed, rule=rule)
            G.set_option(P.OPT_TEMPORAL_BLOCKING, 1); G.set_option(P.OPT_TBLOCK_ROWS, int(rng.integers(0, dims[1] + 3)))
            O = oracle.System(dims, n=1, J=(J, J, J), n_replicas=R, replica_streams=1, seed=seed, rule=orule)
            for n in rng.integers(1, 6, size=3):
                G.sweep(beta, int(n)); O.sweep(beta, int(n)); same(G, O, (dims, R, J, beta, rule, int(n)), kind)
        elif kind == "msc":
            d3 = rng.random() < 0.4
            dims = (int(2 * rng.integers(2, 20)), int(2 * rng.integers(1, 10)), int(2 * rng.integers(1, 5)) if d3 else 1)
            if (dims[0] * dims[1] * dims[2] // 2) % 32: continue
            R = 32 * int(rng.integers(1, 4))
            G = P.SpinSystem(dims, n=1, storage="msc", coupling="bond_pm1", replicas=R, seed=seed, rule=rule)
            O = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, n_replicas=R, seed=seed, rule=orule)
            for n in (1, 2, 35):
                G.sweep(beta, n); O.sweep(beta, n); same(G, O, (dims, R, beta, rule, n), kind)
        elif kind == "pmj":
            d3 = rng.random() < 0.6
            dims = (int(rng.choice([256, 512])), int(2 * rng.integers(1, 8)), int(2 * rng.integers(1, 5)) if d3 else 1)
            R = int(rng.integers(2, 20))
            G = P.SpinSystem(dims, n=1, storage="bitpack", coupling="bond_pm1", replicas=R, seed=seed, rule=rule)
            G.set_option(P.OPT_KERNEL_VARIANT, int(rng.integers(0, 2))); G.set_option(P.OPT_L2_KEEP, int(rng.choice([-2, -1, 0, 1, R // 2, R])))
            G.set_launch_shape(int(rng.choice([64, 128, 256])), 1, 1)
            O = oracle.System(dims, n=1, coupling_kind=oracle.J_BOND_PM1, n_replicas=R, seed=seed, rule=orule)
            dE, dM = G.sweep_record(beta, 3); O.sweep(beta, 3); same(G, O, (dims, R, beta, rule), kind)
            Eo, Mo = O.measure()
            if not (np.array_equal(dE[-1].cpu().numpy(), Eo) and np.array_equal(dM[-1, :, 0].cpu().numpy(), Mo[:, 0])): raise AssertionError(("recorded +-J", dims, R))
            G.sweep(beta, 2); O.sweep(beta, 2); same(G, O, (dims, R, beta, rule, "plain"), kind)
        elif kind == "resident":
            d3 = rng.random() < 0.4
            dims = (64 * int(rng.integers(1, 3)), int(2 * rng.integers(1, 20)), int(2 * rng.integers(1, 4)) if d3 else 1)
            R = int(rng.integers(1, 5)); st = str(rng.choice(["int8", "bitpack"]))
            if dims[0] * dims[1] * dims[2] * R // 64 > 1024: continue
            G = P.SpinSystem(dims, n=1, storage=st, replicas=R, replica_streams=1, seed=seed, rule=rule)
            O = oracle.System(dims, n=1, n_replicas=R, replica_streams=1, seed=seed, rule=orule)
            n = int(rng.integers(1, 80)); dE, dM = G.sweep_record(beta, n)
            Es = []
            for _ in range(n): O.sweep(beta, 1); Es.append(O.measure())
            same(G, O, (dims, R, st, beta, rule, n), kind)
            if not all(np.array_equal(dE[k].cpu().numpy(), Es[k][0]) and np.array_equal(dM[k, :, 0].cpu().numpy(), Es[k][1][:, 0]) for k in range(n)): raise AssertionError(("recorded resident", dims, R, n))
            G.sweep(beta, int(rng.integers(1, 70))); O.sweep(beta, G.sweep_counter - n); same(G, O, (dims, "unrecorded"), kind)
        elif kind == "betas":
            dims = (int(rng.choice([64, 128, 10])), int(2 * rng.integers(2, 8)), 1); R = int(rng.integers(2, 5)); st = "int8" if dims[0] == 10 else str(rng.choice(["int8", "bitpack"]))
            betas = [float(b) for b in rng.uniform(0.0, 1.0, size=R)]
            G = P.SpinSystem(dims, n=1, storage=st, replicas=R, replica_streams=1, seed=seed, rule=rule)
            G.sweep_betas(betas, 3); g = G.get_spins()
            for r in range(R):
                O = oracle.System(dims, n=1, n_replicas=R, replica_streams=1, seed=seed, rule=orule); O.sweep(betas[r], 3)
                if not np.array_equal(g[r], O.get_spins()[r]): raise AssertionError(("temperature axis", dims, r))
        else:
            dims = (8 * int(rng.integers(1, 20)), int(2 * rng.integers(1, 10)), 1); st = "int8"
            G = P.SpinSystem(dims, n=1, storage=st, replicas=2, replica_streams=1, seed=seed)
            G.sweep(0.3, 1); ref = G.get_spins(); bits = G.get_spins_bits()
            if not np.array_equal(bits, np.packbits(ref < 0, axis=1, bitorder="little")): raise AssertionError(("bits", dims))
            H = P.SpinSystem(dims, n=1, storage=st, replicas=2, replica_streams=1, seed=seed + 1); H.set_spins_bits_async(bits)
            torch.cuda.synchronize()
            if not np.array_equal(H.get_spins(), ref): raise AssertionError(("bits set", dims))
        n_ok[kind] += 1
    assert min(n_ok.values()) >= 5, n_ok
