"""The BASELINE.json workloads as plain data (dims, model, storage, beta, sweeps, seed).

Holds none of the method's arithmetic: the tests, bench.py and the oracle harness all read the same
recipes from here and build their own systems from them.  Every input is synthetic and seeded
(hot start and bonds are drawn from the seed by each implementation's own Philox).
"""
SEED = 11075463

# name -> recipe.  `storage` values name the C-ABI enums (binding.STORE_*).
WORKLOADS = {
    # config 1: 2D Ising L = 64, 1000 sweeps, E and M recorded every sweep
    "ising2d_L64_int8": dict(dims=(64, 64, 1), n=1, storage="int8", coupling="uniform", J=(1.0, 1.0, 1.0),
                             beta=0.4406868, sweeps=1000, replicas=1, replica_streams=0, record=True),
    # config 2: 2D Ising L = 16384, 1000 sweeps, int8 and bit-packed
    "ising2d_L16384_int8": dict(dims=(16384, 16384, 1), n=1, storage="int8", coupling="uniform", J=(1.0, 1.0, 1.0),
                                beta=0.4406868, sweeps=1000, replicas=1, replica_streams=0, record=False),
    "ising2d_L16384_bitpack": dict(dims=(16384, 16384, 1), n=1, storage="bitpack", coupling="uniform",
                                   J=(1.0, 1.0, 1.0), beta=0.4406868, sweeps=1000, replicas=1, replica_streams=0,
                                   record=False),
    # config 3: 3D Ising L = 512, 500 sweeps, multi-spin coded
    "ising3d_L512_bitpack": dict(dims=(512, 512, 512), n=1, storage="bitpack", coupling="uniform", J=(1.0, 1.0, 1.0),
                                 beta=0.2216546, sweeps=500, replicas=1, replica_streams=0, record=False),
    # config 4: 3D +-J Edwards-Anderson L = 256, 16 disorder realisations side by side, shared update stream
    "ea3d_L256_R16_bitpack": dict(dims=(256, 256, 256), n=1, storage="bitpack", coupling="bond_pm1",
                                  J=(1.0, 1.0, 1.0), beta=1.0 / 1.1, sweeps=1000, replicas=16, replica_streams=0,
                                  record=False),
    # config 4 read literally ("16 independent replicas"): the same lattices with the replica index in the Philox counter
    "ea3d_L256_R16_bitpack_ownstreams": dict(dims=(256, 256, 256), n=1, storage="bitpack", coupling="bond_pm1",
                                             J=(1.0, 1.0, 1.0), beta=1.0 / 1.1, sweeps=1000, replicas=16, replica_streams=1,
                                             record=False),
    # config 5: 3D Heisenberg L = 256, 500 sweeps
    "heisenberg3d_L256_fp32": dict(dims=(256, 256, 256), n=3, storage="fp32", coupling="uniform", J=(1.0, 1.0, 1.0),
                                   beta=0.693, sweeps=500, replicas=1, replica_streams=0, record=False),
    # extra: 3D XY (named by north_star, absent from the configs)
    "xy3d_L256_fp32": dict(dims=(256, 256, 256), n=2, storage="fp32", coupling="uniform", J=(1.0, 1.0, 1.0),
                           beta=0.4542, sweeps=500, replicas=1, replica_streams=0, record=False),
    # extra (SURVEY 8(d) 5''): the paper's own continuous-spin workload, 2D Heisenberg L = 4096 (Table 1)
    "heisenberg2d_L4096_fp32": dict(dims=(4096, 4096, 1), n=3, storage="fp32", coupling="uniform", J=(1.0, 1.0, 1.0),
                                    beta=0.693, sweeps=500, replicas=1, replica_streams=0, record=False),
    # extra: the shape of the paper's fastest Metropolis row (Table 1: 2D +-J, many
    # realisations, multi-spin coded, one random number per site for all realisations); L = 64 is the smallest
    # lattice the bit-packed layout takes (the paper used L = 32)
    "ea2d_L64_R4096_bitpack": dict(dims=(64, 64, 1), n=1, storage="bitpack", coupling="bond_pm1", J=(1.0, 1.0, 1.0),
                                   beta=1.0, sweeps=1000, replicas=4096, replica_streams=0, record=False),
    # SURVEY 8(f) f2 like for like: the paper's own lattice (2D +-J, L = 32, Table 1) in the paper's word layout
    # (one site of 32 realisations per word, SPIN_STORE_MSC), with enough realisations to fill a B200
    "ea2d_L32_R131072_msc": dict(dims=(32, 32, 1), n=1, storage="msc", coupling="bond_pm1", J=(1.0, 1.0, 1.0),
                                 beta=1.0, sweeps=1000, replicas=131072, replica_streams=0, record=False),
}

# Algorithmic bytes moved per attempted update: read the target colour, read the
# other colour once, write the target colour; +-J adds each bond word once per end point and sweep.
BYTES_PER_UPDATE = {
    "ising2d_L64_int8": 3.0,
    "ising2d_L16384_int8": 3.0,
    "ising2d_L16384_bitpack": 0.375,
    "ising3d_L512_bitpack": 0.375,
    "ea3d_L256_R16_bitpack": 1.125,
    "ea3d_L256_R16_bitpack_ownstreams": 1.125,
    "ea2d_L64_R4096_bitpack": 0.875,   # 3 spin bits + 2 forward bonds from each end = 7 bits
    "ea2d_L32_R131072_msc": 0.875,
    "heisenberg3d_L256_fp32": 36.0,
    "heisenberg2d_L4096_fp32": 36.0,
    "xy3d_L256_fp32": 24.0,
}


def n_sites(name):
    d = WORKLOADS[name]["dims"]
    return d[0] * d[1] * d[2]


def scaled(name, dims):
    """The same recipe on a smaller lattice (parity tests)."""
    w = dict(WORKLOADS[name])
    w["dims"] = tuple(dims)
    return w
