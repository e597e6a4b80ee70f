/*
 * spin_oracle.h -- C interface of the CPU ORACLE.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library.  It
 * shares no code, header, table or constant generator with the CUDA path
 * (paper_1107_5463_b200/csrc); the two only agree on the algorithm written
 * down in DESIGN.md ("The contract").
 *
 * What it computes: the checkerboard single-spin-flip Metropolis sweep for O(n)
 * lattice spin models and the energy / magnetisation sums, exactly as stated in
 *   PAPER.md:31-35  Eq. (1)   H = -sum_<ij> J_ij s_i . s_j, n = 1, 2, 3,
 *                             square / simple-cubic lattice, nearest neighbours
 *   PAPER.md:37-38  Eq. (2)   p_acc = min[1, exp(-beta dE)]
 *   PAPER.md:42               checkerboard decomposition: all spins of one
 *                             sub-lattice, then the other; tabulated Boltzmann
 *                             factors; a random number is drawn for every site
 *   PAPER.md:44               fp32 spins, double-precision aggregates
 *   PAPER.md:46               disorder realisations (replicas) side by side
 * one site at a time, single thread, in the order the paper gives.  Where the
 * paper is silent the readings R-1 ... of DESIGN.md apply (periodic boundaries,
 * k = 1 sweeps, colour 0 first, counter-based Philox-4x32-10, ...).
 *
 * Parity pins: every function below is pinned by tests/test_oracle_*.py (run
 * with -m "not gpu"); see DESIGN.md section "Pins".  Unpinned: equilibrium
 * values of the 3D Heisenberg / XY / +-J models at the BASELINE betas (no
 * closed form) -- "parity unpinned" for those VALUES only; the code path that
 * produces them is pinned through the 1D-chain, beta = 0 and gauge tests.
 */
#ifndef SPIN_ORACLE_H
#define SPIN_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* coupling kinds (values chosen here; the CUDA library has its own enum) */
#define ORACLE_J_UNIFORM 0       /* J[0] on every bond                             */
#define ORACLE_J_PER_DIRECTION 1 /* J[mu] on bonds in direction mu = x, y, z       */
#define ORACLE_J_BOND_PM1 2      /* one +-1 per bond and replica                    */
#define ORACLE_RULE_METROPOLIS 0  /* PAPER.md:37-38 Eq. (2)                            */
#define ORACLE_RULE_HEATBATH 1    /* PAPER.md:40; n = 1 and n = 3                      */
#define ORACLE_INIT_HOT 0
#define ORACLE_INIT_COLD 1

typedef struct oracle_system oracle_system;

/* Philox-4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), as published. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* rand(unit, rho, t, tag) of DESIGN.md: Philox with ctr = (unit, rho, t, tag),
 * key = (seed & 0xffffffff, seed >> 32). */
void oracle_rand(uint64_t seed, uint32_t unit, uint32_t rho, uint32_t t, uint32_t tag, uint32_t out[4]);
/* The random words of the n >= 2 update of one site (compressed same-colour index j): out[0], out[1] feed the proposal
 * (n = 2: out[0] the angle, out[1] the acceptance word; n = 3 Metropolis: out[2] the acceptance word; n = 3 heat bath:
 * out[0] the polar cosine, out[1] the azimuth).  Updates that take two words (n = 2; heat bath) share the call of unit
 * k between sites 2k, 2k + 1 (R-16b).  rule: ORACLE_RULE_METROPOLIS / ORACLE_RULE_HEATBATH. */
void oracle_vector_site_words(uint64_t seed, int n, int rule, uint64_t j, uint32_t rho, uint32_t t, int colour, uint32_t out[4]);

/* n = 1 acceptance uniform of the colour-`colour` site with compressed index j
 * (bit-plane contract, R-16): a 32-bit integer, MSB first digit. */
uint32_t oracle_ising_uniform(uint64_t seed, uint64_t j, uint32_t rho, uint32_t t, int colour);

/* Threshold T(dE) = floor(exp(-beta dE) 2^32), 0 <= T <= 2^32 (PAPER.md:42
 * "pre-tabulation of the Boltzmann factors"). */
uint64_t oracle_threshold(double beta, int dE);

/* Metropolis decision for n = 1: 1 iff dE <= 0 or U < T(dE). */
int oracle_ising_accept(double beta, int dE, uint32_t U);

/* u24(w) and direction(a, b) of DESIGN.md (proposal for n = 2, 3). */
float oracle_u24(uint32_t w);
void oracle_direction3(uint32_t a, uint32_t b, float out[3]);
void oracle_direction2(uint32_t a, float out[2]);
/* Metropolis decision for n >= 2: dE <= 0 or u24(w) < (float)exp((float)beta * -dE). */
int oracle_vector_accept(double beta, float dE, uint32_t w);

/* bonds: host array [replica][mu][i] (mu < d) of +-1, or NULL to draw them from
 * the seed.  Returns NULL on invalid arguments. */
oracle_system *oracle_create(const int32_t dims[3], int32_t n, int32_t coupling_kind, const double J[3],
                             const int8_t *bonds, int32_t n_replicas, int32_t replica_streams, int32_t init,
                             uint64_t seed);
void oracle_destroy(oracle_system *);

/* Local update rule used by oracle_sweep: Metropolis (default) or heat bath.
 * Heat bath: n = 1: s = +1 iff U < T_hb(h), T_hb(h) = floor(2^32 / (1 + exp(-2 beta h))), h = sum_j J s_j;
 * n = 3: cosine about h by inversion, c = 1 + ln(1 - u (1 - e^{-2H})) / H, H = beta |h|, uniform azimuth
 * (details in spin_oracle.cpp).  Returns nonzero for n = 2 (not offered) or a bad rule. */
int oracle_set_update_rule(oracle_system *, int32_t rule);
uint64_t oracle_heatbath_threshold(double beta, int h);
void oracle_heatbath3(double beta, const float h[3], uint32_t w0, uint32_t w1, float out[3]);

/* n_sweeps full sweeps (colour 0 then colour 1) at inverse temperature beta. */
int oracle_sweep(oracle_system *, double beta, int64_t n_sweeps);
/* Same, but also returns, per sweep, how many proposals were accepted. */
int oracle_sweep_count(oracle_system *, double beta, int64_t n_sweeps, int64_t *accepted);
/* Bookkeeping: the sum, over the LAST Metropolis sweep and all replicas, of the energy change dE of
 * every accepted move, as the sweep computed it from its local field.  The update never reads it. */
double oracle_last_sweep_dE(const oracle_system *);

/* E[r] = -sum_bonds J s.s ; M[r*n + a] = sum_i s_i^a. */
int oracle_measure(const oracle_system *, double *E, double *M);

/* canonical layouts: n = 1: int8 [replica][i]; n >= 2: float [replica][i][n];
 * i = x + Lx (y + Ly z). */
int oracle_get_spins(const oracle_system *, void *out, uint64_t bytes);
int oracle_set_spins(oracle_system *, const void *in, uint64_t bytes);
int oracle_get_bonds(const oracle_system *, int8_t *out, uint64_t bytes);
uint64_t oracle_get_sweep_count(const oracle_system *);
void oracle_set_sweep_count(oracle_system *, uint64_t t);

#ifdef __cplusplus
}
#endif
#endif
