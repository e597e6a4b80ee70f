// ising_resident_kernel.cuh -- n = 1, uniform coupling +-1, small lattices: ONE CTA keeps the whole system
// bit-packed in shared memory and runs all n_sweeps sweeps of a spin_sweep / spin_sweep_record call in a single
// launch (the paper keeps a tile in shared memory for k updates; here the "tile" is the entire
// lattice, so the dynamics is the plain k = 1 checkerboard sweep, bit for bit the same as the one-launch-per-
// half-sweep kernels).  BASELINE.json config 1 (64 x 64, E and M after every sweep) is launch-bound otherwise:
// two half-sweep launches plus two measurement launches per sweep.
//
// Work decomposition: thread i owns 32-site word i of BOTH colours (words = R * NW <= 1024); its two words live
// in registers, a copy in shared memory serves the neighbours.  One __syncthreads per half-sweep.  E and M
// are taken from the masks the colour-1 half-sweep has already formed: every bond joins the two
// colours, so E = 2 (#unsatisfied bonds of colour-1 sites) - #bonds and M = N - 2 popcount.
#pragma once
#include "ising_int8_kernel.cuh"
#include "ising_kernels.cuh"

namespace spin {

constexpr int RESIDENT_MAX_WORDS = 1024;

// unsatisfied-bond masks of word gi (replica base rb) of colour `colour` against shared copy `oth` of the other colour
template <int D>
__device__ __forceinline__ void resident_bonds(const uint32_t *oth, uint32_t rb, uint32_t gi, const WordNbrs &n, uint32_t s,
                                               uint32_t av[6]) {
    const uint32_t o = oth[rb + gi], os = oth[rb + n.g_side];
    const uint32_t side = n.p ? ((o >> 1) | (os << 31)) : ((o << 1) | (os >> 31));
    av[0] = s ^ o; av[1] = s ^ side; av[2] = s ^ oth[rb + n.g_ym]; av[3] = s ^ oth[rb + n.g_yp];
    av[4] = 0u; av[5] = 0u;
    if (D == 3) { av[4] = s ^ oth[rb + n.g_zm]; av[5] = s ^ oth[rb + n.g_zp]; }
}

// INT8: the global arrays are the int8 fast layout (ising_int8_kernel.cuh), else bit-packed words.
// d_E / d_M: NULL, or device arrays [n_sweeps][R] that receive E and M after every sweep.
template <int D, bool INT8, bool HB = false>
__global__ void __launch_bounds__(RESIDENT_MAX_WORDS) ising_resident_sweeps(const __grid_constant__ IsingArgs a, uint32_t n_sweeps,
                                                                             double *d_E, double *d_M) {
    __shared__ uint32_t sp[2][RESIDENT_MAX_WORDS];
    __shared__ int acc[2][2][32];   // [sweep parity][unsatisfied, minus spins][replica slot]; R <= 32 when recording
    const uint32_t NW = a.g.NW, words = NW * a.R;
    const uint32_t i = threadIdx.x;
    const bool live = i < words;
    const uint32_t r = live ? i / NW : 0u, gi = live ? i - r * NW : 0u, rb = r * NW;
    const uint32_t rho = a.replica_streams ? r + a.rho_off : 0u;
    const uint32_t jflip = a.jneg ? 0xFFFFFFFFu : 0u;
    WordNbrs nb[2];
    nb[0] = word_neighbours<D>(a.g, 0u, gi);
    nb[1] = word_neighbours<D>(a.g, 1u, gi);
    uint32_t w[2] = {0u, 0u};
    if (live) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            if (INT8) w[c] = int8_pack_unit((const uint8_t *)a.s[c] + (size_t)r * a.g.Nh + 32u * gi);
            else w[c] = ((const uint32_t *)a.s[c])[i];
            sp[c][i] = w[c];
        }
    }
    if (i < 32) { acc[0][0][i] = 0; acc[0][1][i] = 0; acc[1][0][i] = 0; acc[1][1][i] = 0; }
    __syncthreads();
    const bool record = d_E != nullptr;
    const bool warp_one_replica = (NW % 32u) == 0u;   // then all live lanes of a warp share r
    for (uint32_t k = 0; k < n_sweeps; ++k) {
        const uint32_t t = a.t + k;
        int unsat = 0;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            if (live) {
                uint32_t av[6];
                resident_bonds<D>(sp[1 - c], rb, gi, nb[c], w[c] ^ jflip, av);
                const uint32_t fresh = ising_new_word<D, HB>(a, t, (uint32_t)c, gi, rho, w[c], av);
                const uint32_t flip = fresh ^ w[c];
                w[c] = fresh;
                sp[c][i] = w[c];
                if (c == 1 && record) {
                    // after the flip the bond masks of the flipped lanes are inverted
                    unsat = __popc(av[0] ^ flip) + __popc(av[1] ^ flip) + __popc(av[2] ^ flip) + __popc(av[3] ^ flip);
                    if (D == 3) unsat += __popc(av[4] ^ flip) + __popc(av[5] ^ flip);
                }
            }
            if (c == 1 && record) {
                int minus = __popc(w[0]) + __popc(w[1]);
                const uint32_t par = k & 1u;
                if (warp_one_replica) {
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        unsat += __shfl_down_sync(0xFFFFFFFFu, unsat, o);
                        minus += __shfl_down_sync(0xFFFFFFFFu, minus, o);
                    }
                    if ((i & 31u) == 0u && live) { atomicAdd(&acc[par][0][r], unsat); atomicAdd(&acc[par][1][r], minus); }
                } else if (live) {
                    atomicAdd(&acc[par][0][r], unsat);
                    atomicAdd(&acc[par][1][r], minus);
                }
            }
            __syncthreads();
        }
        if (record && i < a.R) {
            // sums of sweep k are complete (barrier above); slot `par` is not touched again before the barrier
            // that ends colour 0 of sweep k + 2, which this thread must reach first
            const uint32_t par = k & 1u;
            const long long nbonds = (long long)D * 64ll * NW;   // d N bonds, N = 64 NW sites
            d_E[(size_t)k * a.R + i] = (double)(2ll * acc[par][0][i] - nbonds);
            d_M[(size_t)k * a.R + i] = (double)(64ll * NW - 2ll * acc[par][1][i]);
            acc[par][0][i] = 0;
            acc[par][1][i] = 0;
        }
    }
    if (live) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            if (INT8) int8_store_unit((uint8_t *)a.s[c] + (size_t)r * a.g.Nh + 32u * gi, w[c]);
            else ((uint32_t *)a.s[c])[i] = w[c];
        }
    }
}

}  // namespace spin

namespace spin {

// ---------------------------------------------------------------------------------------------
// The same kernel with the random masks generated AHEAD of the state (BASELINE config 1: 64 x 64, E and M after every
// sweep).  The lane masks [U < T] of a word depend on (seed, sweep, colour, word) only, not on the spins, so while the
// consumer warps (thread i = word i, as above) apply sweep k, the other warps of the CTA -- up to 30 of them -- build the
// masks of the following sweeps into a double-buffered shared-memory block.  The consumers' half-sweep is then five
// shared-memory loads, the bit-sliced count and one store; the Philox chains (3.45 calls per word, the whole latency of the
// kernel above) run 900-wide beside it.  Decisions are the contract's "U < T" on the same digits: bit-identical.
//   Metropolis: flip = [n_u >= q/2] | ([n_u >= q/2 - 1] & lt_4) | ... | lt_2q  (lt_{k+4} within lt_k), masks lt_masks_full
//   heat bath : new word = ~OR_k (m_k & lt_k) over the 2 D + 1 neighbour counts
constexpr int AHEAD_MAX_WORDS = 256;          // consumer warps: at most 8
constexpr int AHEAD_SMEM_WORDS = 10240;       // 40 KB for the two mask buffers

// MAXT = threads per CTA: 1024 (64 registers per thread, up to 256 words) or 512 (128 registers: no spills in the consumers'
// chain; up to 128 words: config 1 has 64)
template <int D, bool INT8, bool HB, int MAXT = 1024>
__global__ void __launch_bounds__(MAXT) ising_resident_ahead_sweeps(const __grid_constant__ IsingArgs a, uint32_t n_sweeps,
                                                                     double *d_E, double *d_M) {
    constexpr int NT = HB ? 2 * D + 1 : D;
    __shared__ uint32_t sp[2][AHEAD_MAX_WORDS];
    __shared__ uint32_t masks[AHEAD_SMEM_WORDS];   // [buffer][sweep in round][colour][threshold][word]
    __shared__ int acc[2][2][32];
    const uint32_t NW = a.g.NW, words = NW * a.R;
    // Roles.  Warp w issues from sub-core w % 4: the consumer warps are the warps of sub-core 0 (warps 0, 4, 8, ...: word
    // i = 32 (w / 4) + lane), the producers all warps of sub-cores 1 .. 3 (three quarters of the CTA), so that the consumers' short
    // dependent chain never queues behind the Philox chains (measured at 64 x 64, recorded sweeps: 0.64 us with the roles
    // mixed over the sub-cores).
    const uint32_t tid = threadIdx.x, T = blockDim.x, warp = tid >> 5, sub = warp & 3u;
    const uint32_t cthreads = (words + 31u) & ~31u;            // consumer threads (whole warps)
    const uint32_t i = sub == 0u ? ((warp >> 2) << 5) + (tid & 31u) : 0xFFFFFFFFu;   // consumer: the word it owns
    const bool consumer = i < cthreads, live = i < words;
    const bool producer = sub != 0u;
    const uint32_t P = (uint32_t)(MAXT / 128) * 96u, pidx = (((warp >> 2) * 3u + (sub - 1u)) << 5) + (tid & 31u);
    const uint32_t per_sweep = 2u * NT * words;
    const uint32_t DEPTH = min(32u, (uint32_t)AHEAD_SMEM_WORDS / (2u * per_sweep));   // sweeps per round
    const uint32_t r = live ? i / NW : 0u, gi = live ? i - r * NW : 0u, rb = r * NW;
    const uint32_t jflip = a.jneg ? 0xFFFFFFFFu : 0u;
    WordNbrs nb[2];
    nb[0] = word_neighbours<D>(a.g, 0u, gi);
    nb[1] = word_neighbours<D>(a.g, 1u, gi);
    uint32_t w[2] = {0u, 0u};
    if (live) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            if (INT8) w[c] = int8_pack_unit((const uint8_t *)a.s[c] + (size_t)r * a.g.Nh + 32u * gi);
            else w[c] = ((const uint32_t *)a.s[c])[i];
            sp[c][i] = w[c];
        }
    }
    if (tid < 32) { acc[0][0][tid] = 0; acc[0][1][tid] = 0; acc[1][0][tid] = 0; acc[1][1][tid] = 0; }
    // masks of sweeps [k0, k0 + n) into buffer b: one (sweep, colour, word) item per thread and turn; everybody = the
    // first round, when there is nothing to consume yet
    const auto produce = [&](uint32_t b, uint32_t k0, uint32_t n, bool everybody) {
        const uint32_t items = n * 2u * words, step = everybody ? T : P;
        for (uint32_t it = everybody ? tid : pidx; it < items; it += step) {
            const uint32_t ks = it / (2u * words), rem = it - ks * 2u * words, c = rem / words, wi = rem - c * words;
            const uint32_t rr = wi / NW, g2 = wi - rr * NW;
            uint32_t lt[NT];
            lt_masks_full<NT, HB>(a, a.t + k0 + ks, c, g2 + a.g.unit_off, a.replica_streams ? rr + a.rho_off : 0u, lt);
            uint32_t *dst = masks + b * (DEPTH * per_sweep) + ks * per_sweep + c * (NT * words) + wi;
#pragma unroll
            for (int th = 0; th < NT; ++th) dst[th * words] = lt[th];
        }
    };
    const bool record = d_E != nullptr;
    const bool warp_one_replica = (NW % 32u) == 0u;
    produce(0u, 0u, min(DEPTH, n_sweeps), true);
    __syncthreads();
    for (uint32_t k0 = 0, round = 0; k0 < n_sweeps; k0 += DEPTH, ++round) {
        const uint32_t n = min(DEPTH, n_sweeps - k0), b = round & 1u;
        if (!consumer) {
            if (producer && k0 + DEPTH < n_sweeps) produce(b ^ 1u, k0 + DEPTH, min(DEPTH, n_sweeps - k0 - DEPTH), false);
        } else {
            for (uint32_t ks = 0; ks < n; ++ks) {
                const uint32_t k = k0 + ks;
                int unsat = 0;
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    if (live) {
                        uint32_t av[6];
                        resident_bonds<D>(sp[1 - c], rb, gi, nb[c], w[c] ^ jflip, av);
                        const uint32_t *lt = masks + b * (DEPTH * per_sweep) + ks * per_sweep + c * (NT * words) + i;
                        uint32_t fresh;
                        if constexpr (HB) {
                            uint32_t bb[6], m[NT];
#pragma unroll
                            for (int q = 0; q < 6; ++q) bb[q] = q < 2 * D ? av[q] ^ w[c] : 0u;
                            count_masks<D>(bb, m);
                            uint32_t up = 0u;
#pragma unroll
                            for (int q = 0; q < NT; ++q) up |= m[q] & lt[q * words];
                            fresh = ~up;
                        } else if (D == 2) {
                            const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
                            const uint32_t ge2 = c1 | (s1 & av[3]), ge1 = av[0] | av[1] | av[2] | av[3];
                            fresh = w[c] ^ (ge2 | (ge1 & lt[0]) | lt[words]);
                        } else {
                            const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
                            const uint32_t s2 = av[3] ^ av[4] ^ av[5], c2 = maj3(av[3], av[4], av[5]);
                            const uint32_t b0 = s1 ^ s2, c3 = s1 & s2;
                            const uint32_t b1 = c1 ^ c2 ^ c3, b2 = maj3(c1, c2, c3);
                            fresh = w[c] ^ ((b2 | (b1 & b0)) | ((b1 | b2) & lt[0]) | ((b0 | b1 | b2) & lt[words]) | lt[2 * words]);
                        }
                        const uint32_t flip = fresh ^ w[c];
                        w[c] = fresh;
                        sp[c][i] = fresh;
                        if (c == 1 && record) {
                            unsat = __popc(av[0] ^ flip) + __popc(av[1] ^ flip) + __popc(av[2] ^ flip) + __popc(av[3] ^ flip);
                            if (D == 3) unsat += __popc(av[4] ^ flip) + __popc(av[5] ^ flip);
                        }
                    }
                    if (c == 1 && record) {
                        // both sums in one word (unsatisfied bonds of the CTA <= 256 words x 192 < 2^16, minus spins <= 2^14): one
                        // warp reduction instruction (REDUX) and one shared-memory atomic per warp instead of two shuffle trees
                        const int both = unsat + ((__popc(w[0]) + __popc(w[1])) << 16);
                        const uint32_t par = k & 1u;
                        if (warp_one_replica) {
                            const int tot = __reduce_add_sync(0xFFFFFFFFu, live ? both : 0);
                            if ((i & 31u) == 0u && live) atomicAdd(&acc[par][0][r], tot);
                        } else if (live) {
                            atomicAdd(&acc[par][0][r], both);
                        }
                    }
                    asm volatile("bar.sync 1, %0;" ::"r"(cthreads) : "memory");   // the consumer warps only
                }
                if (record && i < a.R) {
                    const uint32_t par = k & 1u;
                    const long long nbonds = (long long)D * 64ll * NW;
                    const int tot = acc[par][0][i];
                    d_E[(size_t)k * a.R + i] = (double)(2ll * (tot & 0xFFFF) - nbonds);
                    d_M[(size_t)k * a.R + i] = (double)(64ll * NW - 2ll * (tot >> 16));
                    acc[par][0][i] = 0;
                }
            }
        }
        __syncthreads();
    }
    if (live) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            if (INT8) int8_store_unit((uint8_t *)a.s[c] + (size_t)r * a.g.Nh + 32u * gi, w[c]);
            else ((uint32_t *)a.s[c])[i] = w[c];
        }
    }
}

}  // namespace spin
