// ising_resident_pmj_kernel.cuh -- n = 1, +-J couplings, MANY realisations of a SMALL lattice with a shared update
// stream (R-17; disorder realisations side by side; Table 1's many-realisation workload):
// a CTA keeps a group of G realisations -- spins of both colours and all coupling words -- in shared memory and runs
// ALL n_sweeps sweeps of a spin_sweep call in one launch (the tile stays on chip for k updates; here
// the tile is the whole lattice of each realisation, so the dynamics is the plain checkerboard sweep, bit for bit
// that of ising_bitpack_halfsweep<D, true, true>, or of ising_bitpack_halfsweep_hb<D, true, true> under the heat-bath rule).  One launch per half-sweep leaves such systems launch- and
// latency-bound (4.6 us per half-sweep of 4096 x 64^2 in a CUDA graph, 0.24 of HBM).
//
// Work decomposition: blockDim = NW * RG threads; thread (gi, rg) serves word position gi of the replicas rg,
// rg + RG, ... of the group.  The acceptance masks of a word position do not depend on the state (shared stream: the
// same random numbers for every replica), so a round first builds the masks of RG half-sweeps at once -- thread
// (gi, rg) those of half-sweep h0 + rg -- into shared memory, then applies them half-sweep by half-sweep with one
// __syncthreads each.  Every mask is built once per CTA and used by its G replicas.
#pragma once
#include "ising_kernels.cuh"

namespace spin {

constexpr int RPMJ_THREADS = 512;

// shared-memory words of a CTA: spins [2][G][NW], coupling words [2][G][D][NW], masks [RG][NW][NT] (RG NW = RPMJ_THREADS);
// NT = D thresholds (Metropolis: dE = 4, 8, 12) or 2 D + 1 probabilities (heat bath: 0 .. 2 D neighbour terms equal to -1)
__host__ __device__ inline size_t rpmj_smem_words(uint32_t G, uint32_t NW, int D, bool hb) {
    return (size_t)2 * G * NW * (1 + D) + (size_t)RPMJ_THREADS * (hb ? 2 * D + 1 : D);
}

// one half-sweep of colour C over the replicas rg, rg + RG, ... of the group: word position gi, masks m[NT] of this half-sweep.
// The colour is a template parameter so that the four array bases are fixed offsets and only rr NW moves in the loop.
template <int D, int C, bool HB>
__device__ __forceinline__ void rpmj_half(uint32_t *sp, const uint32_t *bd, const uint32_t *m, const WordNbrs &n, uint32_t jneg,
                                          uint32_t G, uint32_t Gc, uint32_t NW, uint32_t RG, uint32_t gi, uint32_t rg) {
    constexpr int NT = HB ? 2 * D + 1 : D;
    uint32_t ltf[NT];
#pragma unroll
    for (int th = 0; th < NT; ++th) ltf[th] = m[th];
    const uint32_t *other = sp + ((1 - C) * G + rg) * NW;
    uint32_t *mine = sp + (C * G + rg) * NW;
    const uint32_t *bo = bd + ((C * G + rg) * D) * NW;           // own forward bonds
    const uint32_t *bt = bd + (((1 - C) * G + rg) * D) * NW;     // the other colour's
    const uint32_t step = RG * NW, bstep = step * D;
    for (uint32_t rr = rg; rr < Gc; rr += RG, other += step, mine += step, bo += bstep, bt += bstep) {
        // unsatisfied-bond masks exactly as unsatisfied_bonds<D, true> forms them
        const uint32_t raw = mine[gi];
        const uint32_t s = jneg ? ~raw : raw;
        const uint32_t o = other[gi], os = other[n.g_side];
        const uint32_t side = n.p ? ((o >> 1) | (os << 31)) : ((o << 1) | (os >> 31));
        uint32_t av[6];
        av[0] = s ^ o; av[1] = s ^ side; av[2] = s ^ other[n.g_ym]; av[3] = s ^ other[n.g_yp];
        av[4] = 0u; av[5] = 0u;
        if (D == 3) { av[4] = s ^ other[n.g_zm]; av[5] = s ^ other[n.g_zp]; }
        const uint32_t bx_own = bo[gi], bx_oth = bt[gi];
        if (n.p) { av[0] ^= bx_oth; av[1] ^= bx_own; }
        else { av[0] ^= bx_own; av[1] ^= (bx_oth << 1) | (bt[n.g_side] >> 31); }
        av[2] ^= bt[NW + n.g_ym];
        av[3] ^= bo[NW + gi];
        if (D == 3) { av[4] ^= bt[2 * NW + n.g_zm]; av[5] ^= bo[2 * NW + gi]; }
        if (HB) {
            // ising_bitpack_halfsweep_hb<D, true, true>: cnt[k] = lanes with k neighbour terms J s_j equal to -1, new spin +1 iff U < T_hb
            uint32_t b[6], cnt[2 * D + 1];
#pragma unroll
            for (int k = 0; k < 6; ++k) b[k] = k < 2 * D ? av[k] ^ raw : 0u;
            count_masks<D>(b, cnt);
            uint32_t up = 0u;
#pragma unroll
            for (int k = 0; k < 2 * D + 1; ++k) up |= cnt[k] & ltf[k];
            mine[gi] = ~up;
            continue;
        }
        // the flip mask of bitpack_update_word<D, true, true>
        uint32_t flip;
        if (D == 2) {
            const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
            const uint32_t ge2 = c1 | (s1 & av[3]), ge1 = av[0] | av[1] | av[2] | av[3];
            flip = ge2 | (ge1 & ltf[0]) | ltf[1];
        } else {
            const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
            const uint32_t s2 = av[3] ^ av[4] ^ av[5], c2 = maj3(av[3], av[4], av[5]);
            const uint32_t b0 = s1 ^ s2, c3 = s1 & s2;
            const uint32_t b1 = c1 ^ c2 ^ c3, b2 = maj3(c1, c2, c3);
            const uint32_t ge3 = b2 | (b1 & b0);
            flip = ge3 | ((b1 | b2) & ltf[0]) | ((b0 | b1 | b2) & ltf[1]) | ltf[2];
        }
        mine[gi] = raw ^ flip;
    }
}

template <int D, bool HB = false>
__global__ void __launch_bounds__(RPMJ_THREADS) ising_resident_pmj_sweeps(const __grid_constant__ IsingArgs a, uint32_t n_sweeps,
                                                                            uint32_t G) {
    extern __shared__ uint32_t rpmj_smem[];
    constexpr int NT = HB ? 2 * D + 1 : D;
    const uint32_t NW = a.g.NW, RG = blockDim.x / NW;
    const uint32_t gi = threadIdx.x % NW, rg = threadIdx.x / NW;
    const uint32_t r0 = blockIdx.x * G, Gc = min(G, a.R - r0);
    uint32_t *sp = rpmj_smem;                    // [2][G][NW]
    uint32_t *bd = sp + 2 * G * NW;              // [2][G][D][NW]
    uint32_t *mk = bd + 2 * G * D * NW;          // [RG][NW][NT]
    const uint32_t *__restrict__ bb = (const uint32_t *)a.bonds;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        const uint32_t *__restrict__ src = (const uint32_t *)a.s[c] + (size_t)r0 * NW;
        for (uint32_t i = threadIdx.x; i < Gc * NW; i += blockDim.x) sp[c * G * NW + i] = src[i];
        // global coupling words: [colour][R][3][NW]; the first D planes of a replica are contiguous
        for (uint32_t i = threadIdx.x; i < Gc * D * NW; i += blockDim.x) {
            const uint32_t rr = i / (D * NW), rem = i - rr * D * NW;
            bd[(c * G + rr) * D * NW + rem] = bb[((size_t)(c * a.R + r0 + rr) * 3) * NW + rem];
        }
    }
    const WordNbrs nb0 = word_neighbours<D>(a.g, 0u, gi), nb1 = word_neighbours<D>(a.g, 1u, gi);
    __syncthreads();
    const uint32_t HS = 2u * n_sweeps;
    for (uint32_t h0 = 0; h0 < HS; h0 += RG) {
        {
            const uint32_t h = h0 + rg;
            if (h < HS) {
                uint32_t ltf[NT];
                lt_masks_full<NT, HB>(a, a.t + (h >> 1), h & 1u, gi + a.g.unit_off, 0u, ltf);
#pragma unroll
                for (int th = 0; th < NT; ++th) mk[(rg * NW + gi) * NT + th] = ltf[th];
            }
        }
        __syncthreads();
        const uint32_t hn = min(RG, HS - h0);
        for (uint32_t hh = 0; hh < hn; ++hh) {
            const uint32_t *m = mk + (hh * NW + gi) * NT;
            if ((h0 + hh) & 1u) rpmj_half<D, 1, HB>(sp, bd, m, nb1, a.jneg, G, Gc, NW, RG, gi, rg);
            else rpmj_half<D, 0, HB>(sp, bd, m, nb0, a.jneg, G, Gc, NW, RG, gi, rg);
            __syncthreads();
        }
    }
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        uint32_t *dst = (uint32_t *)a.s[c] + (size_t)r0 * NW;
        for (uint32_t i = threadIdx.x; i < Gc * NW; i += blockDim.x) dst[i] = sp[c * G * NW + i];
    }
}

}  // namespace spin
