// ising_msc_kernel.cuh -- n = 1, +-J couplings, MANY disorder realisations with one random number per site for all of
// them: the paper's asynchronous multi-spin coding ("64-bit multi-spin coding ... down to 2 pico-seconds",
// Table 1 row "2D spin glass, Metro. multi-spin").  A 32-bit word holds ONE SITE of 32
// realisations (bit b of group k = realisation 32 k + b; the paper packs 64 into a 64-bit word -- the B200 integer pipes
// are 32 bits wide, so two 32-bit groups are the same work), and because every realisation of a site sees the same uniform
// (shared update stream, R-17) the acceptance masks of a word are all-ones or all-zeros:
//     flip = [n_u >= q/2] | ([n_u >= q/2 - 1] & b_4) | ... | b_2q,     b_k = (U < T(k)) ? ~0 : 0
// with n_u counted bit-sliced over the 32 realisations exactly as in the site-packed kernels.  Any even lattice with
// N / 2 a multiple of 32 is taken -- L = 32 included, which the site-packed layout (Lx % 64 == 0) refuses.
//
// Layout: spins uint32 S_c[G][Nh] (G = R / 32 groups, compressed site index fastest: a warp reads 128 contiguous bytes),
// couplings uint32 B[2 colours][G][d][Nh] (bit = 1: J = -1; forward bond +mu of the site).
// The site's uniform is the one of the contract: site j is lane j & 31 of unit j >> 5, digit k of its
// uniform = bit `lane` of Philox word k.  A warp serves one unit, lane = site: lanes 0 .. 7 hold the eight Philox calls of
// the unit, and every lane assembles ITS 32-bit uniform from bit `lane` of the 32 words (shuffles), then compares as integers.
#pragma once
#include "ising_kernels.cuh"
#include "setup_kernels.cuh"
#include "vector_kernels.cuh"

namespace spin {

// the 32-bit uniform of site (unit, lane) of the Ising update domain; all 32 lanes of the warp must call it
__device__ __forceinline__ uint32_t msc_site_uniform(const IsingArgs &a, uint32_t unit, uint32_t lane) {
    uint32_t w[4];
    philox4x32_10(unit, 0u, a.t, make_tag(a.colour, DOM_ISING_UPDATE, lane & 7u), a.keys, w);   // lane c < 8 holds call c
    uint32_t U = 0u;
#pragma unroll
    for (int d = 0; d < 32; ++d) {
        const uint32_t W = __shfl_sync(0xFFFFFFFFu, w[d & 3], d >> 2);
        U = (U << 1) | ((W >> lane) & 1u);
    }
    return U;
}

// grid = (ceil(Nh / blockDim.x), group chunks); a thread updates site j of the active colour for the groups of its chunk
template <int D, bool HB, bool MEAS = false>
__global__ void __launch_bounds__(128) ising_msc_halfsweep(const __grid_constant__ IsingArgs a) {
    constexpr int NT = HB ? 2 * D + 1 : D;
    const Geometry &g = a.g;
    const uint32_t Nh = g.Nh, G = a.R >> 5;
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;       // Nh % 32 == 0: warps are whole units
    if (j >= Nh) return;
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t U = msc_site_uniform(a, (j + g.j_off) >> 5, lane);
    uint32_t b[NT];
#pragma unroll
    for (int th = 0; th < NT; ++th) {
        const bool lt = HB ? (((a.hb.Talways >> (2 * D - 2 * th + 6)) & 1u) || U < a.hb.T[2 * D - 2 * th + 6])
                           : (((a.tab.Talways >> (4 * (th + 1))) & 1u) || U < a.tab.T[4 * (th + 1)]);
        b[th] = lt ? 0xFFFFFFFFu : 0u;
    }
    uint32_t nb[6];
    neighbour_indices(g, a.colour, j, nb);
    const uint32_t chunk = (G + gridDim.y - 1) / gridDim.y;
    const uint32_t k0 = blockIdx.y * chunk, k1 = min(G, k0 + chunk);
    const uint32_t oc = 1u - a.colour;
    const uint32_t *__restrict__ So = (const uint32_t *)a.s[oc];
    uint32_t *Sc = (uint32_t *)a.s[a.colour];
    const uint32_t *__restrict__ Bo = (const uint32_t *)a.bonds + (size_t)a.colour * G * D * Nh;   // own forward bonds
    const uint32_t *__restrict__ Bt = (const uint32_t *)a.bonds + (size_t)oc * G * D * Nh;         // the other colour's
#pragma unroll 4
    for (uint32_t k = k0; k < k1; ++k) {
        const uint32_t *so = So + (size_t)k * Nh, *bo = Bo + (size_t)k * D * Nh, *bt = Bt + (size_t)k * D * Nh;
        const uint32_t raw = Sc[(size_t)k * Nh + j];
        uint32_t av[6];
        av[0] = raw ^ __ldg(so + nb[0]) ^ __ldg(bt + nb[0]);               // -x: the neighbour owns the bond
        av[1] = raw ^ __ldg(so + nb[1]) ^ __ldg(bo + j);                   // +x: own forward bond
        av[2] = raw ^ __ldg(so + nb[2]) ^ __ldg(bt + Nh + nb[2]);
        av[3] = raw ^ __ldg(so + nb[3]) ^ __ldg(bo + Nh + j);
        av[4] = 0u; av[5] = 0u;
        if (D == 3) {
            av[4] = raw ^ __ldg(so + nb[4]) ^ __ldg(bt + 2 * (size_t)Nh + nb[4]);
            av[5] = raw ^ __ldg(so + nb[5]) ^ __ldg(bo + 2 * (size_t)Nh + j);
        }
        uint32_t fresh;
        if constexpr (HB) {
            uint32_t bb[6], m[NT];
#pragma unroll
            for (int q = 0; q < 6; ++q) bb[q] = q < 2 * D ? av[q] ^ raw : 0u;   // lanes whose neighbour term J s_j is -1
            count_masks<D>(bb, m);
            uint32_t up = 0u;
#pragma unroll
            for (int q = 0; q < NT; ++q) up |= m[q] & b[q];
            fresh = ~up;
        } else if (D == 2) {
            const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
            const uint32_t ge2 = c1 | (s1 & av[3]), ge1 = av[0] | av[1] | av[2] | av[3];
            fresh = raw ^ (ge2 | (ge1 & b[0]) | b[1]);
        } else {
            const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
            const uint32_t s2 = av[3] ^ av[4] ^ av[5], c2 = maj3(av[3], av[4], av[5]);
            const uint32_t b0 = s1 ^ s2, c3 = s1 & s2;
            const uint32_t b1 = c1 ^ c2 ^ c3, b2 = maj3(c1, c2, c3);
            fresh = raw ^ ((b2 | (b1 & b0)) | ((b1 | b2) & b[0]) | ((b0 | b1 | b2) & b[1]) | b[D - 1]);
        }
        Sc[(size_t)k * Nh + j] = fresh;
    }
}

// E and M of every realisation: acc[slot][r][0] += E, [1] += M.  A thread walks a range of sites of colour 1 for one group and
// counts, per realisation bit, the unsatisfied bonds and the minus spins in bit-sliced counters (ripple-carry over PL
// planes), then unpacks them.  Every bond joins the two colours: the 2 d bonds of the colour-1 sites are all bonds.
// grid = (blocks over site ranges, G); E = 2 unsat - d N, M = N - 2 minus.
constexpr int MSC_PLANES = 12;          // a thread counts at most (2^12 - 1) / 6 sites

__device__ __forceinline__ void msc_count(uint32_t c[MSC_PLANES], uint32_t x) {
#pragma unroll
    for (int p = 0; p < MSC_PLANES; ++p) { const uint32_t carry = c[p] & x; c[p] ^= x; x = carry; }
}

template <int D>
__global__ void __launch_bounds__(128) ising_msc_measure(const __grid_constant__ IsingArgs a, uint32_t sites_per_thread) {
    const Geometry &g = a.g;
    const uint32_t Nh = g.Nh, G = a.R >> 5, k = blockIdx.y;
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t j0 = t * sites_per_thread, j1 = min(Nh, j0 + sites_per_thread);
    if (j0 >= Nh) return;
    const uint32_t *__restrict__ S0 = (const uint32_t *)a.s[0] + (size_t)k * Nh, *__restrict__ S1 = (const uint32_t *)a.s[1] + (size_t)k * Nh;
    const uint32_t *__restrict__ B1 = (const uint32_t *)a.bonds + ((size_t)G + k) * D * Nh;   // colour 1's forward bonds
    const uint32_t *__restrict__ B0 = (const uint32_t *)a.bonds + (size_t)k * D * Nh;         // colour 0's
    uint32_t cu[MSC_PLANES], cm[MSC_PLANES];
#pragma unroll
    for (int p = 0; p < MSC_PLANES; ++p) { cu[p] = 0u; cm[p] = 0u; }
    for (uint32_t j = j0; j < j1; ++j) {
        uint32_t nb[6];
        neighbour_indices(g, 1u, j, nb);
        const uint32_t s = S1[j];
        msc_count(cu, s ^ S0[nb[0]] ^ B0[nb[0]]);
        msc_count(cu, s ^ S0[nb[1]] ^ B1[j]);
        msc_count(cu, s ^ S0[nb[2]] ^ B0[Nh + nb[2]]);
        msc_count(cu, s ^ S0[nb[3]] ^ B1[Nh + j]);
        if (D == 3) {
            msc_count(cu, s ^ S0[nb[4]] ^ B0[2 * (size_t)Nh + nb[4]]);
            msc_count(cu, s ^ S0[nb[5]] ^ B1[2 * (size_t)Nh + j]);
        }
        msc_count(cm, s);
        msc_count(cm, S0[j]);
    }
    const long long sites = (long long)(j1 - j0);
    for (uint32_t bit = 0; bit < 32u; ++bit) {
        long long unsat = 0, minus = 0;
#pragma unroll
        for (int p = 0; p < MSC_PLANES; ++p) { unsat += (long long)((cu[p] >> bit) & 1u) << p; minus += (long long)((cm[p] >> bit) & 1u) << p; }
        acc_add(a, 32u * k + bit, 2 * unsat - 2 * D * sites, 2 * sites - 2 * minus);
    }
}

// ------------------------------------------------------------------ setup / canonical conversion (not timed) ---------
// mode 0: cold, 1: hot (seed contract: realisation r, site i as in ising_fill), 2: from canonical int8 [R][N]
__global__ void __launch_bounds__(256) msc_fill(const __grid_constant__ SetupArgs a, int mode, const int8_t *canon, uint32_t *s0, uint32_t *s1,
                                                const int *d_bad = nullptr) {
    const Geometry &g = a.g;
    if (d_bad && *d_bad) return;
    const uint32_t G = a.R >> 5, per_colour = G * g.Nh, total = 2u * per_colour, N = 2u * g.Nh;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour, k = rem / g.Nh, j = rem - k * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        uint32_t word = 0u;
        for (uint32_t bit = 0; bit < 32u && mode != 0; ++bit) {
            const uint32_t r = 32u * k + bit;
            uint32_t v;
            if (mode == 1) {
                uint32_t w[4];
                philox4x32_10(i >> 7, r, 0u, make_tag(0u, DOM_INIT, 0u), a.keys, w);
                v = (w[(i >> 5) & 3u] >> (i & 31u)) & 1u;
            } else {
                v = canon[(size_t)r * N + i] < 0 ? 1u : 0u;
            }
            word |= v << bit;
        }
        (c ? s1 : s0)[(size_t)k * g.Nh + j] = word;
    }
}

__global__ void __launch_bounds__(256) msc_to_canonical(const __grid_constant__ SetupArgs a, const uint32_t *s0, const uint32_t *s1, int8_t *canon) {
    const Geometry &g = a.g;
    const uint32_t G = a.R >> 5, per_colour = G * g.Nh, total = 2u * per_colour, N = 2u * g.Nh;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour, k = rem / g.Nh, j = rem - k * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        const uint32_t word = (c ? s1 : s0)[(size_t)k * g.Nh + j];
        for (uint32_t bit = 0; bit < 32u; ++bit) canon[(size_t)(32u * k + bit) * N + i] = ((word >> bit) & 1u) ? (int8_t)-1 : (int8_t)1;
    }
}

// couplings bb[colour][G][d][Nh] from the seed (canon == NULL; contract of bonds_draw_canonical) or from canonical int8 [R][d][N]
__global__ void __launch_bounds__(256) msc_bonds_pack(const __grid_constant__ SetupArgs a, const int8_t *canon, uint32_t *bb) {
    const Geometry &g = a.g;
    const uint32_t G = a.R >> 5, per_colour = G * g.Nh, total = 2u * per_colour, N = 2u * g.Nh, d = (uint32_t)g.d;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour, k = rem / g.Nh, j = rem - k * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        uint32_t word[3] = {0u, 0u, 0u};
        for (uint32_t bit = 0; bit < 32u; ++bit) {
            const uint32_t r = 32u * k + bit;
            uint32_t w[4] = {0u, 0u, 0u, 0u};
            if (canon == nullptr) philox4x32_10(i >> 5, r, 0u, make_tag(0u, DOM_BONDS, 0u), a.keys, w);
            for (uint32_t mu = 0; mu < d; ++mu) {
                const uint32_t v = canon ? (canon[((size_t)r * d + mu) * N + i] < 0 ? 1u : 0u) : ((w[mu] >> (i & 31u)) & 1u);
                word[mu] |= v << bit;
            }
        }
        for (uint32_t mu = 0; mu < d; ++mu) bb[(((size_t)c * G + k) * d + mu) * g.Nh + j] = word[mu];
    }
}

__global__ void __launch_bounds__(256) msc_bonds_unpack(const __grid_constant__ SetupArgs a, const uint32_t *bb, int8_t *canon) {
    const Geometry &g = a.g;
    const uint32_t G = a.R >> 5, per_colour = G * g.Nh, total = 2u * per_colour, N = 2u * g.Nh, d = (uint32_t)g.d;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour, k = rem / g.Nh, j = rem - k * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        for (uint32_t mu = 0; mu < d; ++mu) {
            const uint32_t word = bb[(((size_t)c * G + k) * d + mu) * g.Nh + j];
            for (uint32_t bit = 0; bit < 32u; ++bit)
                canon[((size_t)(32u * k + bit) * d + mu) * N + i] = ((word >> bit) & 1u) ? (int8_t)-1 : (int8_t)1;
        }
    }
}

}  // namespace spin
