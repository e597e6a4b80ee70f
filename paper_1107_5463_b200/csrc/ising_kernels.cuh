// ising_kernels.cuh -- n = 1 half-sweep kernels (Eq. (2), PAPER.md:42 checkerboard,
// PAPER.md:46 / 52 replicas and multi-spin coding).  Three kernels share one decision rule:
//   ising_generic_halfsweep  one thread per site, any even dims, any coupling kind  (reference shape)
//   ising_bitpack_halfsweep  one thread per 32-site word, bitwise local field and acceptance
//   ising_int8_halfsweep     one thread per 32 sites stored as bytes, SIMD-in-register byte arithmetic
// All implement: flip iff dE <= 0 or U < T(dE), U the site's bit-plane uniform (common.cuh).
#pragma once
#include "common.cuh"

namespace spin {

struct IsingArgs {
    Geometry g;
    PhiloxKeys keys;
    IsingTable tab;
    void *s[2];          // per colour: int8 -> uint8_t [R][Nh] (0 = +1, 1 = -1); bitpack -> uint32_t [R][NW]
    const void *bonds;   // bitpack: uint32_t [2][R][3][NW] (bit = 1: J = -1); generic: int8 [R][d][N] of +-1
    uint32_t R, replica_streams, t, colour;
    uint32_t rho_off;       // added to the replica index in the Philox counter (temperature axis: one launch per replica, R = 1)
    int32_t coupling_kind;  // 0 uniform, 1 per direction, 2 per bond
    int32_t Jdir[3];        // generic kernel: coupling per direction in {-1, 0, +1}
    uint32_t jneg;          // fast kernels: 1 iff the uniform coupling is -1
    uint32_t rule;          // 0 Metropolis (Eq. (2)), 1 heat bath
    long long *acc;         // [acc_slots][R][2] energy / magnetisation accumulators (measurement kernels and fused measurement)
    uint32_t acc_slots;     // power of two: a CTA adds into slot blockIdx.x & (acc_slots - 1), so that atomics on one address
                            // do not serialise (65 536 of them per launch on two addresses cost 18 us); the finalize sums the slots
    HeatBathTable hb;       // filled when rule = 1
    void *alt[2];           // temporal blocking (ising_tblock_kernel.cuh): the second pair of colour arrays it writes to
    uint32_t tb_rows;       // temporal blocking: rows per stripe
    uint32_t l2_keep;       // +-J quad kernel: replicas whose coupling words are loaded "evict_last" (0xFFFFFFFF: no L2 hints)
    uint32_t defer_cap;     // deferred digit comparison: queue entries per warp in use (<= DEFER_CAP; SPIN_OPT_DEFER_CAP)
    uint32_t prefetch;      // L2 prefetch distance (0 = off): replicas ahead (+-J quad kernel) / CTAs ahead (strip kernels)
};

// digit dg / "always" mask of threshold th of the table in use: HB = false -> Metropolis factors T(4 (th + 1)),
// HB = true -> heat-bath probabilities of k = th neighbour terms equal to -1
template <bool HB>
__device__ __forceinline__ uint32_t tab_digit(const IsingArgs &a, int th, int dg) {
    if constexpr (HB) return a.hb.digit[th][dg]; else return a.tab.digit[th < 3 ? th : 0][dg];
}
template <bool HB>
__device__ __forceinline__ uint32_t tab_always(const IsingArgs &a, int th) {
    if constexpr (HB) return a.hb.always[th]; else return a.tab.always[th < 3 ? th : 0];
}

// ------------------------------------------------------------------ bit-serial U < T ---------
// Lane masks of U < T(4 (th + 1)) for th < NT, for all 32 lanes of `unit`.  Digits are consumed most
// significant first, four per Philox call, until every lane is decided for every threshold
// (about log2(32) + 1.3 digits on average; a warp runs until its slowest thread is done).
template <int NT, bool HB = false>
__device__ __forceinline__ void lt_masks_full(const IsingArgs &a, uint32_t t, uint32_t colour, uint32_t unit, uint32_t rho,
                                              uint32_t lt[NT]) {
    uint32_t eq[NT];
#pragma unroll
    for (int th = 0; th < NT; ++th) { lt[th] = tab_always<HB>(a, th); eq[th] = ~tab_always<HB>(a, th); }
#pragma unroll
    for (int call = 0; call < 8; ++call) {
        uint32_t any = eq[0];
#pragma unroll
        for (int th = 1; th < NT; ++th) any |= eq[th];
        if (any == 0u) break;
        uint32_t w[4];
        philox4x32_10(unit, rho, t, make_tag(colour, DOM_ISING_UPDATE, call), a.keys, w);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
#pragma unroll
            for (int th = 0; th < NT; ++th) {
                const uint32_t tb = tab_digit<HB>(a, th, 4 * call + k);
                lt[th] |= eq[th] & ~w[k] & tb;
                eq[th] &= ~(w[k] ^ tb);
            }
        }
    }
}

// The same comparison when every lane needs only ONE threshold: m[th] are disjoint lane masks
// (lane in m[th] compares against T(4 (th + 1)); lanes in none are not compared).  Returns the
// mask of lanes with U < their threshold.
template <int NT, bool HB = false>
__device__ __forceinline__ uint32_t lt_mask_select(const IsingArgs &a, uint32_t t, uint32_t colour, uint32_t unit, uint32_t rho,
                                                   const uint32_t m[NT]) {
    uint32_t lt = 0u, eq = 0u;
#pragma unroll
    for (int th = 0; th < NT; ++th) { lt |= m[th] & tab_always<HB>(a, th); eq |= m[th] & ~tab_always<HB>(a, th); }
#pragma unroll
    for (int call = 0; call < 8; ++call) {
        if (eq == 0u) break;
        uint32_t w[4];
        philox4x32_10(unit, rho, t, make_tag(colour, DOM_ISING_UPDATE, call), a.keys, w);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int dg = 4 * call + k;
            uint32_t tk = tab_digit<HB>(a, NT - 1, dg);
#pragma unroll
            for (int th = NT - 2; th >= 0; --th) tk = (m[th] & tab_digit<HB>(a, th, dg)) | (~m[th] & tk);
            lt |= eq & ~w[k] & tk;
            eq &= ~(w[k] ^ tk);
        }
    }
    return lt;
}

// ------------------------------------------------------------------ deferred tail of U < T ----
// A warp that runs the lazy digit loop above pays for its slowest thread: 3.45 Philox calls per warp against 2.25 per
// thread (profiles/r01d).  The strip kernels therefore split the comparison: DEFER_CALLS calls are made unconditionally
// by every thread (no divergence, the calls interleave), and a unit that still has undecided lanes afterwards (about one
// in ten) is pushed into a per-warp shared-memory queue; after its strip the warp drains the queue with one pending unit
// per lane, so the tail calls run with all lanes busy.  The contract (R-16) is unchanged: every lane's
// decision is still "U < T" on the same digits.
constexpr int DEFER_CALLS = 2;
constexpr int DEFER_CAP = 32;          // queue entries per warp; a thread that finds it full finishes its unit itself
constexpr int DEFER_FIELDS = 6;        // unit, rho, eq, m[0], m[1], provisional word; + the word's index in its array
struct DeferQueue {
    uint32_t n[4];
    uint32_t f[4][DEFER_FIELDS + 1][DEFER_CAP];
};
// the same for the heat-bath rule: 2 D masks (the last of the 2 D + 1 classes is the default), unit, rho, eq, word, index
template <int D>
struct DeferQueueHB {
    uint32_t n[4];
    uint32_t f[4][2 * D + 5][DEFER_CAP];
};

// digit k of the threshold each lane compares against: lanes of m[th] use T(4 (th + 1)), the rest the last one
// (HB: the heat-bath table, NT = 2 D + 1 masks by the number of neighbour terms equal to -1)
template <int NT, bool HB = false>
__device__ __forceinline__ uint32_t select_digit(const IsingArgs &a, const uint32_t m[NT], int dg) {
    uint32_t tk = tab_digit<HB>(a, NT - 1, dg);
#pragma unroll
    for (int th = NT - 2; th >= 0; --th) tk = (m[th] & tab_digit<HB>(a, th, dg)) | (~m[th] & tk);
    return tk;
}

// calls [0, DEFER_CALLS) of the comparison, unconditionally; returns lt, leaves the undecided lanes in eq
template <int NT, bool HB = false>
__device__ __forceinline__ uint32_t lt_mask_select_head(const IsingArgs &a, uint32_t t, uint32_t colour, uint32_t unit, uint32_t rho,
                                                        const uint32_t m[NT], uint32_t &eq_out) {
    uint32_t lt = 0u, eq = 0u;
#pragma unroll
    for (int th = 0; th < NT; ++th) { lt |= m[th] & tab_always<HB>(a, th); eq |= m[th] & ~tab_always<HB>(a, th); }
#pragma unroll
    for (int call = 0; call < DEFER_CALLS; ++call) {
        uint32_t w[4];
        philox4x32_10(unit, rho, t, make_tag(colour, DOM_ISING_UPDATE, call), a.keys, w);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t tk = select_digit<NT, HB>(a, m, 4 * call + k);
            lt |= eq & ~w[k] & tk;
            eq &= ~(w[k] ^ tk);
        }
    }
    eq_out = eq;
    return lt;
}

// calls [DEFER_CALLS, 8) for the lanes still in eq, lazily; returns the lanes that turn out to have U < T
template <int NT, bool HB = false>
__device__ __forceinline__ uint32_t lt_mask_select_tail(const IsingArgs &a, uint32_t t, uint32_t colour, uint32_t unit, uint32_t rho,
                                                        const uint32_t m[NT], uint32_t eq) {
    uint32_t lt = 0u;
    for (int call = DEFER_CALLS; call < 8; ++call) {
        if (eq == 0u) break;
        uint32_t w[4];
        philox4x32_10(unit, rho, t, make_tag(colour, DOM_ISING_UPDATE, call), a.keys, w);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t tk = select_digit<NT, HB>(a, m, 4 * call + k);
            lt |= eq & ~w[k] & tk;
            eq &= ~(w[k] ^ tk);
        }
    }
    return lt;
}

__device__ __forceinline__ uint32_t maj3(uint32_t x, uint32_t y, uint32_t z) { return (x & y) | (z & (x | y)); }

// Fused measurement: every bond joins the two colours, so the colour-1 half-sweep
// has, in the masks it formed anyway, everything E and M need.  Per 32-site word of colour 1 after its update:
// E += 2 (#unsatisfied bonds) - (#bonds), M += 64 - 2 (minus spins of this word and of the colour-0 word at the same
// index).  Lanes of a warp that serve the same replica are summed with one warp reduction, then one atomic each.
template <int D>
__device__ __forceinline__ void fused_word_sums(const uint32_t av[6], uint32_t raw, uint32_t fresh, uint32_t o_same, int &e, int &m) {
    const uint32_t flip = raw ^ fresh;   // a flipped lane inverts all its bond masks
    int unsat = __popc(av[0] ^ flip) + __popc(av[1] ^ flip) + __popc(av[2] ^ flip) + __popc(av[3] ^ flip);
    if (D == 3) unsat += __popc(av[4] ^ flip) + __popc(av[5] ^ flip);
    e += 2 * unsat - 2 * D * 32;
    m += 64 - 2 * (__popc(fresh) + __popc(o_same));
}
// the accumulator pair of replica r this CTA adds into
__device__ __forceinline__ unsigned long long *acc_slot(const IsingArgs &a, uint32_t r) {
    return (unsigned long long *)a.acc + 2 * ((size_t)(blockIdx.x & (a.acc_slots - 1u)) * a.R + r);
}
__device__ __forceinline__ void acc_add(const IsingArgs &a, uint32_t r, long long e, long long m) {
    unsigned long long *p = acc_slot(a, r);
    atomicAdd(p, (unsigned long long)e);
    atomicAdd(p + 1, (unsigned long long)m);
}
__device__ __forceinline__ void fused_commit(const IsingArgs &a, uint32_t r, int e, int m) {
    const unsigned active = __activemask();
    const unsigned peers = __match_any_sync(active, r);
    const int es = __reduce_add_sync(peers, e), ms = __reduce_add_sync(peers, m);
    if ((threadIdx.x & 31u) == (uint32_t)(__ffs(peers) - 1)) acc_add(a, r, es, ms);
}

// m[k] = lanes in which exactly k of the 2 D masks b[] are set (k = 0 .. 2 D), bit-sliced with full adders
template <int D>
__device__ __forceinline__ void count_masks(const uint32_t b[6], uint32_t m[2 * D + 1]) {
    if (D == 2) {
        const uint32_t s1 = b[0] ^ b[1] ^ b[2], c1 = maj3(b[0], b[1], b[2]);
        const uint32_t b0 = s1 ^ b[3], c2 = s1 & b[3];
        const uint32_t b1 = c1 ^ c2, b2 = c1 & c2;
        m[0] = ~(b0 | b1 | b2); m[1] = b0 & ~b1; m[2] = b1 & ~b0; m[3] = b0 & b1; m[4] = b2;
    } else {
        const uint32_t s1 = b[0] ^ b[1] ^ b[2], c1 = maj3(b[0], b[1], b[2]);
        const uint32_t s2 = b[3] ^ b[4] ^ b[5], c2 = maj3(b[3], b[4], b[5]);
        const uint32_t b0 = s1 ^ s2, c3 = s1 & s2;
        const uint32_t b1 = c1 ^ c2 ^ c3, b2 = maj3(c1, c2, c3);
        m[0] = ~(b0 | b1 | b2); m[1] = b0 & ~b1 & ~b2; m[2] = b1 & ~b0 & ~b2; m[3] = b0 & b1;
        m[4] = b2 & ~b0 & ~b1; m[5] = b2 & b0; m[6] = b2 & b1;
    }
}

// ------------------------------------------------------------------ generic kernel -----------
// One thread per (replica, site of the active colour).  Handles size-2 dimensions (the -mu and +mu
// neighbour coincide and both bonds count), zero couplings and per-bond couplings.
__global__ void __launch_bounds__(256) ising_generic_halfsweep(const __grid_constant__ IsingArgs a) {
    const Geometry &g = a.g;
    const uint32_t total = g.sw_jn * a.R;
    const uint8_t *__restrict__ other_base = (const uint8_t *)a.s[1 - a.colour];
    uint8_t *mine_base = (uint8_t *)a.s[a.colour];
    const uint32_t N = 2u * g.Nh;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t r = idx / g.sw_jn, j = g.sw_j0 + idx - r * g.sw_jn;
        const uint32_t row = fdiv(j, g.divRL), xh = j - row * g.RL;
        const uint32_t z = fdiv(row, g.divLy), y = row - z * (uint32_t)g.Ly;
        const uint32_t p = (y + z + a.colour) & 1u;
        const uint32_t x = 2u * xh + p;
        const uint8_t *other = other_base + (size_t)r * g.Nh;
        // neighbour coordinates (periodic)
        const uint32_t xm = x == 0 ? g.Lx - 1 : x - 1, xp = x == (uint32_t)g.Lx - 1 ? 0 : x + 1;
        const uint32_t ym = y == 0 ? g.Ly - 1 : y - 1, yp = y == (uint32_t)g.Ly - 1 ? 0 : y + 1;
        const uint32_t zm = z == 0 ? g.Lz - 1 : z - 1, zp = z == (uint32_t)g.Lz - 1 ? 0 : z + 1;
        const uint32_t rowbase = row * g.RL;
        int nb[6];
        uint32_t isite[6];  // lexicographic index of the site that owns the connecting forward bond
        nb[0] = other[rowbase + (xm >> 1)];                         isite[0] = xm + g.Lx * row;
        nb[1] = other[rowbase + (xp >> 1)];                         isite[1] = x + g.Lx * row;
        nb[2] = other[(ym + g.Ly * z) * g.RL + xh];                 isite[2] = x + g.Lx * (ym + g.Ly * z);
        nb[3] = other[(yp + g.Ly * z) * g.RL + xh];                 isite[3] = x + g.Lx * row;
        if (g.d == 3) {
            nb[4] = other[(y + g.Ly * zm) * g.RL + xh];             isite[4] = x + g.Lx * (y + g.Ly * zm);
            nb[5] = other[(y + g.Ly * zp) * g.RL + xh];             isite[5] = x + g.Lx * row;
        }
        const int s = 1 - 2 * (int)mine_base[(size_t)r * g.Nh + j];
        int h = 0;
        const int8_t *bonds = (const int8_t *)a.bonds;
        for (int k = 0; k < 2 * g.d; ++k) {
            const int mu = k >> 1;
            int J;
            if (a.coupling_kind == 2) J = bonds[((size_t)r * g.d + mu) * N + isite[k]];
            else J = a.Jdir[mu];
            h += J * (1 - 2 * nb[k]);
        }
        const int dE = 2 * s * h;
        // Metropolis: flip iff dE <= 0 or U < T(dE).  Heat bath: s' = +1 iff U < T_hb(h); `flip` then means "U < T_hb"
        const bool hb = a.rule != 0u;
        bool flip = hb ? ((a.hb.Talways >> (h + 6)) & 1u) != 0u : (dE <= 0 || ((a.tab.Talways >> dE) & 1u));
        if (!flip) {
            const uint32_t T = hb ? a.hb.T[h + 6] : a.tab.T[dE];
            const uint32_t jg = j + g.j_off;   // global compressed index (slab decomposition)
            const uint32_t unit = jg >> 5, lane = jg & 31u;
            const uint32_t rho = a.replica_streams ? r + a.rho_off : 0u;
            bool decided = false;
            for (int call = 0; call < 8 && !decided; ++call) {
                uint32_t w[4];
                philox4x32_10(unit, rho, a.t, make_tag(a.colour, DOM_ISING_UPDATE, call), a.keys, w);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    if (decided) continue;
                    const uint32_t ud = (w[k] >> lane) & 1u, td = (T >> (31 - (4 * call + k))) & 1u;
                    if (ud != td) { decided = true; flip = ud < td; }
                }
            }
        }
        if (hb) mine_base[(size_t)r * g.Nh + j] = (uint8_t)(flip ? 0 : 1);
        else if (flip) mine_base[(size_t)r * g.Nh + j] = (uint8_t)(s > 0 ? 1 : 0);
    }
}

// ------------------------------------------------------------------ bit-packed kernel --------
// Word indices of the neighbours of 32-site word gi = w + WX (y + Ly z) of colour `colour`.
struct WordNbrs {
    uint32_t p, g_side, g_ym, g_yp, g_zm, g_zp;
};
template <int D>
__device__ __forceinline__ WordNbrs word_neighbours(const Geometry &g, uint32_t colour, uint32_t gi) {
    WordNbrs n;
    const uint32_t WX = g.WX;
    const uint32_t row = fdiv(gi, g.divWX), w = gi - row * WX;
    const uint32_t z = fdiv(row, g.divLy), y = row - z * (uint32_t)g.Ly;
    n.p = (y + z + colour) & 1u;
    const uint32_t wside = n.p ? (w + 1 == WX ? 0 : w + 1) : (w == 0 ? WX - 1 : w - 1);
    n.g_side = row * WX + wside;
    n.g_ym = y == 0 ? gi + WX * (g.Ly - 1) : gi - WX;
    n.g_yp = y == (uint32_t)g.Ly - 1 ? gi - WX * (g.Ly - 1) : gi + WX;
    n.g_zm = gi;
    n.g_zp = gi;
    if (D == 3) {
        const uint32_t plane = WX * g.Ly;
        n.g_zm = z == 0 ? gi + plane * (g.Lz - 1) : gi - plane;
        n.g_zp = z == (uint32_t)g.Lz - 1 ? gi - plane * (g.Lz - 1) : gi + plane;
    }
    return n;
}

// av[k] = lane mask of unsatisfied bonds (s_i ^ s_j ^ [J < 0]) of word gi of colour `colour`, replica r,
// towards its 2 D neighbours; bit = 1 means spin -1 / coupling -1.  Returns the word's own spins.
template <int D, bool BONDS>
__device__ __forceinline__ uint32_t unsatisfied_bonds(const IsingArgs &a, uint32_t colour, uint32_t r, uint32_t gi,
                                                      const WordNbrs &n, uint32_t av[6]) {
    const uint32_t NW = a.g.NW;
    const uint32_t *__restrict__ other = (const uint32_t *)a.s[1 - colour] + (size_t)r * NW;
    const uint32_t raw = ((const uint32_t *)a.s[colour])[(size_t)r * NW + gi];  // plain load: this array is written by the kernel
    const uint32_t s = a.jneg ? ~raw : raw;
    const uint32_t o = other[gi], os = other[n.g_side];
    const uint32_t side = n.p ? ((o >> 1) | (os << 31)) : ((o << 1) | (os >> 31));
    av[0] = s ^ o; av[1] = s ^ side; av[2] = s ^ other[n.g_ym]; av[3] = s ^ other[n.g_yp];
    av[4] = 0u; av[5] = 0u;
    if (D == 3) { av[4] = s ^ other[n.g_zm]; av[5] = s ^ other[n.g_zp]; }
    if (BONDS) {
        const uint32_t *__restrict__ bb = (const uint32_t *)a.bonds;
        const uint32_t *__restrict__ bo = bb + ((size_t)(colour * a.R + r) * 3) * NW;        // own forward bonds
        const uint32_t *__restrict__ bt = bb + ((size_t)((1 - colour) * a.R + r) * 3) * NW;  // other colour's
        const uint32_t bx_own = bo[gi], bx_oth = bt[gi];
        if (n.p) { av[0] ^= bx_oth; av[1] ^= bx_own; }
        else { av[0] ^= bx_own; av[1] ^= (bx_oth << 1) | (bt[n.g_side] >> 31); }
        av[2] ^= bt[(size_t)NW + n.g_ym];
        av[3] ^= bo[(size_t)NW + gi];
        if (D == 3) { av[4] ^= bt[2 * (size_t)NW + n.g_zm]; av[5] ^= bo[2 * (size_t)NW + gi]; }
    }
    return raw;
}

// new value of word gi of replica r (see ising_bitpack_halfsweep)
template <int D, bool BONDS, bool SHARED, bool MEAS = false>
__device__ __forceinline__ uint32_t bitpack_update_word(const IsingArgs &a, uint32_t r, uint32_t gi, const WordNbrs &n,
                                                        const uint32_t ltf[D], int *e_sum = nullptr, int *m_sum = nullptr) {
    uint32_t av[6];
    const uint32_t raw = unsatisfied_bonds<D, BONDS>(a, a.colour, r, gi, n, av);
    [[maybe_unused]] const auto finish = [&](uint32_t flip) {
        if (MEAS) fused_word_sums<D>(av, raw, raw ^ flip, ((const uint32_t *)a.s[1 - a.colour])[(size_t)r * a.g.NW + gi], *e_sum, *m_sum);
        return raw ^ flip;
    };
    uint32_t flip;
    if (D == 2) {
        const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
        const uint32_t ge2 = c1 | (s1 & av[3]), ge1 = av[0] | av[1] | av[2] | av[3];
        if (SHARED) flip = ge2 | (ge1 & ltf[0]) | ltf[1];
        else {
            const uint32_t m[2] = {ge1 & ~ge2, ~ge1};
            flip = ge2 | lt_mask_select<2>(a, a.t, a.colour, gi + a.g.unit_off, a.replica_streams ? r + a.rho_off : 0u, m);
        }
    } else {
        const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
        const uint32_t s2 = av[3] ^ av[4] ^ av[5], c2 = maj3(av[3], av[4], av[5]);
        const uint32_t b0 = s1 ^ s2, c3 = s1 & s2;
        const uint32_t b1 = c1 ^ c2 ^ c3, b2 = maj3(c1, c2, c3);
        const uint32_t ge3 = b2 | (b1 & b0);
        if (SHARED) flip = ge3 | ((b1 | b2) & ltf[0]) | ((b0 | b1 | b2) & ltf[1]) | ltf[2];
        else {
            const uint32_t m[3] = {b1 & ~b0 & ~b2, b0 & ~b1 & ~b2, ~(b0 | b1 | b2)};
            flip = ge3 | lt_mask_select<3>(a, a.t, a.colour, gi + a.g.unit_off, a.replica_streams ? r + a.rho_off : 0u, m);
        }
    }
    return finish(flip);
}

// One thread per 32-site word of the active colour; loops over the replicas.  dE = 2q - 4 n_u with n_u
// the number of unsatisfied bonds, counted bit-sliced with full adders.  SHARED: all replicas see
// the same random numbers (R > 1, replica_streams = 0), so the masks are built once per word and
// reused R times (batching four replicas' loads per thread was measured slower: 58 vs 40 us); otherwise each lane is compared against the one
// threshold it needs.
// MEAS: the colour-1 half-sweep of a recorded sweep also accumulates E and M into a.acc (fused_word_sums).
template <int D, bool BONDS, bool SHARED, bool MEAS = false>
__global__ void __launch_bounds__(256) ising_bitpack_halfsweep(const __grid_constant__ IsingArgs a) {
    constexpr int NT = D;  // thresholds: dE = 4, 8 (2D) and 12 (3D)
    const uint32_t NW = a.g.NW, gi_end = (a.g.sw_j0 + a.g.sw_jn) >> 5;
    uint32_t *mine_base = (uint32_t *)a.s[a.colour];
    for (uint32_t gi = (a.g.sw_j0 >> 5) + blockIdx.x * blockDim.x + threadIdx.x; gi < gi_end; gi += gridDim.x * blockDim.x) {
        const WordNbrs n = word_neighbours<D>(a.g, a.colour, gi);
        const bool owned = gi >= (a.g.own_j0 >> 5) && gi < (a.g.own_j1 >> 5);
        uint32_t ltf[NT];
        uint32_t r0 = 0u, r1 = a.R;
        if (SHARED) {
            // gridDim.y > 1: the replicas are split into gridDim.y chunks (many realisations of a small lattice)
            const uint32_t chunk = (a.R + gridDim.y - 1) / gridDim.y;
            r0 = blockIdx.y * chunk; r1 = min(a.R, r0 + chunk);
            lt_masks_full<NT>(a, a.t, a.colour, gi + a.g.unit_off, 0u, ltf);
        }
        for (uint32_t r = r0; r < r1; ++r) {
            int e = 0, m = 0;
            mine_base[(size_t)r * NW + gi] = bitpack_update_word<D, BONDS, SHARED, MEAS>(a, r, gi, n, ltf, &e, &m);
            if (MEAS && owned) {
                // every lane of the warp that is in this loop serves replica r: one reduction, one atomic pair
                const unsigned act = __activemask();
                const int es = __reduce_add_sync(act, e), ms = __reduce_add_sync(act, m);
                if ((threadIdx.x & 31u) == (uint32_t)(__ffs(act) - 1)) acc_add(a, r, es, ms);
            }
        }
    }
}

// Heat-bath version of ising_bitpack_halfsweep: av[k] ^ raw = lanes whose neighbour term J s_j is -1;
// with k of them the local field is h = 2 D - 2 k and the new spin is +1 iff U < T_hb(h) (HeatBathTable).
// SHARED: the 2 D + 1 masks U < T_hb are built once per word and reused by every replica.
template <int D, bool BONDS, bool SHARED>
__global__ void __launch_bounds__(256) ising_bitpack_halfsweep_hb(const __grid_constant__ IsingArgs a) {
    constexpr int NT = 2 * D + 1;
    const uint32_t NW = a.g.NW, gi_end = (a.g.sw_j0 + a.g.sw_jn) >> 5;
    uint32_t *mine_base = (uint32_t *)a.s[a.colour];
    for (uint32_t gi = (a.g.sw_j0 >> 5) + blockIdx.x * blockDim.x + threadIdx.x; gi < gi_end; gi += gridDim.x * blockDim.x) {
        const WordNbrs n = word_neighbours<D>(a.g, a.colour, gi);
        uint32_t ltf[NT];
        if (SHARED) lt_masks_full<NT, true>(a, a.t, a.colour, gi + a.g.unit_off, 0u, ltf);
        const uint32_t chunk = SHARED ? (a.R + gridDim.y - 1) / gridDim.y : a.R;
        const uint32_t r0 = SHARED ? blockIdx.y * chunk : 0u, r1 = min(a.R, r0 + chunk);
        for (uint32_t r = r0; r < r1; ++r) {
            uint32_t av[6], b[6], m[NT];
            const uint32_t raw = unsatisfied_bonds<D, BONDS>(a, a.colour, r, gi, n, av);
#pragma unroll
            for (int k = 0; k < 6; ++k) b[k] = k < 2 * D ? av[k] ^ raw : 0u;
            count_masks<D>(b, m);
            uint32_t up;   // lanes whose new spin is +1
            if (SHARED) {
                up = 0u;
#pragma unroll
                for (int k = 0; k < NT; ++k) up |= m[k] & ltf[k];
            } else {
                up = lt_mask_select<NT, true>(a, a.t, a.colour, gi + a.g.unit_off, a.replica_streams ? r + a.rho_off : 0u, m);
            }
            mine_base[(size_t)r * NW + gi] = ~up;
        }
    }
}

// ------------------------------------------------------------------ +-J, shared stream, one thread per quad of words ----
// Lx % 256 == 0: a row of one colour is a whole number of quads of four 32-site words, and a quad is one aligned 128-bit
// access in the spin arrays and in every coupling plane.  One thread updates a quad for all replicas of its chunk:
// 8 (d = 2) or 12 (d = 3) 128-bit loads and one 128-bit store per replica, plus, when the row is longer than one quad,
// two scalar loads for the x-neighbour word (and its coupling word) in the adjacent quad.  At Lx = 256 (BASELINE
// config 4) the row is the quad and the periodic x-neighbour of every word is inside it: no scalar loads at all.
__device__ __forceinline__ uint32_t u4c(const uint4 &v, int i) { return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w)); }

// geometry of one quad (uint4 index `me` inside one replica's array) of the active colour
struct QuadGeom {
    uint32_t me, p, q_ym, q_yp, q_zm, q_zp, w_edge, QX, NW4;
};
template <int D>
__device__ __forceinline__ QuadGeom quad_geometry(const IsingArgs &a, uint32_t item) {
    const Geometry &g = a.g;
    const uint32_t Ly = (uint32_t)g.Ly, Lz = (uint32_t)g.Lz, QX = g.WX >> 2;
    QuadGeom k;
    const uint32_t row = QX == 1u ? item : fdiv(item, g.divQW), q = item - row * QX;
    const uint32_t z = fdiv(row, g.divLy), y = row - z * Ly;
    k.p = (y + z + a.colour) & 1u;
    k.me = item; k.QX = QX; k.NW4 = g.NW >> 2;   // uint4 per (replica, plane)
    // uint4 indices of the quads at y -+ 1, z -+ 1
    k.q_ym = y == 0 ? item + QX * (Ly - 1) : item - QX; k.q_yp = y == Ly - 1 ? item - QX * (Ly - 1) : item + QX;
    k.q_zm = D == 3 ? (z == 0 ? item + QX * Ly * (Lz - 1) : item - QX * Ly) : item;
    k.q_zp = D == 3 ? (z == Lz - 1 ? item - QX * Ly * (Lz - 1) : item + QX * Ly) : item;
    // word index of the x-neighbour outside the quad: p = 1 -> first word of the next quad, p = 0 -> last of the previous
    k.w_edge = row * (4u * QX) + (k.p ? (q + 1u == QX ? 0u : 4u * q + 4u) : (q == 0u ? 4u * QX - 1u : 4u * q - 1u));
    return k;
}

// the update of quad k of replica r: ltf[i][th] = lanes of word i with U < threshold th (shared by all replicas)
template <int D, bool HB, int NT, bool MEAS = false>
__device__ __forceinline__ void pmj_quad_replica(const IsingArgs &a, const QuadGeom &k, uint32_t r, const uint32_t ltf[4][NT]) {
    int e_sum = 0, m_sum = 0;
    const uint32_t oc = 1u - a.colour, me = k.me, p = k.p, NW4 = k.NW4;
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
    const uint4 *__restrict__ So = (const uint4 *)a.s[oc] + (size_t)r * NW4;
    uint4 *Sc = (uint4 *)a.s[a.colour] + (size_t)r * NW4;
    const uint4 *__restrict__ Bo = (const uint4 *)a.bonds + ((size_t)(a.colour * a.R + r) * 3) * NW4;   // own forward bonds
    const uint4 *__restrict__ Bt = (const uint4 *)a.bonds + ((size_t)(oc * a.R + r) * 3) * NW4;         // other colour's
    uint4 raw, o, ym, yp, zm = zero, zp = zero, bx_own, bx_oth, by_m, by_own, bz_m = zero, bz_own = zero;
    const bool hints = a.l2_keep != 0xFFFFFFFFu;
    uint64_t keep = 0;
    if (hints) {
        // L2 eviction priorities: the working set (spins + coupling words of all replicas) is a little larger
        // than L2, and a cyclic pass over it would evict every line before its reuse.  The spins and the coupling words of the
        // first l2_keep replicas are loaded (and the spins stored) "evict_last", the other coupling words "evict_first": the
        // first part stays resident from half-sweep to half-sweep, only the second streams from HBM.
        keep = l2_policy_evict_last();
        const uint64_t stream = l2_policy_evict_first();
        const uint64_t pb = r < a.l2_keep ? keep : stream;
        raw = ld_hint(Sc + me, keep);
        o = ldg_hint(So + me, keep); ym = ldg_hint(So + k.q_ym, keep); yp = ldg_hint(So + k.q_yp, keep);
        if (D == 3) { zm = ldg_hint(So + k.q_zm, keep); zp = ldg_hint(So + k.q_zp, keep); }
        bx_own = ldg_hint(Bo + me, pb); bx_oth = ldg_hint(Bt + me, pb);
        by_m = ldg_hint(Bt + NW4 + k.q_ym, pb); by_own = ldg_hint(Bo + NW4 + me, pb);
        if (D == 3) { bz_m = ldg_hint(Bt + 2 * (size_t)NW4 + k.q_zm, pb); bz_own = ldg_hint(Bo + 2 * (size_t)NW4 + me, pb); }
    } else {
        raw = Sc[me];   // plain load: this array is written by the kernel
        o = __ldg(So + me); ym = __ldg(So + k.q_ym); yp = __ldg(So + k.q_yp);
        if (D == 3) { zm = __ldg(So + k.q_zm); zp = __ldg(So + k.q_zp); }
        bx_own = __ldg(Bo + me); bx_oth = __ldg(Bt + me);
        by_m = __ldg(Bt + NW4 + k.q_ym); by_own = __ldg(Bo + NW4 + me);
        if (D == 3) { bz_m = __ldg(Bt + 2 * (size_t)NW4 + k.q_zm); bz_own = __ldg(Bo + 2 * (size_t)NW4 + me); }
    }
    // the neighbour word outside the quad and (p = 0 only) its forward x coupling; inside the quad when QX == 1
    uint32_t o_edge, b_edge = 0u;
    if (k.QX == 1u) { o_edge = p ? o.x : o.w; b_edge = bx_oth.w; }
    else {
        o_edge = __ldg((const uint32_t *)So + k.w_edge);
        if (!p) b_edge = __ldg((const uint32_t *)Bt + k.w_edge);
    }
    uint32_t out[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t rw = u4c(raw, i), s = a.jneg ? ~rw : rw, oi = u4c(o, i);
        uint32_t av[6];
        if (p) {
            const uint32_t nx = i == 3 ? o_edge : u4c(o, (i + 1) & 3);
            av[0] = s ^ oi ^ u4c(bx_oth, i); av[1] = s ^ ((oi >> 1) | (nx << 31)) ^ u4c(bx_own, i);
        } else {
            const uint32_t pv = i == 0 ? o_edge : u4c(o, (i + 3) & 3), bp = i == 0 ? b_edge : u4c(bx_oth, (i + 3) & 3);
            av[0] = s ^ oi ^ u4c(bx_own, i); av[1] = s ^ ((oi << 1) | (pv >> 31)) ^ ((u4c(bx_oth, i) << 1) | (bp >> 31));
        }
        av[2] = s ^ u4c(ym, i) ^ u4c(by_m, i); av[3] = s ^ u4c(yp, i) ^ u4c(by_own, i);
        av[4] = D == 3 ? s ^ u4c(zm, i) ^ u4c(bz_m, i) : 0u; av[5] = D == 3 ? s ^ u4c(zp, i) ^ u4c(bz_own, i) : 0u;
        if constexpr (HB) {
            uint32_t b[6], m[NT];
#pragma unroll
            for (int kk = 0; kk < 6; ++kk) b[kk] = kk < 2 * D ? av[kk] ^ rw : 0u;
            count_masks<D>(b, m);
            uint32_t up = 0u;
#pragma unroll
            for (int kk = 0; kk < NT; ++kk) up |= m[kk] & ltf[i][kk];
            out[i] = ~up;
        } else if (D == 2) {
            const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
            const uint32_t ge2 = c1 | (s1 & av[3]), ge1 = av[0] | av[1] | av[2] | av[3];
            out[i] = rw ^ (ge2 | (ge1 & ltf[i][0]) | ltf[i][1]);
        } else {
            const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
            const uint32_t s2 = av[3] ^ av[4] ^ av[5], c2 = maj3(av[3], av[4], av[5]);
            const uint32_t b0 = s1 ^ s2, c3 = s1 & s2;
            const uint32_t b1 = c1 ^ c2 ^ c3, b2 = maj3(c1, c2, c3);
            out[i] = rw ^ ((b2 | (b1 & b0)) | ((b1 | b2) & ltf[i][0]) | ((b0 | b1 | b2) & ltf[i][1]) | ltf[i][D - 1]);
        }
        if (MEAS) fused_word_sums<D>(av, rw, out[i], oi, e_sum, m_sum);
    }
    if (hints) st_hint(Sc + me, make_uint4(out[0], out[1], out[2], out[3]), keep);
    else Sc[me] = make_uint4(out[0], out[1], out[2], out[3]);
    if (MEAS) {
        // all live lanes of the warp are at replica r: one reduction, one atomic pair per warp
        const unsigned act = __activemask();
        const int es = __reduce_add_sync(act, e_sum), ms = __reduce_add_sync(act, m_sum);
        if ((threadIdx.x & 31u) == (uint32_t)(__ffs(act) - 1)) acc_add(a, r, es, ms);
    }
}

// L2 prefetch of replica rn's rows for the warp whose first quad is me0 (one lane calls this): eight bulk requests
template <int D>
__device__ __forceinline__ void pmj_quad_prefetch(const IsingArgs &a, uint32_t rn, uint32_t me0, uint32_t pf_bytes, uint32_t pf_ym,
                                                  uint32_t pf_zm, uint32_t NW4) {
    const uint32_t oc = 1u - a.colour;
    const uint4 *Sn = (const uint4 *)a.s[oc] + (size_t)rn * NW4, *Cn = (const uint4 *)a.s[a.colour] + (size_t)rn * NW4;
    const uint4 *Bon = (const uint4 *)a.bonds + ((size_t)(a.colour * a.R + rn) * 3) * NW4;
    const uint4 *Btn = (const uint4 *)a.bonds + ((size_t)(oc * a.R + rn) * 3) * NW4;
    l2_prefetch_bulk(Cn + me0, pf_bytes);
    l2_prefetch_bulk(Sn + me0, pf_bytes);
    l2_prefetch_bulk(Bon + me0, pf_bytes);
    l2_prefetch_bulk(Btn + me0, pf_bytes);
    l2_prefetch_bulk(Bon + NW4 + me0, pf_bytes);
    l2_prefetch_bulk(Btn + NW4 + pf_ym, 512u);
    if (D == 3) {
        l2_prefetch_bulk(Bon + 2 * (size_t)NW4 + me0, pf_bytes);
        l2_prefetch_bulk(Btn + 2 * (size_t)NW4 + pf_zm, 512u);
    }
}

// One thread per quad; the thread builds the masks of its four words and loops over the replicas of its chunk
// (blockIdx.y).  The A/B partner of the cooperative kernel below (SPIN_OPT_KERNEL_VARIANT = 1).
template <int D, bool HB, bool MEAS = false>
__global__ void __launch_bounds__(128) ising_pmj_quad_halfsweep(const __grid_constant__ IsingArgs a) {
    constexpr int NT = HB ? 2 * D + 1 : D;
    const Geometry &g = a.g;
    const uint32_t items = (uint32_t)g.Ly * (uint32_t)g.Lz * (g.WX >> 2);
    const uint32_t item = blockIdx.x * blockDim.x + threadIdx.x;
    if (item >= items) return;
    const QuadGeom k = quad_geometry<D>(a, item);
    uint32_t ltf[4][NT];
#pragma unroll
    for (int i = 0; i < 4; ++i) lt_masks_full<NT, HB>(a, a.t, a.colour, 4u * item + (uint32_t)i + g.unit_off, 0u, ltf[i]);
    const uint32_t chunk = (a.R + gridDim.y - 1) / gridDim.y;
    const uint32_t r0 = blockIdx.y * chunk, r1 = min(a.R, r0 + chunk);
    // L2 prefetch of the next replica's rows (one lane per warp): the replica loop is a chain of dependent DRAM round
    // trips otherwise (61 % of the stall samples were long-scoreboard waits, profiles/r02a)
    const uint32_t lane = threadIdx.x & 31u, me0 = item - lane;
    const uint32_t pf_bytes = 16u * min(32u, items - me0);
    const uint32_t pf_ym = min(__shfl_sync(__activemask(), k.q_ym, 0), k.NW4 - 32u), pf_zm = min(__shfl_sync(__activemask(), k.q_zm, 0), k.NW4 - 32u);
    for (uint32_t r = r0; r < r1; ++r) {
        if (a.prefetch && lane == 0u && r + a.prefetch < r1 && k.NW4 >= 32u) pmj_quad_prefetch<D>(a, r + a.prefetch, me0, pf_bytes, pf_ym, pf_zm, k.NW4);
        pmj_quad_replica<D, HB, NT, MEAS>(a, k, r, ltf);
    }
}

// Cooperative version: a CTA of CH warps serves 32 consecutive quads.  Phase 1: its threads build the masks of the 128
// words of those quads, one word per thread (stride blockDim.x), into shared memory.  Phase 2: warp c updates the 32
// quads (one per lane: coalesced 512-byte accesses) for the replicas of chunk c, reading the masks from shared memory.
// Against the one-thread-per-quad kernel the Philox work per thread is 1 / 4 (the total is unchanged), the replica loop is
// CH times shorter and CH times more warps keep loads in flight; CTAs in different phases overlap on an SM.
template <int D, bool HB, bool MEAS = false>
__global__ void __launch_bounds__(256) ising_pmj_quad_coop_halfsweep(const __grid_constant__ IsingArgs a) {
    constexpr int NT = HB ? 2 * D + 1 : D;
    __shared__ __align__(16) uint32_t sm_lt[NT][128];   // [threshold][word of the CTA's 32 quads]
    const Geometry &g = a.g;
    const uint32_t items = (uint32_t)g.Ly * (uint32_t)g.Lz * (g.WX >> 2);
    const uint32_t me0 = blockIdx.x * 32u, lane = threadIdx.x & 31u, warp = threadIdx.x >> 5, CH = blockDim.x >> 5;
    for (uint32_t wi = threadIdx.x; wi < 128u; wi += blockDim.x) {
        if (me0 + (wi >> 2) < items) {
            uint32_t lt[NT];
            lt_masks_full<NT, HB>(a, a.t, a.colour, 4u * me0 + wi + g.unit_off, 0u, lt);
#pragma unroll
            for (int th = 0; th < NT; ++th) sm_lt[th][wi] = lt[th];
        }
    }
    const uint32_t item = me0 + lane;
    const uint32_t chunk = (a.R + CH - 1) / CH;
    const uint32_t r0 = warp * chunk, r1 = min(a.R, r0 + chunk);
    const bool live = item < items;
    const QuadGeom k = quad_geometry<D>(a, live ? item : 0u);
    const uint32_t pf_bytes = 16u * min(32u, items - me0);
    const uint32_t pf_ym = min(__shfl_sync(0xFFFFFFFFu, k.q_ym, 0), k.NW4 - 32u), pf_zm = min(__shfl_sync(0xFFFFFFFFu, k.q_zm, 0), k.NW4 - 32u);
    if (a.prefetch && lane == 0u && r0 < r1 && k.NW4 >= 32u) pmj_quad_prefetch<D>(a, r0, me0, pf_bytes, pf_ym, pf_zm, k.NW4);
    __syncthreads();
    if (!live) return;
    uint32_t ltf[4][NT];
#pragma unroll
    for (int th = 0; th < NT; ++th) {
        const uint4 v = *(const uint4 *)&sm_lt[th][4u * lane];
        ltf[0][th] = v.x; ltf[1][th] = v.y; ltf[2][th] = v.z; ltf[3][th] = v.w;
    }
    for (uint32_t r = r0; r < r1; ++r) {
        if (a.prefetch && lane == 0u && r + a.prefetch < r1 && k.NW4 >= 32u) pmj_quad_prefetch<D>(a, r + a.prefetch, me0, pf_bytes, pf_ym, pf_zm, k.NW4);
        pmj_quad_replica<D, HB, NT, MEAS>(a, k, r, ltf);
    }
}

}  // namespace spin
