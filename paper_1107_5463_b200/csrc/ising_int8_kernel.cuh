// ising_int8_kernel.cuh -- n = 1, one byte per spin (0 = +1, 1 = -1), uniform coupling +-1, Lx % 64 == 0.
// PAPER.md:37-38 (Eq. (2)), PAPER.md:42 (checkerboard, pre-tabulated Boltzmann factors).
//
// Layout: a unit = 32 consecutive same-colour sites of a row = 32 consecutive bytes;
// inside a unit, site sigma (0..31, position along x) sits at byte 4 (sigma & 7) + (sigma >> 3).  With that
// order the eight 32-bit words w0..w7 of a unit pack into the lane mask of the unit (bit sigma = spin of site
// sigma) by m = w0 + 2 w1 + 4 w2 + ... + 128 w7 -- seven IMADs on the FMA pipe and no ALU-pipe work -- and
// unpack by w_k = (m >> k) & 0x01010101.  Everything between load and store is the bit-sliced logic of the
// multi-spin-coded kernel, 32 sites per instruction.
//
// Work decomposition: one thread owns unit column w over K consecutive rows (a "strip") and rolls the other
// colour's rows through registers, so each neighbour row is loaded and packed (K + 2) / K times instead of 3.
#pragma once
#include <type_traits>

#include "ising_kernels.cuh"

namespace spin {

// byte offset of site sigma inside its 32-byte unit (int8 fast layout)
__host__ __device__ __forceinline__ uint32_t int8_byte_of_lane(uint32_t sigma) { return 4u * (sigma & 7u) + (sigma >> 3); }

// lane mask of the 32-byte unit at p (bytes are exactly 0 or 1)
__device__ __forceinline__ uint32_t int8_pack_unit(const uint8_t *p) {
    const uint4 lo = __ldg((const uint4 *)p), hi = __ldg((const uint4 *)p + 1);
    uint32_t m = lo.x;
    m = lo.y * 2u + m;
    m = lo.z * 4u + m;
    m = lo.w * 8u + m;
    m = hi.x * 16u + m;
    m = hi.y * 32u + m;
    m = hi.z * 64u + m;
    m = hi.w * 128u + m;
    return m;
}

__device__ __forceinline__ void int8_store_unit(uint8_t *p, uint32_t m) {
    const uint32_t c = 0x01010101u;
    uint4 *dst = (uint4 *)p;
    dst[0] = make_uint4(m & c, (m >> 1) & c, (m >> 2) & c, (m >> 3) & c);
    dst[1] = make_uint4((m >> 4) & c, (m >> 5) & c, (m >> 6) & c, (m >> 7) & c);
}

// Lane mask of the x-neighbour that is not at the same compressed index: p = 1 -> site xh + 1, p = 0 -> xh - 1
// (periodic along the row).  o = this unit of the other colour, rowp = start of that row, w = unit in row.
__device__ __forceinline__ uint32_t int8_side_mask(const uint8_t *rowp, uint32_t o, uint32_t p, uint32_t w, uint32_t WX) {
    if (p) {
        const uint32_t wn = w + 1u == WX ? 0u : w + 1u;
        return (o >> 1) | ((uint32_t)__ldg(rowp + 32u * wn) << 31);       // lane 0 of the next unit: byte 0
    }
    const uint32_t wn = w == 0u ? WX - 1u : w - 1u;
    return (o << 1) | (uint32_t)__ldg(rowp + 32u * wn + 31u);              // lane 31 of the previous unit: byte 31
}

// flip mask of one unit from its unsatisfied-bond masks av[0 .. 2 D): flip iff dE <= 0 or U < T(dE)
template <int D>
__device__ __forceinline__ uint32_t ising_flip_mask(const IsingArgs &a, uint32_t t, uint32_t colour, uint32_t unit, uint32_t rho,
                                                    const uint32_t av[6]) {
    if (D == 2) {
        const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
        const uint32_t ge2 = c1 | (s1 & av[3]), ge1 = av[0] | av[1] | av[2] | av[3];
        const uint32_t m[2] = {ge1 & ~ge2, ~ge1};
        return ge2 | lt_mask_select<2>(a, t, colour, unit, rho, m);
    }
    const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
    const uint32_t s2 = av[3] ^ av[4] ^ av[5], c2 = maj3(av[3], av[4], av[5]);
    const uint32_t b0 = s1 ^ s2, c3 = s1 & s2;
    const uint32_t b1 = c1 ^ c2 ^ c3, b2 = maj3(c1, c2, c3);
    const uint32_t ge3 = b2 | (b1 & b0);
    const uint32_t m[3] = {b1 & ~b0 & ~b2, b0 & ~b1 & ~b2, ~(b0 | b1 | b2)};
    return ge3 | lt_mask_select<3>(a, t, colour, unit, rho, m);
}

// New value of a unit's word (bit = 1: spin -1) from its own word `raw` and its unsatisfied-bond masks av[].
//   HB = false (Metropolis, Eq. (2)): raw ^ flip mask.
//   HB = true  (heat bath): av[k] ^ raw = lanes whose neighbour term J s_j is -1; with k of them the
//   local field is h = 2 D - 2 k and the new spin is +1 iff U < T_hb(h).
template <int D, bool HB>
__device__ __forceinline__ uint32_t ising_new_word(const IsingArgs &a, uint32_t t, uint32_t colour, uint32_t unit, uint32_t rho,
                                                   uint32_t raw, const uint32_t av[6]) {
    if constexpr (!HB) {
        return raw ^ ising_flip_mask<D>(a, t, colour, unit, rho, av);
    } else {
        uint32_t b[6], m[2 * D + 1];
#pragma unroll
        for (int k = 0; k < 6; ++k) b[k] = k < 2 * D ? av[k] ^ raw : 0u;
        count_masks<D>(b, m);
        return ~lt_mask_select<2 * D + 1, true>(a, t, colour, unit, rho, m);
    }
}

// Metropolis word with the comparison cut after DEFER_CALLS calls: returns raw ^ (flip mask so far); eq = lanes still
// undecided (their final flip bits are lt_mask_select_tail of the same unit and masks m[], XORed into the word)
template <int D>
__device__ __forceinline__ uint32_t ising_new_word_head(const IsingArgs &a, uint32_t t, uint32_t colour, uint32_t unit, uint32_t rho,
                                                        uint32_t raw, const uint32_t av[6], uint32_t &eq, uint32_t m[D]) {
    if (D == 2) {
        const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
        const uint32_t ge2 = c1 | (s1 & av[3]), ge1 = av[0] | av[1] | av[2] | av[3];
        m[0] = ge1 & ~ge2; m[1] = ~ge1;
        return raw ^ (ge2 | lt_mask_select_head<D>(a, t, colour, unit, rho, m, eq));
    }
    const uint32_t s1 = av[0] ^ av[1] ^ av[2], c1 = maj3(av[0], av[1], av[2]);
    const uint32_t s2 = av[3] ^ av[4] ^ av[5], c2 = maj3(av[3], av[4], av[5]);
    const uint32_t b0 = s1 ^ s2, c3 = s1 & s2;
    const uint32_t b1 = c1 ^ c2 ^ c3, b2 = maj3(c1, c2, c3);
    const uint32_t ge3 = b2 | (b1 & b0);
    m[0] = b1 & ~b0 & ~b2; m[1] = b0 & ~b1 & ~b2; m[D - 1] = ~(b0 | b1 | b2);
    return raw ^ (ge3 | lt_mask_select_head<D>(a, t, colour, unit, rho, m, eq));
}

// Owner side of the deferred tail: the word is complete (returns true: store it) or it went into the warp's queue
// (returns false: the drain stores it); a full queue makes the owner finish the unit itself.
template <int D>
__device__ __forceinline__ bool defer_or_finish(const IsingArgs &a, DeferQueue &q, uint32_t warp, uint32_t unit, uint32_t rho,
                                                uint32_t eq, const uint32_t m[D], uint32_t &word, uint32_t index) {
    if (eq == 0u) return true;
    const uint32_t pos = atomicAdd(&q.n[warp], 1u);
    if (pos >= a.defer_cap) {
        word ^= lt_mask_select_tail<D>(a, a.t, a.colour, unit, rho, m, eq);
        return true;
    }
    q.f[warp][0][pos] = unit; q.f[warp][1][pos] = rho; q.f[warp][2][pos] = eq;
    q.f[warp][3][pos] = m[0]; q.f[warp][4][pos] = D == 3 ? m[1] : 0u;
    q.f[warp][5][pos] = word; q.f[warp][6][pos] = index;
    return false;
}

// Drain: lane l finishes pending unit l (l + 32, ... never: the queue holds at most DEFER_CAP = 32 entries).
// store(index, word) writes the finished word.  Call with the whole warp converged.
template <int D, typename Store>
__device__ __forceinline__ void defer_drain(const IsingArgs &a, DeferQueue &q, uint32_t warp, uint32_t lane, Store store) {
    __syncwarp();
    const uint32_t n = min(q.n[warp], a.defer_cap);
    if (lane < n) {
        uint32_t m[D];
        m[0] = q.f[warp][3][lane];
        if (D == 3) m[1] = q.f[warp][4][lane];
        m[D - 1] = 0u;   // the last mask never enters select_digit (its lanes take the default digit)
        const uint32_t lt = lt_mask_select_tail<D>(a, a.t, a.colour, q.f[warp][0][lane], q.f[warp][1][lane], m, q.f[warp][2][lane]);
        store(q.f[warp][6][lane], q.f[warp][5][lane] ^ lt);
    }
}

// Heat-bath counterparts of the three helpers above (bit-packed strip kernel): head = two unconditional calls against the
// 2 D + 1 heat-bath thresholds, the new word is ~(U < T_hb); a queued word is patched by XOR with its tail, as for Metropolis
// (the tail's lanes are undecided lanes, whose provisional bit is 1).
template <int D>
__device__ __forceinline__ uint32_t ising_new_word_head_hb(const IsingArgs &a, uint32_t t, uint32_t colour, uint32_t unit, uint32_t rho,
                                                           uint32_t raw, const uint32_t av[6], uint32_t &eq, uint32_t m[2 * D + 1]) {
    uint32_t b[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) b[k] = k < 2 * D ? av[k] ^ raw : 0u;
    count_masks<D>(b, m);
    return ~lt_mask_select_head<2 * D + 1, true>(a, t, colour, unit, rho, m, eq);
}
template <int D>
__device__ __forceinline__ bool defer_or_finish_hb(const IsingArgs &a, DeferQueueHB<D> &q, uint32_t warp, uint32_t unit, uint32_t rho,
                                                   uint32_t eq, const uint32_t m[2 * D + 1], uint32_t &word, uint32_t index) {
    if (eq == 0u) return true;
    const uint32_t pos = atomicAdd(&q.n[warp], 1u);
    if (pos >= a.defer_cap) {
        word ^= lt_mask_select_tail<2 * D + 1, true>(a, a.t, a.colour, unit, rho, m, eq);
        return true;
    }
    q.f[warp][0][pos] = unit; q.f[warp][1][pos] = rho; q.f[warp][2][pos] = eq; q.f[warp][3][pos] = word; q.f[warp][4][pos] = index;
#pragma unroll
    for (int k = 0; k < 2 * D; ++k) q.f[warp][5 + k][pos] = m[k];
    return false;
}
template <int D, typename Store>
__device__ __forceinline__ void defer_drain_hb(const IsingArgs &a, DeferQueueHB<D> &q, uint32_t warp, uint32_t lane, Store store) {
    __syncwarp();
    const uint32_t n = min(q.n[warp], a.defer_cap);
    if (lane < n) {
        uint32_t m[2 * D + 1];
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) m[k] = q.f[warp][5 + k][lane];
        m[2 * D] = 0u;   // the last class takes the default digit
        const uint32_t lt = lt_mask_select_tail<2 * D + 1, true>(a, a.t, a.colour, q.f[warp][0][lane], q.f[warp][1][lane], m, q.f[warp][2][lane]);
        store(q.f[warp][4][lane], q.f[warp][3][lane] ^ lt);
    }
}

// the 32 bytes of a unit as loaded, before packing (kept in flight while the previous row is being updated)
struct Int8RawUnit {
    uint4 lo, hi;
};
__device__ __forceinline__ Int8RawUnit int8_load_unit(const uint8_t *p) {
    Int8RawUnit u;
    u.lo = __ldg((const uint4 *)p);
    u.hi = __ldg((const uint4 *)p + 1);
    return u;
}
// the same for the array being updated: plain (coherent) loads -- the non-coherent path is for data that stays
// read-only for the whole kernel
__device__ __forceinline__ Int8RawUnit int8_load_unit_rw(const uint8_t *p) {
    Int8RawUnit u;
    u.lo = *((const uint4 *)p);
    u.hi = *((const uint4 *)p + 1);
    return u;
}
__device__ __forceinline__ uint32_t int8_pack_raw(const Int8RawUnit &u) {
    uint32_t m = u.lo.x;
    m = u.lo.y * 2u + m;
    m = u.lo.z * 4u + m;
    m = u.lo.w * 8u + m;
    m = u.hi.x * 16u + m;
    m = u.hi.y * 32u + m;
    m = u.hi.z * 64u + m;
    m = u.hi.w * 128u + m;
    return m;
}
// the one byte of the x-neighbour outside the unit: p = 1 -> lane 0 of the next unit, p = 0 -> lane 31 of the previous
__device__ __forceinline__ uint32_t int8_side_byte(const uint8_t *rowp, uint32_t p, uint32_t w, uint32_t WX) {
    if (p) return __ldg(rowp + 32u * (w + 1u == WX ? 0u : w + 1u));
    return __ldg(rowp + 32u * (w == 0u ? WX - 1u : w - 1u) + 31u);
}

// One thread per (replica, z, strip of K rows, unit column w); w is the fastest index, so a warp reads
// 1 KB of consecutive bytes per row.  Software-pipelined: the loads of row k + 1 are issued before the
// update of row k is computed, so their latency hides behind the Philox / bit-slice work.
// At most 128 threads per CTA; d = 2: 7 CTAs per SM, i.e. at most 72 registers (one more costs a whole CTA of occupancy:
// measured 72.6 vs 75.0 us at L = 16384).
template <int D, int K, bool HB = false, bool MEAS = false, bool RANGED = false>
__global__ void __launch_bounds__(128, D == 2 ? 7 : 4) ising_int8_halfsweep(const __grid_constant__ IsingArgs a) {
    const Geometry &g = a.g;
    const uint32_t WX = g.WX, Ly = (uint32_t)g.Ly, Lz = (uint32_t)g.Lz;
    // RANGED: the launch updates rows (d = 2) / planes (d = 3) [sw_p0, sw_p0 + sw_pn) of the slowest axis only (slab handles, half-sweeps
    // in pieces); a template parameter because the whole-lattice instance is 4 % faster without the offsets (3D L = 512: 33.1 vs 34.5 us)
    const uint32_t ys0 = (RANGED && D == 2) ? g.sw_p0 : 0u, Lys = (RANGED && D == 2) ? g.sw_pn : Ly;
    const uint32_t zs0 = (RANGED && D == 3) ? g.sw_p0 : 0u, Lzs = (RANGED && D == 3) ? g.sw_pn : Lz;
    const uint32_t nstrip = (Lys + K - 1) / K;
    const uint32_t per_replica = WX * nstrip * Lzs;
    const uint32_t item = blockIdx.x * blockDim.x + threadIdx.x;
    // The deferred tail of the digit comparison (ising_bitpack_strip_halfsweep) is compiled out for Metropolis: measured on B200
    // the queue's live state pushes the d = 2 instance past its 72 registers (7 CTAs per SM): 87.7 us against 72.8 us without.
    // The heat-bath rule, whose inline tail is longer, gains from it: 2D L = 16384 83.5 -> 78.1 us, 3D L = 512 47.4 us (= Metropolis)
    constexpr bool DEFER = HB && !MEAS;
    __shared__ typename std::conditional<HB, DeferQueueHB<D>, DeferQueue>::type dq;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    if (DEFER) { if (lane == 0u) dq.n[warp] = 0u; __syncwarp(); }
    if (item < per_replica * a.R) {
    const uint32_t r = item / per_replica, it = item - r * per_replica;
    const uint32_t sz = fdiv(it, g.divWX), w = it - sz * WX;      // sz = strip + nstrip * z
    const uint32_t zl = sz / nstrip, z = zs0 + zl, y0 = ys0 + (sz - zl * nstrip) * K;
    const uint32_t kend = min((uint32_t)K, ys0 + Lys - y0);
    const uint8_t *__restrict__ other = (const uint8_t *)a.s[1 - a.colour] + (size_t)r * g.Nh;
    uint8_t *mine = (uint8_t *)a.s[a.colour] + (size_t)r * g.Nh;
    const uint32_t rho = a.replica_streams ? r + a.rho_off : 0u;
    const uint32_t jflip = a.jneg ? 0xFFFFFFFFu : 0u;
    const size_t rowbytes = g.RL, plane = rowbytes * Ly;
    const size_t zoff = (size_t)z * plane;
    const size_t zm_off = (D == 3) ? (size_t)(z == 0 ? Lz - 1 : z - 1) * plane : 0;
    const size_t zp_off = (D == 3) ? (size_t)(z == Lz - 1 ? 0 : z + 1) * plane : 0;
    const uint32_t ym0 = y0 == 0 ? Ly - 1 : y0 - 1;
    uint32_t p = (y0 + z + a.colour) & 1u;
    // prologue: rows y0 - 1 and y0 of the other colour, and everything row y0 needs
    const Int8RawUnit r_prev = int8_load_unit(other + zoff + ym0 * rowbytes + 32u * w);
    const Int8RawUnit r_cur = int8_load_unit(other + zoff + y0 * rowbytes + 32u * w);
    Int8RawUnit pf_next, pf_mine, pf_zm, pf_zp;
    uint32_t pf_side;
    {
        const uint32_t yp = y0 + 1 == Ly ? 0u : y0 + 1;
        const size_t off = y0 * rowbytes + 32u * w;
        pf_next = int8_load_unit(other + zoff + yp * rowbytes + 32u * w);
        pf_mine = int8_load_unit_rw(mine + zoff + off);
        pf_side = int8_side_byte(other + zoff + y0 * rowbytes, p, w, WX);
        if (D == 3) { pf_zm = int8_load_unit(other + zm_off + off); pf_zp = int8_load_unit(other + zp_off + off); }
    }
    uint32_t o_prev = int8_pack_raw(r_prev), o_cur = int8_pack_raw(r_cur);
    const uint32_t unit0 = (y0 + Ly * z) * WX + w + g.unit_off;   // global Philox unit of row y0 (slab offset included)
    int e_sum = 0, m_sum = 0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        if ((uint32_t)k < kend) {
            const uint32_t y = y0 + k;
            const size_t off = y * rowbytes + 32u * w;
            const uint32_t o_next = int8_pack_raw(pf_next), raw = int8_pack_raw(pf_mine);
            const uint32_t side = p ? ((o_cur >> 1) | (pf_side << 31)) : ((o_cur << 1) | pf_side);
            uint32_t o_zm = 0u, o_zp = 0u;
            if (D == 3) { o_zm = int8_pack_raw(pf_zm); o_zp = int8_pack_raw(pf_zp); }
            if (k + 1 < K && (uint32_t)(k + 1) < kend) {
                // row y + 1 <= Ly - 1 exists inside this strip: issue its loads now
                const uint32_t y1 = y + 1, y2 = y1 + 1 == Ly ? 0u : y1 + 1;
                const size_t off1 = y1 * rowbytes + 32u * w;
                pf_next = int8_load_unit(other + zoff + y2 * rowbytes + 32u * w);
                pf_mine = int8_load_unit_rw(mine + zoff + off1);
                pf_side = int8_side_byte(other + zoff + y1 * rowbytes, p ^ 1u, w, WX);
                if (D == 3) { pf_zm = int8_load_unit(other + zm_off + off1); pf_zp = int8_load_unit(other + zp_off + off1); }
            }
            const uint32_t s = raw ^ jflip;
            uint32_t av[6];
            av[0] = s ^ o_cur; av[1] = s ^ side; av[2] = s ^ o_prev; av[3] = s ^ o_next;
            if (D == 3) { av[4] = s ^ o_zm; av[5] = s ^ o_zp; }
            const uint32_t unit = unit0 + (uint32_t)k * WX;
            if (D == 2) { av[4] = 0u; av[5] = 0u; }
            if constexpr (DEFER && HB) {
                uint32_t eq, mm[2 * D + 1];
                uint32_t fresh = ising_new_word_head_hb<D>(a, a.t, a.colour, unit, rho, raw, av, eq, mm);
                // index of the unit in the whole colour array (32-byte units)
                const uint32_t uidx = (uint32_t)(((size_t)r * g.Nh + zoff + off) >> 5);
                if (defer_or_finish_hb<D>(a, dq, warp, unit, rho, eq, mm, fresh, uidx)) int8_store_unit(mine + zoff + off, fresh);
            } else if constexpr (DEFER) {
                uint32_t eq, mm[D];
                uint32_t fresh = ising_new_word_head<D>(a, a.t, a.colour, unit, rho, raw, av, eq, mm);
                const uint32_t uidx = (uint32_t)(((size_t)r * g.Nh + zoff + off) >> 5);
                if (defer_or_finish<D>(a, dq, warp, unit, rho, eq, mm, fresh, uidx)) int8_store_unit(mine + zoff + off, fresh);
            } else {
                const uint32_t fresh = ising_new_word<D, HB>(a, a.t, a.colour, unit, rho, raw, av);
                int8_store_unit(mine + zoff + off, fresh);
                if (MEAS) fused_word_sums<D>(av, raw, fresh, o_cur, e_sum, m_sum);
            }
            o_prev = o_cur;
            o_cur = o_next;
            p ^= 1u;
        }
    }
    if (MEAS) fused_commit(a, r, e_sum, m_sum);
    }
    if constexpr (DEFER && HB) {
        uint8_t *base = (uint8_t *)a.s[a.colour];
        defer_drain_hb<D>(a, dq, warp, lane, [&](uint32_t uidx, uint32_t word) { int8_store_unit(base + 32u * (size_t)uidx, word); });
    } else if constexpr (DEFER) {
        uint8_t *base = (uint8_t *)a.s[a.colour];
        defer_drain<D>(a, dq, warp, lane, [&](uint32_t uidx, uint32_t word) { int8_store_unit(base + 32u * (size_t)uidx, word); });
    }
}

// The same strip walk for BIT-PACKED storage with uniform couplings (own random stream per replica or one replica):
// one thread per (replica, z, strip of K rows, word column w); words of the other colour are rolled through
// registers over the rows, the loads of row k + 1 are issued before row k is computed, and the index arithmetic is
// paid once per strip instead of once per word.  Results are bit-identical to ising_bitpack_halfsweep.
template <int D, int K, bool HB = false, bool MEAS = false, bool RANGED = false>
__global__ void __launch_bounds__(128, (D == 3 && K == 4 && !HB && !MEAS) ? 6 : 0) ising_bitpack_strip_halfsweep(const __grid_constant__ IsingArgs a) {
    const Geometry &g = a.g;
    const uint32_t WX = g.WX, Ly = (uint32_t)g.Ly, Lz = (uint32_t)g.Lz;
    // RANGED: the launch updates rows (d = 2) / planes (d = 3) [sw_p0, sw_p0 + sw_pn) of the slowest axis only (slab handles, half-sweeps
    // in pieces); a template parameter because the whole-lattice instance is 4 % faster without the offsets (3D L = 512: 33.1 vs 34.5 us)
    const uint32_t ys0 = (RANGED && D == 2) ? g.sw_p0 : 0u, Lys = (RANGED && D == 2) ? g.sw_pn : Ly;
    const uint32_t zs0 = (RANGED && D == 3) ? g.sw_p0 : 0u, Lzs = (RANGED && D == 3) ? g.sw_pn : Lz;
    const uint32_t nstrip = (Lys + K - 1) / K;
    const uint32_t per_replica = WX * nstrip * Lzs;
    const uint32_t item = blockIdx.x * blockDim.x + threadIdx.x;
    constexpr bool DEFER = !MEAS;          // deferred tail of the digit comparison (both rules; recorded sweeps finish their words inline)
    __shared__ typename std::conditional<HB, DeferQueueHB<D>, DeferQueue>::type dq;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    if (DEFER) { if (lane == 0u) dq.n[warp] = 0u; __syncwarp(); }
    if (item < per_replica * a.R) {
    const uint32_t r = item / per_replica, it = item - r * per_replica;
    const uint32_t sz = fdiv(it, g.divWX), w = it - sz * WX;      // sz = strip + nstrip * z
    const uint32_t zl = sz / nstrip, z = zs0 + zl, y0 = ys0 + (sz - zl * nstrip) * K;
    const uint32_t kend = min((uint32_t)K, ys0 + Lys - y0);
    const uint32_t *__restrict__ other = (const uint32_t *)a.s[1 - a.colour] + (size_t)r * g.NW;
    uint32_t *mine = (uint32_t *)a.s[a.colour] + (size_t)r * g.NW;
    const uint32_t rho = a.replica_streams ? r + a.rho_off : 0u;
    const uint32_t jflip = a.jneg ? 0xFFFFFFFFu : 0u;
    const uint32_t plane = WX * Ly, zoff = z * plane;
    const uint32_t zm_off = (D == 3) ? (z == 0 ? Lz - 1 : z - 1) * plane : 0u;
    const uint32_t zp_off = (D == 3) ? (z == Lz - 1 ? 0u : z + 1) * plane : 0u;
    const uint32_t w_next = w + 1u == WX ? 0u : w + 1u, w_prev = w == 0u ? WX - 1u : w - 1u;
    const uint32_t ym0 = y0 == 0 ? Ly - 1 : y0 - 1;
    uint32_t p = (y0 + z + a.colour) & 1u;
    uint32_t o_prev = __ldg(other + zoff + ym0 * WX + w), o_cur = __ldg(other + zoff + y0 * WX + w);
    uint32_t pf_next, pf_mine, pf_side, pf_zm = 0u, pf_zp = 0u;
    {
        const uint32_t yp = y0 + 1 == Ly ? 0u : y0 + 1, off = y0 * WX + w;
        pf_next = __ldg(other + zoff + yp * WX + w);
        pf_mine = mine[zoff + off];
        pf_side = __ldg(other + zoff + y0 * WX + (p ? w_next : w_prev));
        if (D == 3) { pf_zm = __ldg(other + zm_off + off); pf_zp = __ldg(other + zp_off + off); }
    }
    const uint32_t unit0 = (y0 + Ly * z) * WX + w + g.unit_off;
    int e_sum = 0, m_sum = 0;
    bool whole_strip = false;
    if constexpr (!HB) if (K > 1 && kend == (uint32_t)K) {   // Metropolis (DEFER or MEAS)
        whole_strip = true;
        // whole strip (the steady state): every load first, then the K heads of the digit comparison as straight-line code --
        // 2 K independent Philox chains in flight -- and only then the queue pushes and stores
        uint32_t o_row[K + 2], raw_k[K], side_k[K], zm_k[K], zp_k[K];
        o_row[0] = o_prev; o_row[1] = o_cur; o_row[2] = pf_next;
        raw_k[0] = pf_mine; side_k[0] = pf_side; zm_k[0] = pf_zm; zp_k[0] = pf_zp;
#pragma unroll
        for (int k = 1; k < K; ++k) {
            const uint32_t y1 = y0 + k, y2 = y1 + 1 == Ly ? 0u : y1 + 1, off1 = y1 * WX + w;
            o_row[k + 2] = __ldg(other + zoff + y2 * WX + w);
            raw_k[k] = mine[zoff + off1];
            side_k[k] = __ldg(other + zoff + y1 * WX + (((p + k) & 1u) ? w_next : w_prev));
            zm_k[k] = D == 3 ? __ldg(other + zm_off + off1) : 0u;
            zp_k[k] = D == 3 ? __ldg(other + zp_off + off1) : 0u;
        }
        uint32_t fresh_k[K], eq_k[K], mm_k[K][D];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t pk = (p + k) & 1u, oc = o_row[k + 1];
            const uint32_t side = pk ? ((oc >> 1) | (side_k[k] << 31)) : ((oc << 1) | (side_k[k] >> 31));
            const uint32_t s = raw_k[k] ^ jflip;
            uint32_t av[6];
            av[0] = s ^ oc; av[1] = s ^ side; av[2] = s ^ o_row[k]; av[3] = s ^ o_row[k + 2];
            av[4] = D == 3 ? s ^ zm_k[k] : 0u; av[5] = D == 3 ? s ^ zp_k[k] : 0u;
            fresh_k[k] = ising_new_word_head<D>(a, a.t, a.colour, unit0 + (uint32_t)k * WX, rho, raw_k[k], av, eq_k[k], mm_k[k]);
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t off = (y0 + k) * WX + w;
            if constexpr (MEAS) {
                // recorded sweep: the word is finished here (the few undecided lanes inline) so that E and M can be taken from it
                if (eq_k[k] != 0u) fresh_k[k] ^= lt_mask_select_tail<D>(a, a.t, a.colour, unit0 + (uint32_t)k * WX, rho, mm_k[k], eq_k[k]);
                mine[zoff + off] = fresh_k[k];
                const uint32_t pk = (p + k) & 1u, oc = o_row[k + 1];
                const uint32_t side = pk ? ((oc >> 1) | (side_k[k] << 31)) : ((oc << 1) | (side_k[k] >> 31));
                const uint32_t s = raw_k[k] ^ jflip;
                uint32_t av[6];
                av[0] = s ^ oc; av[1] = s ^ side; av[2] = s ^ o_row[k]; av[3] = s ^ o_row[k + 2];
                av[4] = D == 3 ? s ^ zm_k[k] : 0u; av[5] = D == 3 ? s ^ zp_k[k] : 0u;
                fused_word_sums<D>(av, raw_k[k], fresh_k[k], oc, e_sum, m_sum);
            } else {
                if (defer_or_finish<D>(a, dq, warp, unit0 + (uint32_t)k * WX, rho, eq_k[k], mm_k[k], fresh_k[k], r * g.NW + zoff + off)) mine[zoff + off] = fresh_k[k];
            }
        }
    }
    if (!whole_strip)
#pragma unroll
    for (int k = 0; k < K; ++k) {
        if ((uint32_t)k < kend) {
            const uint32_t y = y0 + k, off = y * WX + w;
            const uint32_t o_next = pf_next, raw = pf_mine, o_zm = pf_zm, o_zp = pf_zp;
            const uint32_t side = p ? ((o_cur >> 1) | (pf_side << 31)) : ((o_cur << 1) | (pf_side >> 31));
            if (k + 1 < K && (uint32_t)(k + 1) < kend) {
                const uint32_t y1 = y + 1, y2 = y1 + 1 == Ly ? 0u : y1 + 1, off1 = y1 * WX + w;
                pf_next = __ldg(other + zoff + y2 * WX + w);
                pf_mine = mine[zoff + off1];
                pf_side = __ldg(other + zoff + y1 * WX + (p ? w_prev : w_next));   // row y + 1 has the other parity
                if (D == 3) { pf_zm = __ldg(other + zm_off + off1); pf_zp = __ldg(other + zp_off + off1); }
            }
            const uint32_t s = raw ^ jflip;
            uint32_t av[6];
            av[0] = s ^ o_cur; av[1] = s ^ side; av[2] = s ^ o_prev; av[3] = s ^ o_next;
            av[4] = D == 3 ? s ^ o_zm : 0u; av[5] = D == 3 ? s ^ o_zp : 0u;
            if constexpr (DEFER && HB) {
                uint32_t eq, mm[2 * D + 1];
                const uint32_t unit = unit0 + (uint32_t)k * WX;
                uint32_t fresh = ising_new_word_head_hb<D>(a, a.t, a.colour, unit, rho, raw, av, eq, mm);
                if (defer_or_finish_hb<D>(a, dq, warp, unit, rho, eq, mm, fresh, r * g.NW + zoff + off)) mine[zoff + off] = fresh;
            } else if constexpr (DEFER) {
                uint32_t eq, mm[D];
                const uint32_t unit = unit0 + (uint32_t)k * WX;
                uint32_t fresh = ising_new_word_head<D>(a, a.t, a.colour, unit, rho, raw, av, eq, mm);
                if (defer_or_finish<D>(a, dq, warp, unit, rho, eq, mm, fresh, r * g.NW + zoff + off)) mine[zoff + off] = fresh;
            } else {
                const uint32_t fresh = ising_new_word<D, HB>(a, a.t, a.colour, unit0 + (uint32_t)k * WX, rho, raw, av);
                mine[zoff + off] = fresh;
                if (MEAS) fused_word_sums<D>(av, raw, fresh, o_cur, e_sum, m_sum);
            }
            o_prev = o_cur;
            o_cur = o_next;
            p ^= 1u;
        }
    }
    if (MEAS) fused_commit(a, r, e_sum, m_sum);
    }
    if constexpr (DEFER && HB) {
        uint32_t *base = (uint32_t *)a.s[a.colour];
        defer_drain_hb<D>(a, dq, warp, lane, [&](uint32_t widx, uint32_t word) { base[widx] = word; });
    } else if constexpr (DEFER) {
        uint32_t *base = (uint32_t *)a.s[a.colour];
        defer_drain<D>(a, dq, warp, lane, [&](uint32_t widx, uint32_t word) { base[widx] = word; });
    }
}

}  // namespace spin
