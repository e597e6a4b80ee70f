// ising_tblock_kernel.cuh -- exact temporal blocking for the 2D Ising models: TWO full sweeps (four
// half-sweeps) per pass over the lattice, results bit-identical to four plain half-sweeps.  The results-neutral
// counterpart of the paper's "k updates per tile load" (its k-fold multi-hit changes the dynamics, R-1).
//
// A CTA owns a stripe of H full rows and marches down it with a ring of 16 rows (both colours, bit-packed, one 32-site
// word per thread and row) in shared memory.  Half-sweep s = 1 .. 4 (colour 0, colour 1 of sweep t, then of sweep t + 1)
// of a row needs its three neighbour rows at half-sweep s - 1, so the four half-sweeps follow the load front at a
// distance of 2 rows each: in iteration i the CTA loads row i, applies half-sweep 1 to row i - 2, half-sweep 2 to row
// i - 4, 3 to row i - 6, 4 to row i - 8 and stores row i - 8.  With that skew everything an iteration reads was written in
// an earlier one (ONE barrier per iteration; see the hazard table in DESIGN.md section 5) and the five pieces of work are
// independent (four Philox chains per thread in flight).  Each row is read from HBM once and written once per TWO sweeps:
// 1 byte per update (int8) instead of 3.  A stripe starts 4 rows above its first row and ends 4 below its last
// (shrinking halo: 12 redundant row updates per stripe = 3 / H of the work), reading from one pair of colour arrays and
// writing to the other (ping-pong: a neighbouring stripe may still need the old rows), which the host swaps afterwards.
//
// Random numbers: the same Philox unit (global row and word), sweep index and colour as the plain kernels, so the
// update sequence is unchanged (north_star (b)).  Acceptance: the lazy digit comparison with the deferred tail of the strip
// kernels -- two Philox calls per word unconditionally, words with undecided lanes queued per warp and finished one per
// lane before the barrier.
#pragma once
#include "ising_int8_kernel.cuh"

namespace spin {

constexpr int TB_RING = 16;          // ring slots (rows) per colour; 10 are live
constexpr int TB_QCAP = 128;         // deferred-tail queue entries per warp and iteration: 4 half-sweeps x 32 lanes, it cannot overflow
constexpr int TB_QFIELDS = 4;        // one uint4 per entry: unit, eq, m[0], index of the word in the ring | (sweep offset, colour) << 30

__host__ __device__ constexpr size_t tblock_smem_bytes(uint32_t WX) {
    return (size_t)(2u * TB_RING * WX + (WX / 32u) * (4u + TB_QFIELDS * TB_QCAP)) * 4u;
}

// INT8: global arrays in the int8 fast layout (32-byte units), else bit-packed words.  grid = (stripes, R),
// block = WX threads (one per word of a row; 32 <= WX <= MAXT), dynamic shared memory = tblock_smem_bytes(WX).
// Reads a.s[0], a.s[1]; writes a.alt[0], a.alt[1]; sweeps a.t and a.t + 1.
// HB: heat-bath rule: the new word comes from the lazy comparison against the 2 d + 1 heat-bath thresholds, no queue.
template <bool INT8, int MAXT, bool HB = false>
__global__ void __launch_bounds__(MAXT, MAXT <= 256 ? 2 : 1) ising_tblock2_sweeps(const __grid_constant__ IsingArgs a) {
    extern __shared__ __align__(16) uint32_t tb_smem[];
    const Geometry &g = a.g;
    const uint32_t WX = g.WX, Ly = (uint32_t)g.Ly, w = threadIdx.x, r = blockIdx.y;
    const uint32_t warp = w >> 5, lane = w & 31u;
    uint32_t *const qn = tb_smem + 2u * TB_RING * WX + warp * (4u + TB_QFIELDS * TB_QCAP);   // this warp's queue: count (16 bytes), entries
    uint32_t *const qf = qn + 4;
    const uint32_t H = a.tb_rows, y0 = blockIdx.x * H;
    if (y0 >= Ly) return;
    const int Hs = (int)min(H, Ly - y0);
    const uint32_t w_next = w + 1u == WX ? 0u : w + 1u, w_prev = w == 0u ? WX - 1u : w - 1u;
    const uint32_t rho = a.replica_streams ? r + a.rho_off : 0u;
    const uint32_t jflip = a.jneg ? 0xFFFFFFFFu : 0u;
    const size_t rep = INT8 ? (size_t)r * g.Nh : (size_t)r * g.NW * 4u;           // byte offset of the replica
    const uint8_t *const src0 = (const uint8_t *)a.s[0] + rep, *const src1 = (const uint8_t *)a.s[1] + rep;
    uint8_t *const dst0 = (uint8_t *)a.alt[0] + rep, *const dst1 = (uint8_t *)a.alt[1] + rep;
    const uint32_t rowbytes = INT8 ? 32u * WX : 4u * WX, wbytes = INT8 ? 32u * w : 4u * w;
    // global row of local row 0 (4 above the stripe, periodic); y_s = global row of the row half-sweep s works on
    uint32_t y_in = (y0 + 4u * Ly - 4u) % Ly;
    uint32_t y_st[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) y_st[s] = (y_in + 8u * Ly - 2u * (uint32_t)(s + 1)) % Ly;
    if (lane == 0u) *qn = 0u;
    // the other colour's words of rows l and l + 1 of each half-sweep, kept for the next iteration (where they are rows l - 1 and l):
    // both were final when they were read, so in the steady state a half-sweep loads one new row instead of three
    uint32_t roll_prev[4] = {0u, 0u, 0u, 0u}, roll_cur[4] = {0u, 0u, 0u, 0u};
    for (int i = 0; i <= Hs + 11; ++i) {
        // ---- the loads of local row i, consumed at the end of the iteration
        const bool loading = i <= Hs + 7;
        Int8RawUnit ld0, ld1;
        uint32_t lw0 = 0u, lw1 = 0u;
        if (loading) {
            const size_t off = (size_t)y_in * rowbytes + wbytes;
            if (INT8) { ld0 = int8_load_unit(src0 + off); ld1 = int8_load_unit(src1 + off); }
            else { lw0 = __ldg((const uint32_t *)(src0 + off)); lw1 = __ldg((const uint32_t *)(src1 + off)); }
        }
        // ---- half-sweeps 1 .. 4 on local rows i - 2, i - 4, i - 6, i - 8.  In the steady state (all four rows inside their
        // ranges) the four updates are straight-line code, so that the scheduler can interleave their Philox chains
        const auto half_sweep = [&](int s, bool rolled) {
            const int l = i - 2 * s;
            const uint32_t c = (uint32_t)(s - 1) & 1u, tt = a.t + (uint32_t)(s > 2), y = y_st[s - 1];
            uint32_t *const mine_r = tb_smem + c * (TB_RING * WX);
            const uint32_t *const oth_r = tb_smem + (1u - c) * (TB_RING * WX);
            const uint32_t slot = ((uint32_t)l & (TB_RING - 1u)) * WX;
            const uint32_t raw = mine_r[slot + w];
            const uint32_t o_cur = rolled ? roll_cur[s - 1] : oth_r[slot + w];
            const uint32_t o_prev = rolled ? roll_prev[s - 1] : oth_r[(((uint32_t)l - 1u) & (TB_RING - 1u)) * WX + w];
            const uint32_t o_next = oth_r[(((uint32_t)l + 1u) & (TB_RING - 1u)) * WX + w];
            roll_prev[s - 1] = o_cur; roll_cur[s - 1] = o_next;
            const uint32_t p = (y + c) & 1u;
            const uint32_t o_side = oth_r[slot + (p ? w_next : w_prev)];
            const uint32_t side = p ? ((o_cur >> 1) | (o_side << 31)) : ((o_cur << 1) | (o_side >> 31));
            const uint32_t sp = raw ^ jflip;
            uint32_t av[6];
            av[0] = sp ^ o_cur; av[1] = sp ^ side; av[2] = sp ^ o_prev; av[3] = sp ^ o_next; av[4] = 0u; av[5] = 0u;
            const uint32_t unit = y * WX + w + g.unit_off;
            if constexpr (HB) {
                mine_r[slot + w] = ising_new_word<2, true>(a, tt, c, unit, rho, raw, av);
                return;
            }
            uint32_t eq, mm[2];
            const uint32_t fresh = ising_new_word_head<2>(a, tt, c, unit, rho, raw, av, eq, mm);
            mine_r[slot + w] = fresh;
            if (eq != 0u) {
                const uint32_t pos = atomicAdd(qn, 1u);   // < TB_QCAP: at most 4 x 32 pushes per warp and iteration
                ((uint4 *)qf)[pos] = make_uint4(unit, eq, mm[0], (c * (TB_RING * WX) + slot + w) | ((2u * (uint32_t)(s > 2) + c) << 30));
            }
        };
        if (i >= 12 && i <= Hs + 8) {
            const bool rolled = i > 12;   // the iteration before ran all four half-sweeps as well
            half_sweep(1, rolled); half_sweep(2, rolled); half_sweep(3, rolled); half_sweep(4, rolled);
        } else {
#pragma unroll 1
            for (int s = 1; s <= 4; ++s) {
                const int l = i - 2 * s;
                if (l >= s && l <= Hs + 7 - s) {
                    if (s == 1) half_sweep(1, false); else if (s == 2) half_sweep(2, false); else if (s == 3) half_sweep(3, false); else half_sweep(4, false);
                }
            }
        }
        // ---- deferred tails: one queued word per lane (two rounds if more than 32 are pending), patched in the ring
        __syncwarp();
        {
            const uint32_t nq = *qn;
            for (uint32_t e = lane; e < nq; e += 32u) {
                const uint4 q = ((const uint4 *)qf)[e];
                uint32_t mm[2];
                mm[0] = q.z; mm[1] = 0u;
                const uint32_t tc = q.w >> 30;
                const uint32_t lt = lt_mask_select_tail<2>(a, a.t + (tc >> 1), tc & 1u, q.x, rho, mm, q.y);
                tb_smem[q.w & 0x3FFFFFFFu] ^= lt;
            }
            __syncwarp();
            if (lane == 0u) *qn = 0u;
        }
        // ---- store local row i - 8 (half-sweep 4 done: both colours final)
        {
            const int l = i - 8;
            if (l >= 4 && l <= Hs + 3) {
                const uint32_t slot = ((uint32_t)l & (TB_RING - 1u)) * WX;
                const uint32_t f0 = tb_smem[slot + w], f1 = tb_smem[TB_RING * WX + slot + w];
                const size_t off = (size_t)y_st[3] * rowbytes + wbytes;
                if (INT8) { int8_store_unit(dst0 + off, f0); int8_store_unit(dst1 + off, f1); }
                else { *(uint32_t *)(dst0 + off) = f0; *(uint32_t *)(dst1 + off) = f1; }
            }
        }
        // ---- local row i into the ring
        if (loading) {
            const uint32_t slot = ((uint32_t)i & (TB_RING - 1u)) * WX;
            tb_smem[slot + w] = INT8 ? int8_pack_raw(ld0) : lw0;
            tb_smem[TB_RING * WX + slot + w] = INT8 ? int8_pack_raw(ld1) : lw1;
        }
        y_in = y_in + 1u == Ly ? 0u : y_in + 1u;
#pragma unroll
        for (int s = 0; s < 4; ++s) y_st[s] = y_st[s] + 1u == Ly ? 0u : y_st[s] + 1u;
        __syncthreads();
    }
}

}  // namespace spin
