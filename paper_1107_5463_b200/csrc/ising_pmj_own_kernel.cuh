// ising_pmj_own_kernel.cuh -- n = 1, per-bond +-1 couplings, bit-packed, every replica with its OWN update stream
// (replica_streams = 1: the literal "16 independent replicas" reading of BASELINE config 4), Lx % 256 == 0.
// With own streams the acceptance masks of a word cannot be shared between replicas, so every (replica, word) pays its own
// random numbers; what this kernel shares with ising_pmj_quad_halfsweep is the access pattern (one thread per quad of four
// words: 128-bit loads of spins and coupling planes) and with the strip kernels the comparison: the first two Philox calls
// of the four words unconditionally as straight-line code (eight chains in flight), words with undecided lanes pushed into
// the per-warp shared-memory queue and finished one per lane after each replica (lt_mask_select_head / _tail).
#pragma once
#include "ising_int8_kernel.cuh"

namespace spin {

// grid = (ceil(quads / blockDim.x), replica chunks); Metropolis rule
template <int D>
__global__ void __launch_bounds__(128) ising_pmj_quad_own_halfsweep(const __grid_constant__ IsingArgs a) {
    __shared__ DeferQueue dq;
    const Geometry &g = a.g;
    const uint32_t items = (uint32_t)g.Ly * (uint32_t)g.Lz * (g.WX >> 2);
    const uint32_t item = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const bool live = item < items;
    if (lane == 0u) dq.n[warp] = 0u;
    __syncwarp();
    const QuadGeom k = quad_geometry<D>(a, live ? item : 0u);
    const uint32_t chunk = (a.R + gridDim.y - 1) / gridDim.y;
    const uint32_t r0 = blockIdx.y * chunk, r1 = min(a.R, r0 + chunk);
    const uint32_t oc = 1u - a.colour, me = k.me, p = k.p, NW4 = k.NW4;
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
    uint32_t *const base = (uint32_t *)a.s[a.colour];
    for (uint32_t r = r0; r < r1; ++r) {      // every lane of the warp runs the same replicas: the drain below is warp-wide
        if (live) {
            const uint4 *__restrict__ So = (const uint4 *)a.s[oc] + (size_t)r * NW4;
            uint4 *Sc = (uint4 *)a.s[a.colour] + (size_t)r * NW4;
            const uint4 *__restrict__ Bo = (const uint4 *)a.bonds + ((size_t)(a.colour * a.R + r) * 3) * NW4;   // own forward bonds
            const uint4 *__restrict__ Bt = (const uint4 *)a.bonds + ((size_t)(oc * a.R + r) * 3) * NW4;         // other colour's
            const uint4 raw = Sc[me];   // plain load: this array is written by the kernel
            const uint4 o = __ldg(So + me), ym = __ldg(So + k.q_ym), yp = __ldg(So + k.q_yp);
            const uint4 zm = D == 3 ? __ldg(So + k.q_zm) : zero, zp = D == 3 ? __ldg(So + k.q_zp) : zero;
            const uint4 bx_own = __ldg(Bo + me), bx_oth = __ldg(Bt + me);
            const uint4 by_m = __ldg(Bt + NW4 + k.q_ym), by_own = __ldg(Bo + NW4 + me);
            const uint4 bz_m = D == 3 ? __ldg(Bt + 2 * (size_t)NW4 + k.q_zm) : zero, bz_own = D == 3 ? __ldg(Bo + 2 * (size_t)NW4 + me) : zero;
            uint32_t o_edge, b_edge = 0u;
            if (k.QX == 1u) { o_edge = p ? o.x : o.w; b_edge = bx_oth.w; }
            else {
                o_edge = __ldg((const uint32_t *)So + k.w_edge);
                if (!p) b_edge = __ldg((const uint32_t *)Bt + k.w_edge);
            }
            const uint32_t rho = a.replica_streams ? r + a.rho_off : 0u;
            uint32_t fresh[4], eq[4], mm[4][D];
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
                fresh[i] = ising_new_word_head<D>(a, a.t, a.colour, 4u * me + (uint32_t)i + g.unit_off, rho, rw, av, eq[i], mm[i]);
            }
            // words with undecided lanes go to the queue with their provisional value (a full queue finishes them here); the quad
            // is stored as it stands and the drain below overwrites the queued words (same warp, ordered by __syncwarp)
#pragma unroll
            for (int i = 0; i < 4; ++i)
                (void)defer_or_finish<D>(a, dq, warp, 4u * me + (uint32_t)i + g.unit_off, rho, eq[i], mm[i], fresh[i], r * g.NW + 4u * me + (uint32_t)i);
            Sc[me] = make_uint4(fresh[0], fresh[1], fresh[2], fresh[3]);
        }
        defer_drain<D>(a, dq, warp, lane, [&](uint32_t widx, uint32_t word) { base[widx] = word; });
        __syncwarp();
        if (lane == 0u) dq.n[warp] = 0u;
        __syncwarp();
    }
}

}  // namespace spin
