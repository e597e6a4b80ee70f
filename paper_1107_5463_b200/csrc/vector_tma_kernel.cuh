// vector_tma_kernel.cuh -- n = 2 (XY) and n = 3 (Heisenberg) half-sweep on simple-cubic lattices with every tile and its
// halo staged in shared memory by the TMA unit (cp.async.bulk.tensor + mbarrier), north_star (a); the B200 counterpart
// of the paper's "tile + boundary layer in shared memory" (Fig. 1 at PAPER.md:50), with k = 1 (R-1).
//
// Work decomposition.  A tile is TY consecutive rows y of one plane z, full rows (TX = Lx / 2 sites of one colour,
// TX <= 256).  One CTA marches along z through a column of tiles (fixed replica and row block) and keeps the other
// colour's tiles of planes z - 1, z, z + 1 in a ring of four shared-memory slots, the fourth being filled for z + 2
// while z is computed: every other-colour tile enters shared memory ONCE per column and serves three steps (as the
// +z, the in-plane and the -z neighbour), instead of being fetched five times through L1 / L2 as in the strip kernel.
// A slot is one TMA box of TY rows x NC components plus two single-row boxes (the rows below and above, periodic).  The
// CTA's own spins are used once, so they go from global memory to registers and back (128-bit, issued at the top of a
// step and consumed at its end).  The (row block, z) steps of a replica are cut into equal contiguous ranges, one per
// CTA (all CTAs resident: 3 per SM, 2 for the heat-bath and fused-measurement variants), so a CTA restarts its ring at most once or twice.
// Arithmetic: vector_quad_update (vector_kernels.cuh), the same fp32 operations in the same order as the strip and the
// plain kernel -- results are bit-identical to both.
//
// MEAS (colour-1 half-sweep of spin_sweep_record): every bond joins the two colours,
// so E = -sum_{i in colour 1} s'_i . h_i with the local field h_i this half-sweep has formed anyway, and M = sum of
// the new colour-1 spins plus the colour-0 spins at the same compressed indices (in the centre slot).  Per-site terms
// in fp32 (each product and sum rounded separately), accumulated in fp64 per thread, reduced per CTA in a fixed order
// and written as one partial per CTA; vector_measure_finalize sums the partials in a fixed order (deterministic).
#pragma once
#include <cuda.h>

#include "measure_kernels.cuh"
#include "vector_kernels.cuh"

namespace spin {

constexpr int TMA_CONSUMER_WARPS = 8;
constexpr int TMA_THREADS = (TMA_CONSUMER_WARPS + 1) * 32;   // + the producer warp
constexpr int TMA_SLOTS = 6;        // other-colour ring: planes z - 1, z, z + 1 and three in flight
// resident CTAs per SM the kernel is compiled for: 3 (80 registers) for the plain Metropolis half-sweep, 2 for the variants
// that need more registers (heat bath, fused measurement)
__host__ __device__ constexpr int tma_ctas_per_sm(bool hb, bool meas) { return 2; }

struct VectorTmaArgs {
    VectorArgs v;
    CUtensorMap main_map[2];   // per colour array: box (TX, TY, 1, NC, 1) of float [R][NC][Lz][Ly][TX]
    CUtensorMap row_map[2];    // per colour array: box (TX, 1, 1, NC, 1)
    uint32_t TY;               // rows per tile (the last row block of a plane may hold fewer)
    uint32_t nyb;              // row blocks per plane = ceil(Ly / TY)
    double *part;              // MEAS: [R][gridDim.x][1 + NC] partial sums
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// the producer's wait: it is hundreds of cycles ahead of the consumers, so it sleeps between probes instead of
// spending issue slots
__device__ __forceinline__ void mbar_wait_backoff(uint64_t *bar, uint32_t parity) {
    uint32_t done = 0;
    while (true) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (done) break;
        __nanosleep(200);
    }
}
// box of tensor map `map` at coordinates (0, y, z, 0, r) -> shared memory at dst, completion counted on `bar`
__device__ __forceinline__ void tma_load_box(void *dst, const CUtensorMap *map, uint64_t *bar, uint32_t y, uint32_t z, uint32_t r) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(0), "r"((int)y), "r"((int)z), "r"(0), "r"((int)r)
        : "memory");
}

__host__ __device__ constexpr uint32_t tma_align128(uint32_t v) { return (v + 127u) & ~127u; }
// bytes of one ring slot and of the whole dynamic shared memory of a CTA
__host__ __device__ constexpr uint32_t tma_main_bytes(int NC, int TY, uint32_t TX) { return tma_align128((uint32_t)NC * TY * TX * 4u); }
__host__ __device__ constexpr uint32_t tma_row_bytes(int NC, uint32_t TX) { return tma_align128((uint32_t)NC * TX * 4u); }
__host__ __device__ constexpr uint32_t tma_slot_bytes(int NC, int TY, uint32_t TX) { return tma_main_bytes(NC, TY, TX) + 2u * tma_row_bytes(NC, TX); }
__host__ __device__ constexpr uint32_t tma_smem_bytes(int NC, int TY, uint32_t TX) {
    return TMA_SLOTS * tma_slot_bytes(NC, TY, TX) + 128u;
}

template <int NC>
__device__ __forceinline__ Quad<NC> lds_quad(const float *base, uint32_t comp_stride, uint32_t off) {
    Quad<NC> q;
#pragma unroll
    for (int c = 0; c < NC; ++c) q.c[c] = *(const float4 *)(base + c * comp_stride + off);
    return q;
}

// grid = (CTAs per replica, R); block = TMA_THREADS; dynamic shared memory = tma_smem_bytes(NC, TY, TX).
// Ly need not be a multiple of TY: the rows of the last block beyond Ly are zero-filled by the TMA unit and skipped.
// Warp roles: warps 0 .. 7 update the sites; warp 8 is the producer -- one lane issues the slot fills as slots are
// released.  There is no CTA-wide barrier in the loop: a slot is handed back through an mbarrier that every consumer warp
// arrives on when it has finished the last step that reads the slot, so the warps of a CTA drift apart by up to a step.
template <int NC, bool UNITJ, bool HB, bool MEAS>
__global__ void __launch_bounds__(TMA_THREADS, tma_ctas_per_sm(HB, MEAS)) vector_tma_halfsweep(const __grid_constant__ VectorTmaArgs ta) {
    extern __shared__ __align__(1024) uint8_t tma_smem[];
    const VectorArgs &a = ta.v;
    const Geometry &g = a.g;
    const uint32_t TX = g.RL, QX = TX >> 2, Ly = (uint32_t)g.Ly, Lz = (uint32_t)g.Lz, Nh = g.Nh, TY = ta.TY;
    const uint32_t main_b = tma_main_bytes(NC, TY, TX), row_b = tma_row_bytes(NC, TX), slot_b = main_b + 2u * row_b;
    uint64_t *const full = (uint64_t *)(tma_smem + TMA_SLOTS * slot_b);   // per ring slot: "the fill has landed"
    uint64_t *const empty = full + TMA_SLOTS;                             // per ring slot: "every consumer warp is done with it"
    const uint32_t r = blockIdx.y, tid = threadIdx.x;
    const uint32_t S = ta.nyb * Lz;                                // steps (row block, z) of one replica, z fastest
    const uint32_t sa = (uint32_t)((uint64_t)S * blockIdx.x / gridDim.x), sb = (uint32_t)((uint64_t)S * (blockIdx.x + 1u) / gridDim.x);
    const uint32_t oc = 1u - a.colour;
    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < TMA_SLOTS; ++k) { mbar_init(&full[k], 1u); mbar_init(&empty[k], TMA_CONSUMER_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    double e_acc = 0.0, m_acc[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) m_acc[c] = 0.0;
    if (sa < sb && tid >= TMA_CONSUMER_WARPS * 32) {
        // ---- producer: the flat sequence of slot fills.  A segment is a maximal run of steps in one column; its fills are
        // planes z_first - 1 .. z_last + 1 (periodic), in order; fill l goes to slot l % TMA_SLOTS once that slot's previous
        // occupant (fill l - TMA_SLOTS) has been released.
        if (tid == TMA_CONSUMER_WARPS * 32) {
            const uint32_t slot_tx = (uint32_t)NC * TX * 4u * (TY + 2u);
            uint32_t issued = 0u;
            for (uint32_t seg = sa; seg < sb;) {
                const uint32_t yb = seg / Lz, z0 = seg - yb * Lz, y0 = yb * TY, len = min(Lz - z0, sb - seg);
                for (uint32_t i = 0; i < len + 2u; ++i, ++issued) {
                    uint32_t z = z0 + i;                            // plane z0 - 1 + i, periodic
                    z = z == 0u ? Lz - 1u : (z - 1u >= Lz ? z - 1u - Lz : z - 1u);
                    const uint32_t slot_i = issued % TMA_SLOTS;
                    if (issued >= (uint32_t)TMA_SLOTS) mbar_wait_backoff(&empty[slot_i], (issued / TMA_SLOTS - 1u) & 1u);
                    uint8_t *slot = tma_smem + slot_i * slot_b;
                    mbar_arrive_expect_tx(&full[slot_i], slot_tx);
                    tma_load_box(slot, &ta.main_map[oc], &full[slot_i], y0, z, r);
                    tma_load_box(slot + main_b, &ta.row_map[oc], &full[slot_i], y0 == 0u ? Ly - 1u : y0 - 1u, z, r);
                    tma_load_box(slot + main_b + row_b, &ta.row_map[oc], &full[slot_i], y0 + TY >= Ly ? 0u : y0 + TY, z, r);
                }
                seg += len;
            }
        }
    } else if (sa < sb) {
        // ---- consumers
        const uint32_t rho = a.replica_streams ? r + a.rho_off : 0u;
        const uint32_t tag = make_tag(a.colour, DOM_VECTOR_UPDATE, 0);
        const float Jx = a.Jdir[0], Jy = a.Jdir[1], Jz = a.Jdir[2];
        const uint32_t cs_main = TY * TX;                           // component stride inside a main box (floats)
        float *const mine = a.s[a.colour] + (size_t)r * NC * Nh;
        const uint32_t plane = TX * Ly;
        uint32_t b = 0u;          // first fill the current step needs (then b + 1, b + 2)
        uint32_t waited = 0u;     // fills [0, waited) have been waited for
        uint32_t yb = sa / Lz, z = sa - yb * Lz;
        for (uint32_t s = sa; s < sb; ++s) {
            const uint32_t y0 = yb * TY;
            for (; waited < b + 3u; ++waited) mbar_wait(&full[waited % TMA_SLOTS], (waited / TMA_SLOTS) & 1u);
            const float *const zm_s = (const float *)(tma_smem + (b % TMA_SLOTS) * slot_b);
            const float *const ce_s = (const float *)(tma_smem + ((b + 1u) % TMA_SLOTS) * slot_b);
            const float *const zp_s = (const float *)(tma_smem + ((b + 2u) % TMA_SLOTS) * slot_b);
            const float *const top_s = (const float *)((const uint8_t *)ce_s + main_b);
            const float *const bot_s = (const float *)((const uint8_t *)ce_s + main_b + row_b);
            const uint32_t rows = min(TY, Ly - y0);                 // valid rows of this tile
            for (uint32_t qi = tid; qi < rows * QX; qi += TMA_CONSUMER_WARPS * 32) {
                const uint32_t ly = fdiv(qi, g.divQX), x4 = (qi - ly * QX) << 2, y = y0 + ly;
                const uint32_t p = (y + z + a.colour) & 1u;
                const uint32_t in_tile = ly * TX + x4;
                const uint32_t off = z * plane + y * TX + x4;       // compressed index of the quad's first site
                // the quad's own spins are used once: global memory -> registers, in flight during the field sums and proposals
                Quad<NC> own;
#pragma unroll
                for (int c = 0; c < NC; ++c) own.c[c] = *(const float4 *)(mine + (size_t)c * Nh + off);
                float2 hp[2][NC];
                Quad<NC> o_cur;
                {
                    o_cur = lds_quad<NC>(ce_s, cs_main, in_tile);
                    const Quad<NC> o_zm = lds_quad<NC>(zm_s, cs_main, in_tile), o_zp = lds_quad<NC>(zp_s, cs_main, in_tile);
                    const Quad<NC> o_prev = ly == 0u ? lds_quad<NC>(top_s, TX, x4) : lds_quad<NC>(ce_s, cs_main, in_tile - TX);
                    const Quad<NC> o_next = ly == rows - 1u ? lds_quad<NC>(bot_s, TX, x4) : lds_quad<NC>(ce_s, cs_main, in_tile + TX);
                    // the one x-neighbour outside the quad, periodic along the (full) row
                    const uint32_t xs = p ? (x4 + 4u == TX ? 0u : x4 + 4u) : (x4 == 0u ? TX - 1u : x4 - 1u);
                    float side[NC];
#pragma unroll
                    for (int c = 0; c < NC; ++c) side[c] = ce_s[c * cs_main + ly * TX + xs];
                    vector_quad_field<NC, 3, UNITJ>(Jx, Jy, Jz, p, o_cur, side, o_prev, o_next, o_zm, o_zp, hp);
                }
                float res[NC][4];
                vector_quad_accept<NC, HB>(a, hp, own, off + g.j_off, rho, tag, res);
#pragma unroll
                for (int c = 0; c < NC; ++c)
                    *(float4 *)(mine + (size_t)c * Nh + off) = make_float4(res[c][0], res[c][1], res[c][2], res[c][3]);
                if (MEAS && off >= g.own_j0 && off < g.own_j1) {
                    float eq = 0.0f;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const float2 *hh = hp[i >> 1];
                        float dot = __fmul_rn(res[0][i], (i & 1) ? hh[0].y : hh[0].x);
#pragma unroll
                        for (int c = 1; c < NC; ++c) dot = __fadd_rn(dot, __fmul_rn(res[c][i], (i & 1) ? hh[c].y : hh[c].x));
                        eq = __fadd_rn(eq, dot);
                    }
                    e_acc -= (double)eq;
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        const float4 o = o_cur.c[c];
                        const float mq = __fadd_rn(__fadd_rn(__fadd_rn(res[c][0], res[c][1]), __fadd_rn(res[c][2], res[c][3])),
                                                   __fadd_rn(__fadd_rn(o.x, o.y), __fadd_rn(o.z, o.w)));
                        m_acc[c] += (double)mq;
                    }
                }
            }
            // next step; the fills below its first one are handed back to the producer by this warp
            if (++z == Lz) { z = 0u; ++yb; }
            const uint32_t b_next = b + (z == 0u ? 3u : 1u);
            __syncwarp();
            if ((tid & 31u) == 0u && s + 1u < sb)
                for (uint32_t l = b; l < b_next; ++l)
                    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&empty[l % TMA_SLOTS])) : "memory");
            b = b_next;
        }
    }
    if (MEAS) {
        __shared__ double red[32];
        double *out = ta.part + ((size_t)r * gridDim.x + blockIdx.x) * (1 + NC);
        const double e = block_sum(e_acc, red);
        if (tid == 0) out[0] = e;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const double v = block_sum(m_acc[c], red);
            if (tid == 0) out[1 + c] = v;
        }
    }
}

}  // namespace spin
