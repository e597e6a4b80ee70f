// ising_int8_kernel.cuh -- n = 1, one byte per spin (0 = +1, 1 = -1), uniform coupling +-1, Lx % 64 == 0.
// One thread per 32-site unit: two 128-bit loads per neighbour row, byte-parallel arithmetic on
// 32-bit registers (4 sites each), acceptance masks from the bit-serial comparison expanded from
// bits to bytes, two 128-bit stores.  PAPER.md:37-38 (Eq. (2)), PAPER.md:42 (checkerboard, table).
#pragma once
#include "ising_kernels.cuh"

namespace spin {

__device__ __forceinline__ void load32(const uint8_t *p, uint32_t v[8]) {
    const uint4 lo = __ldg((const uint4 *)p), hi = __ldg((const uint4 *)p + 1);
    v[0] = lo.x; v[1] = lo.y; v[2] = lo.z; v[3] = lo.w;
    v[4] = hi.x; v[5] = hi.y; v[6] = hi.z; v[7] = hi.w;
}

// lanes 4k .. 4k+3 of mask m as bit 0 of the four bytes of the result (other bits are junk)
__device__ __forceinline__ uint32_t expand4(uint32_t m, int k) {
    return ((m >> (4 * k)) & 0xFu) * 0x00204081u;
}

template <int D>
__global__ void __launch_bounds__(256) ising_int8_halfsweep(const __grid_constant__ IsingArgs a) {
    const Geometry &g = a.g;
    constexpr int NT = D;
    const uint32_t NW = g.NW, WX = g.WX;
    const uint8_t *__restrict__ other_base = (const uint8_t *)a.s[1 - a.colour];
    uint8_t *mine_base = (uint8_t *)a.s[a.colour];
    const uint32_t jmask = a.jneg ? 0x01010101u : 0u;
    for (uint32_t gi = blockIdx.x * blockDim.x + threadIdx.x; gi < NW; gi += gridDim.x * blockDim.x) {
        const uint32_t row = fdiv(gi, g.divWX), w = gi - row * WX;
        const uint32_t z = fdiv(row, g.divLy), y = row - z * (uint32_t)g.Ly;
        const uint32_t p = (y + z + a.colour) & 1u;
        // byte index of the one neighbour outside this unit's own 32 bytes of the other colour's row
        const uint32_t xh0 = 32u * w;
        const uint32_t xs = p ? (xh0 + 32u == g.RL ? 0u : xh0 + 32u) : (xh0 == 0u ? g.RL - 1u : xh0 - 1u);
        const size_t b_side = (size_t)row * g.RL + xs;
        const size_t b_c = (size_t)gi * 32u;
        const size_t rowbytes = g.RL;
        const size_t b_ym = y == 0 ? b_c + rowbytes * (g.Ly - 1) : b_c - rowbytes;
        const size_t b_yp = y == (uint32_t)g.Ly - 1 ? b_c - rowbytes * (g.Ly - 1) : b_c + rowbytes;
        size_t b_zm = b_c, b_zp = b_c;
        if (D == 3) {
            const size_t plane = rowbytes * g.Ly;
            b_zm = z == 0 ? b_c + plane * (g.Lz - 1) : b_c - plane;
            b_zp = z == (uint32_t)g.Lz - 1 ? b_c - plane * (g.Lz - 1) : b_c + plane;
        }
        uint32_t lt[NT];
        for (uint32_t r = 0; r < a.R; ++r) {
            const uint8_t *__restrict__ other = other_base + (size_t)r * g.Nh;
            uint8_t *mine = mine_base + (size_t)r * g.Nh;
            uint32_t s[8], o[8], nu[8];
            load32(mine + b_c, s);
            load32(other + b_c, o);
            const uint32_t sb = other[b_side];
            {
                uint32_t u[8], v[8];
                load32(other + b_ym, u);
                load32(other + b_yp, v);
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    // the neighbour at (x >> 1) -+ 1: this row shifted by one byte
                    const uint32_t sd = p ? __byte_perm(o[k], k < 7 ? o[k + 1] : sb, 0x4321)
                                          : __byte_perm(k ? o[k - 1] : (sb << 24), o[k], 0x6543);
                    const uint32_t sj = s[k] ^ jmask;
                    nu[k] = (sj ^ o[k]) + (sj ^ sd) + (sj ^ u[k]) + (sj ^ v[k]);
                }
            }
            if (D == 3) {
                uint32_t u[8], v[8];
                load32(other + b_zm, u);
                load32(other + b_zp, v);
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const uint32_t sj = s[k] ^ jmask;
                    nu[k] += (sj ^ u[k]) + (sj ^ v[k]);
                }
            }
            if (r == 0 || a.replica_streams) lt_masks_full<NT>(a, gi, a.replica_streams ? r : 0u, lt);
            // flip = [n_u >= q/2] | [n_u >= q/2 - 1] & lt4 | ... | lt_{2q}, evaluated on the bits of n_u
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const uint32_t x = nu[k], x1 = x >> 1, x2 = x >> 2;
                uint32_t f;
                if (D == 2) {
                    // n_u in 0..4: flip = (n_u >= 2) | (n_u odd & lt4) | lt8
                    f = x1 | x2 | (x & expand4(lt[0], k)) | expand4(lt[1], k);
                } else {
                    // n_u in 0..6 = (x2 x1 x0): flip = x2 | x1 & (x0 | lt4) | x0 & lt8 | lt12
                    f = x2 | (x1 & (x | expand4(lt[0], k))) | (x & expand4(lt[1], k)) | expand4(lt[2], k);
                }
                s[k] ^= f & 0x01010101u;
            }
            uint4 *dst = (uint4 *)(mine + b_c);
            dst[0] = make_uint4(s[0], s[1], s[2], s[3]);
            dst[1] = make_uint4(s[4], s[5], s[6], s[7]);
        }
    }
}

}  // namespace spin
