// setup_kernels.cuh -- initial states, bond tables and conversion between the canonical (lexicographic)
// layouts of the ABI and the colour-split device layouts.  Not on the timed path.
// Random draws follow DESIGN.md "The contract":
//   hot start n = 1 : s_i = -1 iff bit (i & 31) of word ((i >> 5) & 3) of rand(i >> 7, r, 0, INIT)
//   hot start n >= 2: direction(w0, w1) of rand(i, r, 0, INIT)
//   bonds           : J[r][mu][i] = -1 iff bit (i & 31) of word mu of rand(i >> 5, r, 0, BONDS)
#pragma once
#include "ising_kernels.cuh"
#include "vector_kernels.cuh"

namespace spin {

struct SetupArgs {
    Geometry g;
    PhiloxKeys keys;
    uint32_t R;
    int32_t bitpack;  // n = 1 only
    int32_t int8perm; // n = 1, int8 fast layout: site sigma of a unit at byte 4 (sigma & 7) + (sigma >> 3)
    int32_t nc;       // 1, 2, 3
};

// byte index of compressed site j in an int8 colour array
__device__ __forceinline__ uint32_t int8_byte_index(const SetupArgs &a, uint32_t j) {
    return a.int8perm ? ((j & ~31u) | (4u * (j & 7u) + ((j >> 3) & 3u))) : j;
}

// (colour c, compressed index j) -> lexicographic site index
__device__ __forceinline__ uint32_t lex_index(const Geometry &g, uint32_t c, uint32_t j) {
    const uint32_t row = fdiv(j, g.divRL), xh = j - row * g.RL;
    const uint32_t z = fdiv(row, g.divLy), y = row - z * (uint32_t)g.Ly;
    const uint32_t p = (y + z + c) & 1u;
    return 2u * xh + p + (uint32_t)g.Lx * row;
}

// mode 0: cold, 1: hot (from seed), 2: from canonical int8 [R][N] of +-1.
// idx runs over (colour, replica, j); with bit-packing a warp covers exactly one word (Nh % 32 == 0).
// d_bad (mode 2): nonzero = the canonical array failed its +-1 check: leave the arrays alone
__global__ void __launch_bounds__(256) ising_fill(const __grid_constant__ SetupArgs a, int mode, const int8_t *canon,
                                                  void *s0, void *s1, const int *d_bad = nullptr) {
    const Geometry &g = a.g;
    if (d_bad && *d_bad) return;
    const uint32_t per_colour = a.R * g.Nh, total = 2u * per_colour;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour;
        const uint32_t r = rem / g.Nh, j = rem - r * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        uint32_t bit = 0u;
        if (mode == 1) {
            uint32_t w[4];
            const uint32_t ig = i + g.i_off;   // global site index (slab decomposition)
            philox4x32_10(ig >> 7, r, 0u, make_tag(0u, DOM_INIT, 0u), a.keys, w);
            bit = (w[(ig >> 5) & 3u] >> (ig & 31u)) & 1u;
        } else if (mode == 2) {
            // canonical arrays hold the owned sites only (ghost planes of a slab keep what the halo exchange wrote)
            const uint32_t io = i - g.own_i0;
            if (io < g.own_in) bit = canon[(size_t)r * g.own_in + io] < 0 ? 1u : 0u;
            else if (a.bitpack) bit = (((const uint32_t *)(c ? s1 : s0))[(size_t)r * g.NW + (j >> 5)] >> (j & 31u)) & 1u;
            else bit = ((const uint8_t *)(c ? s1 : s0))[(size_t)r * g.Nh + int8_byte_index(a, j)];
        }
        void *dst = c ? s1 : s0;
        if (a.bitpack) {
            const uint32_t word = __ballot_sync(0xFFFFFFFFu, bit);
            if ((threadIdx.x & 31) == 0) ((uint32_t *)dst)[(size_t)r * g.NW + (j >> 5)] = word;
        } else {
            ((uint8_t *)dst)[(size_t)r * g.Nh + int8_byte_index(a, j)] = (uint8_t)bit;
        }
    }
}

// Canonical BIT arrays (n = 1; spin_set_spins_bits / spin_get_spins_bits): bit (i & 7) of byte (r N + i) >> 3 is 1 iff spin i of
// replica r is -1 -- an eighth of the int8 canonical array over PCIe, and every bit pattern is a valid configuration (no check).
// A thread converts 8 consecutive canonical sites (one byte): 4 of each colour.  Whole-lattice handles only (Lx % 8 == 0).
__global__ void __launch_bounds__(256) ising_bits_convert(const __grid_constant__ SetupArgs a, uint8_t *bits, void *s0, void *s1, bool to_arrays) {
    const Geometry &g = a.g;
    const uint32_t N = 2u * g.Nh, nbytes = a.R * (N >> 3);
    for (uint32_t b = blockIdx.x * blockDim.x + threadIdx.x; b < nbytes; b += gridDim.x * blockDim.x) {
        const uint32_t r = b / (N >> 3), i0 = (b - r * (N >> 3)) << 3;       // 8 sites of one row: Lx % 8 == 0
        const uint32_t row = i0 / (uint32_t)g.Lx, x0 = i0 - row * (uint32_t)g.Lx;
        const uint32_t z = fdiv(row, g.divLy), y = row - z * (uint32_t)g.Ly;
        uint32_t v = to_arrays ? bits[b] : 0u;
#pragma unroll
        for (uint32_t k = 0; k < 8u; ++k) {
            const uint32_t x = x0 + k, c = (x + y + z) & 1u, j = (x >> 1) + g.RL * row;
            void *arr = c ? s1 : s0;
            if (a.bitpack) {
                uint32_t *wp = (uint32_t *)arr + (size_t)r * g.NW + (j >> 5);
                if (to_arrays) { if ((v >> k) & 1u) atomicOr(wp, 1u << (j & 31u)); }
                else v |= ((*wp >> (j & 31u)) & 1u) << k;
            } else {
                uint8_t *bp = (uint8_t *)arr + (size_t)r * g.Nh + int8_byte_index(a, j);
                if (to_arrays) *bp = (uint8_t)((v >> k) & 1u); else v |= (uint32_t)(*bp & 1u) << k;
            }
        }
        if (!to_arrays) bits[b] = (uint8_t)v;
    }
}

// *bad = 1 if any byte of canon[0 .. n) is not +1 or -1
__global__ void __launch_bounds__(256) ising_validate_canonical(const int8_t *canon, size_t n, int *bad) {
    int local = 0;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
        const int v = canon[k];
        local |= (v != 1 && v != -1);
    }
    if (local) *bad = 1;
}

__global__ void __launch_bounds__(256) ising_to_canonical(const __grid_constant__ SetupArgs a, const void *s0, const void *s1,
                                                          int8_t *canon) {
    const Geometry &g = a.g;
    const uint32_t per_colour = a.R * g.Nh, total = 2u * per_colour;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour;
        const uint32_t r = rem / g.Nh, j = rem - r * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        const void *src = c ? s1 : s0;
        uint32_t bit;
        if (a.bitpack) bit = (((const uint32_t *)src)[(size_t)r * g.NW + (j >> 5)] >> (j & 31u)) & 1u;
        else bit = ((const uint8_t *)src)[(size_t)r * g.Nh + int8_byte_index(a, j)];
        const uint32_t io = i - g.own_i0;
        if (io < g.own_in) canon[(size_t)r * g.own_in + io] = bit ? (int8_t)-1 : (int8_t)1;
    }
}

// mode 0: cold, 1: hot, 2: from canonical float [R][N][nc]
template <int NC>
__global__ void __launch_bounds__(256) vector_fill(const __grid_constant__ SetupArgs a, int mode, const float *canon,
                                                   float *s0, float *s1) {
    const Geometry &g = a.g;
    const uint32_t per_colour = a.R * g.Nh, total = 2u * per_colour;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour;
        const uint32_t r = rem / g.Nh, j = rem - r * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        float v[3] = {0.0f, 0.0f, 0.0f};
        if (mode == 0) {
            if (NC == 3) v[2] = 1.0f; else v[0] = 1.0f;
        } else if (mode == 1) {
            uint32_t w[4];
            philox4x32_10(i + g.i_off, r, 0u, make_tag(0u, DOM_INIT, 0u), a.keys, w);
            if (NC == 3) direction3(w[0], w[1], v); else direction2(w[0], v);
        } else {
            const uint32_t io = i - g.own_i0;
            if (io >= g.own_in) continue;   // ghost planes keep what the halo exchange wrote
#pragma unroll
            for (int k = 0; k < NC; ++k) v[k] = canon[((size_t)r * g.own_in + io) * NC + k];
        }
        float *dst = (c ? s1 : s0) + (size_t)r * NC * g.Nh;
#pragma unroll
        for (int k = 0; k < NC; ++k) dst[(size_t)k * g.Nh + j] = v[k];
    }
}

template <int NC>
__global__ void __launch_bounds__(256) vector_to_canonical(const __grid_constant__ SetupArgs a, const float *s0, const float *s1,
                                                           float *canon) {
    const Geometry &g = a.g;
    const uint32_t per_colour = a.R * g.Nh, total = 2u * per_colour;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour;
        const uint32_t r = rem / g.Nh, j = rem - r * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        const float *src = (c ? s1 : s0) + (size_t)r * NC * g.Nh;
        const uint32_t io = i - g.own_i0;
        if (io >= g.own_in) continue;
#pragma unroll
        for (int k = 0; k < NC; ++k) canon[((size_t)r * g.own_in + io) * NC + k] = src[(size_t)k * g.Nh + j];
    }
}

// Canonical int8 bonds [R][d][N] drawn from the seed (generic kernels keep this layout).
__global__ void __launch_bounds__(256) bonds_draw_canonical(const __grid_constant__ SetupArgs a, int8_t *canon) {
    const Geometry &g = a.g;
    const uint32_t N = 2u * g.Nh, total = a.R * N;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t r = idx / N, i = idx - r * N;
        uint32_t w[4];
        philox4x32_10(i >> 5, r, 0u, make_tag(0u, DOM_BONDS, 0u), a.keys, w);
        for (int mu = 0; mu < g.d; ++mu)
            canon[((size_t)r * g.d + mu) * N + i] = ((w[mu] >> (i & 31u)) & 1u) ? (int8_t)-1 : (int8_t)1;
    }
}

// Bit planes bb[colour][r][3][NW] (bit = 1: J = -1) from the seed (canon == NULL) or a canonical array.
__global__ void __launch_bounds__(256) bonds_pack(const __grid_constant__ SetupArgs a, const int8_t *canon, uint32_t *bb) {
    const Geometry &g = a.g;
    const uint32_t per_colour = a.R * g.Nh, total = 2u * per_colour, N = 2u * g.Nh;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour;
        const uint32_t r = rem / g.Nh, j = rem - r * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        uint32_t w[4] = {0u, 0u, 0u, 0u};
        if (canon == nullptr) philox4x32_10(i >> 5, r, 0u, make_tag(0u, DOM_BONDS, 0u), a.keys, w);
        for (int mu = 0; mu < 3; ++mu) {
            uint32_t bit = 0u;
            if (mu < g.d) bit = canon ? (canon[((size_t)r * g.d + mu) * N + i] < 0 ? 1u : 0u) : ((w[mu] >> (i & 31u)) & 1u);
            const uint32_t word = __ballot_sync(0xFFFFFFFFu, bit);
            if ((threadIdx.x & 31) == 0) bb[((size_t)(c * a.R + r) * 3 + mu) * g.NW + (j >> 5)] = word;
        }
    }
}

__global__ void __launch_bounds__(256) bonds_unpack(const __grid_constant__ SetupArgs a, const uint32_t *bb, int8_t *canon) {
    const Geometry &g = a.g;
    const uint32_t per_colour = a.R * g.Nh, total = 2u * per_colour, N = 2u * g.Nh;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t c = idx / per_colour, rem = idx - c * per_colour;
        const uint32_t r = rem / g.Nh, j = rem - r * g.Nh;
        const uint32_t i = lex_index(g, c, j);
        for (int mu = 0; mu < g.d; ++mu) {
            const uint32_t bit = (bb[((size_t)(c * a.R + r) * 3 + mu) * g.NW + (j >> 5)] >> (j & 31u)) & 1u;
            canon[((size_t)r * g.d + mu) * N + i] = bit ? (int8_t)-1 : (int8_t)1;
        }
    }
}

// Halo faces of a slab handle: `rows` pieces of `plane_elems` elements each, piece q of face f at
// arr + plane[f] * plane_elems + q * stride_elems in the colour array and at buf + (f * rows + q) * plane_elems in the message
// buffer.  pack = true: array -> buffer (the two owned boundary planes), false: buffer -> array (the two ghost planes).
// One launch for both faces (four cudaMemcpy2DAsync per exchange before: 16 us of launch latency per half-sweep).
template <typename T>
__global__ void __launch_bounds__(256) halo_faces_copy(T *arr, T *buf, size_t plane_elems, size_t stride_elems, uint32_t rows,
                                                       uint32_t plane_lo, uint32_t plane_hi, bool pack) {
    const size_t per_face = plane_elems * rows, total = 2 * per_face;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t f = i / per_face, rem = i - f * per_face, q = rem / plane_elems, e = rem - q * plane_elems;
        T *a = arr + (f ? plane_hi : plane_lo) * plane_elems + q * stride_elems + e;
        if (pack) buf[i] = *a; else *a = buf[i];
    }
}

// Peer stores ("direct peer stores over NVLink 5 / NVSwitch"): my two owned boundary planes go straight into the ghost
// planes of the two neighbour slabs' colour arrays -- below: its ghost above its owned planes (plane own + 2), above: its ghost
// below (plane 1).  dst_below / dst_above are device pointers to the neighbours' colour arrays of the same layout and slab
// thickness, valid on this device (the same device, or peer-mapped memory of another GPU).  One kernel, no message buffer.
template <typename T>
__global__ void __launch_bounds__(256) halo_faces_push(const T *src, T *dst_below, T *dst_above, size_t plane_elems, size_t stride_elems,
                                                       uint32_t rows, uint32_t own) {
    const size_t per_face = plane_elems * rows, total = 2 * per_face;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t f = i / per_face, rem = i - f * per_face, q = rem / plane_elems, e = rem - q * plane_elems;
        const size_t off = q * stride_elems + e;
        if (f == 0) dst_below[(own + 2u) * plane_elems + off] = src[2u * plane_elems + off];      // my lowest plane -> its upper ghost
        else dst_above[1u * plane_elems + off] = src[(own + 1u) * plane_elems + off];             // my highest plane -> its lower ghost
    }
}

// a single slab that is its own neighbour (one rank, periodic): ghost below <- highest owned plane, ghost above <- lowest
template <typename T>
__global__ void __launch_bounds__(256) halo_faces_wrap(T *arr, size_t plane_elems, size_t stride_elems, uint32_t rows, uint32_t own) {
    const size_t per_face = plane_elems * rows, total = 2 * per_face;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t f = i / per_face, rem = i - f * per_face, q = rem / plane_elems, e = rem - q * plane_elems;
        const size_t src = f ? 2u : own + 1u, dst = f ? own + 2u : 1u;
        arr[dst * plane_elems + q * stride_elems + e] = arr[src * plane_elems + q * stride_elems + e];
    }
}

}  // namespace spin
