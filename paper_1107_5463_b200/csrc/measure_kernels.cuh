// measure_kernels.cuh -- energy and magnetisation sums (Eq. (1); "aggregate
// quantities such as the total energy are calculated in double precision").
// Every bond joins the two colours, so E = -sum_{i in colour 1} s_i . h_i with h_i the local field over
// all 2d neighbours counts each bond exactly once; M sums both colours.
//   n = 1 : exact int64 sums (warp shuffle -> shared -> one 64-bit atomic per CTA and quantity)
//   n >= 2: fp64 per-CTA partials, summed in a fixed order by the finalize kernel (deterministic)
#pragma once
#include "ising_int8_kernel.cuh"
#include "ising_kernels.cuh"
#include "vector_kernels.cuh"

namespace spin {

template <typename T>
__device__ __forceinline__ T block_sum(T v, T *smem /* >= 32 */) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xFFFFFFFFu, v, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) smem[wid] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? smem[threadIdx.x] : T(0);
    if (wid == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xFFFFFFFFu, v, o);
    }
    return v;  // valid in thread 0
}

// a.acc[slot][r][0] += E, [1] += M for int8 storage (any dims / couplings).  grid = (blocks, R).
__global__ void __launch_bounds__(256) ising_generic_measure(const __grid_constant__ IsingArgs a) {
    __shared__ long long sm[32];
    const Geometry &g = a.g;
    const uint32_t r = blockIdx.y;
    const uint8_t *__restrict__ s0 = (const uint8_t *)a.s[0] + (size_t)r * g.Nh;
    const uint8_t *__restrict__ s1 = (const uint8_t *)a.s[1] + (size_t)r * g.Nh;
    const int8_t *__restrict__ bonds = (const int8_t *)a.bonds;
    const uint32_t N = 2u * g.Nh;
    long long e = 0, m = 0;
    for (uint32_t j = g.own_j0 + blockIdx.x * blockDim.x + threadIdx.x; j < g.own_j1; j += gridDim.x * blockDim.x) {
        const uint32_t row = fdiv(j, g.divRL), xh = j - row * g.RL;
        const uint32_t z = fdiv(row, g.divLy), y = row - z * (uint32_t)g.Ly;
        const uint32_t p = (y + z + 1u) & 1u;  // colour-1 site
        const uint32_t x = 2u * xh + p;
        const uint32_t xm = x == 0 ? g.Lx - 1 : x - 1, xp = x == (uint32_t)g.Lx - 1 ? 0 : x + 1;
        const uint32_t ym = y == 0 ? g.Ly - 1 : y - 1, yp = y == (uint32_t)g.Ly - 1 ? 0 : y + 1;
        const uint32_t zm = z == 0 ? g.Lz - 1 : z - 1, zp = z == (uint32_t)g.Lz - 1 ? 0 : z + 1;
        int nb[6];
        uint32_t isite[6];
        nb[0] = s0[row * g.RL + (xm >> 1)];            isite[0] = xm + g.Lx * row;
        nb[1] = s0[row * g.RL + (xp >> 1)];            isite[1] = x + g.Lx * row;
        nb[2] = s0[(ym + g.Ly * z) * g.RL + xh];       isite[2] = x + g.Lx * (ym + g.Ly * z);
        nb[3] = s0[(yp + g.Ly * z) * g.RL + xh];       isite[3] = x + g.Lx * row;
        if (g.d == 3) {
            nb[4] = s0[(y + g.Ly * zm) * g.RL + xh];   isite[4] = x + g.Lx * (y + g.Ly * zm);
            nb[5] = s0[(y + g.Ly * zp) * g.RL + xh];   isite[5] = x + g.Lx * row;
        }
        const int s = 1 - 2 * (int)s1[j];
        int h = 0;
        for (int k = 0; k < 2 * g.d; ++k) {
            const int mu = k >> 1;
            const int J = a.coupling_kind == 2 ? (int)bonds[((size_t)r * g.d + mu) * N + isite[k]] : a.Jdir[mu];
            h += J * (1 - 2 * nb[k]);
        }
        e -= s * h;
        m += s + (1 - 2 * (int)s0[j]);
    }
    e = block_sum(e, sm);
    m = block_sum(m, sm);
    if (threadIdx.x == 0) acc_add(a, r, e, m);
}

// Bit-packed storage: E = 2 n_unsatisfied - n_bonds, M = N - 2 popcount.  grid = (blocks, R).
template <int D, bool BONDS>
__global__ void __launch_bounds__(256) ising_bitpack_measure(const __grid_constant__ IsingArgs a) {
    __shared__ long long sm[32];
    const uint32_t r = blockIdx.y, NW = a.g.NW;
    const uint32_t *__restrict__ s0 = (const uint32_t *)a.s[0] + (size_t)r * NW;
    long long e = 0, m = 0;
    for (uint32_t gi = (a.g.own_j0 >> 5) + blockIdx.x * blockDim.x + threadIdx.x; gi < (a.g.own_j1 >> 5); gi += gridDim.x * blockDim.x) {
        const WordNbrs n = word_neighbours<D>(a.g, 1u, gi);
        uint32_t av[6];
        const uint32_t raw = unsatisfied_bonds<D, BONDS>(a, 1u, r, gi, n, av);
        int unsat = __popc(av[0]) + __popc(av[1]) + __popc(av[2]) + __popc(av[3]);
        if (D == 3) unsat += __popc(av[4]) + __popc(av[5]);
        e += 2 * unsat - 2 * D * 32;
        m += 64 - 2 * (__popc(raw) + __popc(s0[gi]));
    }
    e = block_sum(e, sm);
    m = block_sum(m, sm);
    if (threadIdx.x == 0) acc_add(a, r, e, m);
}

// int8 fast layout (uniform J = +-1): units packed to lane masks, then as the bit-packed kernel.  grid = (blocks, R).
template <int D>
__global__ void __launch_bounds__(256) ising_int8_measure(const __grid_constant__ IsingArgs a) {
    __shared__ long long sm[32];
    const Geometry &g = a.g;
    const uint32_t r = blockIdx.y;
    const uint8_t *__restrict__ s0 = (const uint8_t *)a.s[0] + (size_t)r * g.Nh;
    const uint8_t *__restrict__ s1 = (const uint8_t *)a.s[1] + (size_t)r * g.Nh;
    const uint32_t jflip = a.jneg ? 0xFFFFFFFFu : 0u;
    long long e = 0, m = 0;
    for (uint32_t gi = (g.own_j0 >> 5) + blockIdx.x * blockDim.x + threadIdx.x; gi < (g.own_j1 >> 5); gi += gridDim.x * blockDim.x) {
        const WordNbrs n = word_neighbours<D>(g, 1u, gi);
        const uint32_t row = fdiv(gi, g.divWX), w = gi - row * g.WX;
        const uint32_t raw = int8_pack_unit(s1 + 32u * (size_t)gi);
        const uint32_t o = int8_pack_unit(s0 + 32u * (size_t)gi);
        const uint32_t side = int8_side_mask(s0 + (size_t)row * g.RL, o, n.p, w, g.WX);
        const uint32_t s = raw ^ jflip;
        int unsat = __popc(s ^ o) + __popc(s ^ side) + __popc(s ^ int8_pack_unit(s0 + 32u * (size_t)n.g_ym)) +
                    __popc(s ^ int8_pack_unit(s0 + 32u * (size_t)n.g_yp));
        if (D == 3)
            unsat += __popc(s ^ int8_pack_unit(s0 + 32u * (size_t)n.g_zm)) + __popc(s ^ int8_pack_unit(s0 + 32u * (size_t)n.g_zp));
        e += 2 * unsat - 2 * D * 32;
        m += 64 - 2 * (__popc(raw) + __popc(o));
    }
    e = block_sum(e, sm);
    m = block_sum(m, sm);
    if (threadIdx.x == 0) acc_add(a, r, e, m);
}

// sum of the slots of acc -> doubles at outE[r], outM[r]; clears acc for the next measurement.  One warp per replica,
// lane k takes slots k, k + 32, ... (integer sums: exact in any order).  block = 128 threads = 4 replicas.
__global__ void __launch_bounds__(128) ising_measure_finalize(long long *acc, uint32_t R, uint32_t slots, double *outE, double *outM) {
    const uint32_t r = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31u;
    if (r >= R) return;
    long long e = 0, m = 0;
    for (uint32_t k = lane; k < slots; k += 32u) {
        longlong2 *p = (longlong2 *)(acc + 2 * ((size_t)k * R + r));
        const longlong2 v = *p;
        e += v.x; m += v.y;
        *p = make_longlong2(0, 0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { e += __shfl_down_sync(0xFFFFFFFFu, e, o); m += __shfl_down_sync(0xFFFFFFFFu, m, o); }
    if (lane == 0u) { outE[r] = (double)e; outM[r] = (double)m; }
}

// n >= 2: part[r][block][1 + NC].  grid = (blocks, R).
template <int NC>
__global__ void __launch_bounds__(256) vector_measure(const __grid_constant__ VectorArgs a, double *part) {
    __shared__ double sm[32];
    const Geometry &g = a.g;
    const uint32_t r = blockIdx.y;
    const float *__restrict__ s0 = a.s[0] + (size_t)r * NC * g.Nh;
    const float *__restrict__ s1 = a.s[1] + (size_t)r * NC * g.Nh;
    double e = 0.0, m[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) m[c] = 0.0;
    const int q = 2 * g.d;
    for (uint32_t j = g.own_j0 + blockIdx.x * blockDim.x + threadIdx.x; j < g.own_j1; j += gridDim.x * blockDim.x) {
        uint32_t nb[6];
        neighbour_indices(g, 1u, j, nb);
        float si[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) { si[c] = s1[(size_t)c * g.Nh + j]; m[c] += (double)si[c] + (double)s0[(size_t)c * g.Nh + j]; }
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            if (k < q) {
                double dot = 0.0;
#pragma unroll
                for (int c = 0; c < NC; ++c) dot += (double)si[c] * (double)s0[(size_t)c * g.Nh + nb[k]];
                e -= (double)a.Jdir[k >> 1] * dot;
            }
        }
    }
    double *out = part + ((size_t)r * gridDim.x + blockIdx.x) * (1 + NC);
    e = block_sum(e, sm);
    if (threadIdx.x == 0) out[0] = e;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const double v = block_sum(m[c], sm);
        if (threadIdx.x == 0) out[1 + c] = v;
    }
}

// Sums the per-CTA partials of replica blockIdx.x in a fixed order.  One CTA of 256 threads per replica.
__global__ void __launch_bounds__(256) vector_measure_finalize(const double *part, uint32_t nblocks, int nc,
                                                               double *outE, double *outM) {
    __shared__ double sm[32];
    const uint32_t r = blockIdx.x;
    for (int k = 0; k < 1 + nc; ++k) {
        double v = 0.0;
        for (uint32_t b = threadIdx.x; b < nblocks; b += blockDim.x) v += part[((size_t)r * nblocks + b) * (1 + nc) + k];
        v = block_sum(v, sm);
        if (threadIdx.x == 0) {
            if (k == 0) outE[r] = v;
            else outM[(size_t)r * nc + (k - 1)] = v;
        }
    }
}

// Two-level, single-launch version for many partials (the fused strip kernel leaves one per warp): grid = (F, R).
// Block (f, r) sums its contiguous share of part[r][0 .. nparts) in a fixed order into mid[r][f]; the block that finishes
// last for replica r (ticket from counter[r]) sums mid[r][0 .. F) in a fixed order.  Which block is last does not change
// any order of summation, so the result is deterministic.
__global__ void __launch_bounds__(256) vector_partials_finalize(const double *part, uint32_t nparts, int nc, double *mid,
                                                                unsigned int *counter, double *outE, double *outM) {
    __shared__ double sm[32];
    __shared__ unsigned int ticket;
    const uint32_t r = blockIdx.y, F = gridDim.x, f = blockIdx.x;
    const uint32_t share = (nparts + F - 1) / F, b0 = f * share, b1 = min(nparts, b0 + share);
    for (int k = 0; k < 1 + nc; ++k) {
        double v = 0.0;
        for (uint32_t b = b0 + threadIdx.x; b < b1; b += blockDim.x) v += part[((size_t)r * nparts + b) * (1 + nc) + k];
        v = block_sum(v, sm);
        if (threadIdx.x == 0) mid[((size_t)r * F + f) * (1 + nc) + k] = v;
    }
    if (threadIdx.x == 0) {
        __threadfence();
        ticket = atomicAdd(&counter[r], 1u);
    }
    __syncthreads();
    if (ticket != F - 1) return;
    __threadfence();
    for (int k = 0; k < 1 + nc; ++k) {
        double v = 0.0;
        for (uint32_t b = threadIdx.x; b < F; b += blockDim.x) v += __ldcg(&mid[((size_t)r * F + b) * (1 + nc) + k]);
        v = block_sum(v, sm);
        if (threadIdx.x == 0) {
            if (k == 0) outE[r] = v;
            else outM[(size_t)r * nc + (k - 1)] = v;
        }
    }
    if (threadIdx.x == 0) counter[r] = 0u;
}

}  // namespace spin
