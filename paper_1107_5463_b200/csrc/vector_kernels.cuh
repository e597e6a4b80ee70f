// vector_kernels.cuh -- n = 2 (XY) and n = 3 (Heisenberg) half-sweep: fp32 unit vectors stored as one
// plane per component and colour, one thread per site.  PAPER.md:31-38 (Eq. (1), (2))
// (fp32 spins, special functions).  Proposal = a fresh uniform direction (R-11, R-12):
//   z = 2 u24(w0) - 1, rho = sqrt(max(0, 1 - z z)), phi = 2 pi u24(w1), s' = (rho cos phi, rho sin phi, z)
//   n = 2: s' = (cos 2 pi u24(w0), sin 2 pi u24(w0))
// Local field h = sum_nbrs J s_j in the order -x, +x, -y, +y, -z, +z, dE = -(s' - s) . h, accept iff
// dE <= 0 or u24(w_acc) < expf(-beta dE).  The sums use explicitly rounded fp32 operations in the
// order DESIGN.md fixes (no FMA contraction), so only sincospif / expf can differ from the oracle.
#pragma once
#include "common.cuh"

namespace spin {

struct VectorArgs {
    Geometry g;
    PhiloxKeys keys;
    float *s[2];          // per colour: float [R][NC][Nh]
    uint32_t R, replica_streams, t, colour;
    float Jdir[3];
    float beta;
};

__device__ __forceinline__ float u24(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-08f; }

__device__ __forceinline__ void direction3(uint32_t w0, uint32_t w1, float out[3]) {
    const float z = __fsub_rn(__fmul_rn(2.0f, u24(w0)), 1.0f);
    const float om = fmaxf(__fsub_rn(1.0f, __fmul_rn(z, z)), 0.0f);
    const float rho = __fsqrt_rn(om);
    float sn, cs;
    sincospif(__fmul_rn(2.0f, u24(w1)), &sn, &cs);
    out[0] = __fmul_rn(rho, cs);
    out[1] = __fmul_rn(rho, sn);
    out[2] = z;
}

__device__ __forceinline__ void direction2(uint32_t w0, float out[2]) {
    float sn, cs;
    sincospif(__fmul_rn(2.0f, u24(w0)), &sn, &cs);
    out[0] = cs;
    out[1] = sn;
}

// neighbour indices (compressed, other colour) of site j of colour `colour`, order -x,+x,-y,+y,-z,+z
__device__ __forceinline__ void neighbour_indices(const Geometry &g, uint32_t colour, uint32_t j, uint32_t nb[6]) {
    const uint32_t row = fdiv(j, g.divRL), xh = j - row * g.RL;
    const uint32_t z = fdiv(row, g.divLy), y = row - z * (uint32_t)g.Ly;
    const uint32_t p = (y + z + colour) & 1u;
    const uint32_t xs = p ? (xh + 1 == g.RL ? 0 : xh + 1) : (xh == 0 ? g.RL - 1 : xh - 1);
    const uint32_t jside = row * g.RL + xs;
    nb[0] = p ? j : jside;
    nb[1] = p ? jside : j;
    nb[2] = y == 0 ? j + g.RL * (g.Ly - 1) : j - g.RL;
    nb[3] = y == (uint32_t)g.Ly - 1 ? j - g.RL * (g.Ly - 1) : j + g.RL;
    const uint32_t plane = g.RL * g.Ly;
    nb[4] = z == 0 ? j + plane * (g.Lz - 1) : j - plane;
    nb[5] = z == (uint32_t)g.Lz - 1 ? j - plane * (g.Lz - 1) : j + plane;
}

template <int NC>
__global__ void __launch_bounds__(256) vector_halfsweep(const __grid_constant__ VectorArgs a) {
    const Geometry &g = a.g;
    const uint32_t total = g.Nh * a.R;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t r = idx / g.Nh, j = idx - r * g.Nh;
        const float *__restrict__ other = a.s[1 - a.colour] + (size_t)r * NC * g.Nh;
        float *mine = a.s[a.colour] + (size_t)r * NC * g.Nh;
        uint32_t nb[6];
        neighbour_indices(g, a.colour, j, nb);
        float h[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) h[c] = 0.0f;
        const int q = 2 * g.d;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            if (k < q) {
                const float J = a.Jdir[k >> 1];
#pragma unroll
                for (int c = 0; c < NC; ++c) h[c] = __fadd_rn(h[c], __fmul_rn(J, __ldg(other + (size_t)c * g.Nh + nb[k])));
            }
        }
        uint32_t w[4];
        philox4x32_10(j, a.replica_streams ? r : 0u, a.t, make_tag(a.colour, DOM_VECTOR_UPDATE, 0), a.keys, w);
        float sn[NC];
        uint32_t wacc;
        if (NC == 3) { direction3(w[0], w[1], sn); wacc = w[2]; }
        else { direction2(w[0], sn); wacc = w[1]; }
        float so[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) so[c] = mine[(size_t)c * g.Nh + j];
        float acc = __fmul_rn(__fsub_rn(sn[0], so[0]), h[0]);
#pragma unroll
        for (int c = 1; c < NC; ++c) acc = __fadd_rn(acc, __fmul_rn(__fsub_rn(sn[c], so[c]), h[c]));
        const float dE = -acc;
        bool accept = dE <= 0.0f;
        if (!accept) accept = u24(wacc) < expf(__fmul_rn(-a.beta, dE));
        if (accept) {
#pragma unroll
            for (int c = 0; c < NC; ++c) mine[(size_t)c * g.Nh + j] = sn[c];
        }
    }
}

}  // namespace spin
