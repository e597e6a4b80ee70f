// vector_kernels.cuh -- n = 2 (XY) and n = 3 (Heisenberg) half-sweep: fp32 unit vectors stored as one
// plane per component and colour, one thread per site.  PAPER.md:31-38 (Eq. (1), (2))
// (fp32 spins, special functions).  Proposal = a fresh uniform direction (R-11, R-12):
//   z = 2 u24(w0) - 1, rho = sqrt(max(0, 1 - z z)), phi = 2 pi u24(w1), s' = (rho cos phi, rho sin phi, z)
//   n = 2: s' = (cos 2 pi u24(w0), sin 2 pi u24(w0))
// Local field h = sum_nbrs J s_j in the order -x, +x, -y, +y, -z, +z, dE = -(s' - s) . h, accept iff
// dE <= 0 or u24(w_acc) < expf(-beta dE).  The sums use explicitly rounded fp32 operations in the
// order DESIGN.md fixes (no FMA contraction), so only sincospi_u24 / expf can differ from the oracle.
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
    uint32_t rule;        // 0 Metropolis (Eq. (2)), 1 heat bath (n = 3 only)
};

__device__ __forceinline__ float u24(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-08f; }
// 2 u24(w): the product by 2 is exact, so one multiplication by 2^-23 gives the same float
__device__ __forceinline__ float two_u24(uint32_t w) { return (float)(w >> 8) * 1.1920928955078125e-07f; }

// sin(pi x), cos(pi x) for x = 2 u24(w) = k 2^-23, k = w >> 8 < 2^24 (R-12).  The argument is an integer, so the range
// reduction is exact integer arithmetic: q = round(2 x) in 0 .. 4, r = x - q / 2 = (k - q 2^22) 2^-23 in [-1/4, 1/4];
// then two polynomials in r^2 (least-squares fits on Chebyshev nodes, reweighted towards minimax; checked over all
// 2^22 + 1 values of r: sin within 1.7 ulp, cos within 1.0 ulp, absolute error below 9e-8) and the quadrant symmetries
// q = 0: (s, c), 1: (c, -s), 2: (-s, -c), 3: (-c, s).  About 10 instructions fewer than sincospif, which must also
// serve arbitrary floats.
__device__ __forceinline__ void sincospi_u24(uint32_t w, float *sn, float *cs) {
    const uint32_t k = w >> 8;
    const uint32_t q = (k + (1u << 21)) >> 22;
    const float r = (float)(int)(k - (q << 22)) * 1.1920928955078125e-07f;
    const float u = r * r;
    float ps = fmaf(-0.589078654592815f, u, 2.5497672980581947f);
    ps = fmaf(ps, u, -5.167707829131533f);
    ps = fmaf(ps, u, 3.1415926439336053f);
    const float sr = ps * r;
    float cr = fmaf(0.2313297165900991f, u, -1.3350445644556512f);
    cr = fmaf(cr, u, 4.058707263029904f);
    cr = fmaf(cr, u, -4.934802162589503f);
    cr = fmaf(cr, u, 1.0f);
    const float a = (q & 1u) ? cr : sr, b = (q & 1u) ? sr : cr;
    *sn = __uint_as_float(__float_as_uint(a) ^ ((q & 2u) << 30));
    *cs = __uint_as_float(__float_as_uint(b) ^ (((q + 1u) & 2u) << 30));
}

__device__ __forceinline__ void direction3(uint32_t w0, uint32_t w1, float out[3]) {
    const float z = __fsub_rn(two_u24(w0), 1.0f);  // exact: (k - 2^23) 2^-23 with k < 2^24
    const float om = fmaxf(__fsub_rn(1.0f, __fmul_rn(z, z)), 0.0f);
    const float rho = __fsqrt_rn(om);
    float sn, cs;
    sincospi_u24(w1, &sn, &cs);
    out[0] = __fmul_rn(rho, cs);
    out[1] = __fmul_rn(rho, sn);
    out[2] = z;
}

__device__ __forceinline__ void direction2(uint32_t w0, float out[2]) {
    float sn, cs;
    sincospi_u24(w0, &sn, &cs);
    out[0] = cs;
    out[1] = sn;
}

// Heat bath for n = 3: the new spin is drawn from exp(beta s.h) on the sphere.
// With H = beta |h| the cosine about h is c = 1 + ln(1 - u (1 - e^{-2H})) / H (inversion of its distribution
// function), the azimuth is uniform, and the frame is hhat plus the branch-free orthonormal pair of Duff et al.
// Every fp32 operation is rounded separately, in the order the oracle states them; only expf, logf and sincospi_u24
// can differ from its double-evaluated, once-rounded values.
__device__ __forceinline__ void heatbath3(float beta, const float h[3], uint32_t w0, uint32_t w1, float out[3]) {
    const float hh = __fadd_rn(__fadd_rn(__fmul_rn(h[0], h[0]), __fmul_rn(h[1], h[1])), __fmul_rn(h[2], h[2]));
    const float hn = __fsqrt_rn(hh);
    const float H = __fmul_rn(beta, hn);
    if (!(H > 0.0f)) { direction3(w0, w1, out); return; }
    const float u = u24(w0);
    const float e2H = expf(__fmul_rn(-2.0f, H));
    const float arg = __fsub_rn(1.0f, __fmul_rn(u, __fsub_rn(1.0f, e2H)));
    float c = __fadd_rn(1.0f, __fdiv_rn(logf(arg), H));
    c = fminf(fmaxf(c, -1.0f), 1.0f);
    const float st = __fsqrt_rn(fmaxf(__fsub_rn(1.0f, __fmul_rn(c, c)), 0.0f));
    float sp, cp;
    sincospi_u24(w1, &sp, &cp);
    const float inv = __fdiv_rn(1.0f, hn);
    const float x = __fmul_rn(h[0], inv), y = __fmul_rn(h[1], inv), z = __fmul_rn(h[2], inv);
    const float sg = signbit(z) ? -1.0f : 1.0f;
    const float a = __fdiv_rn(-1.0f, __fadd_rn(sg, z));
    const float b = __fmul_rn(__fmul_rn(x, y), a);
    const float e1[3] = {__fadd_rn(1.0f, __fmul_rn(__fmul_rn(sg, __fmul_rn(x, x)), a)), __fmul_rn(sg, b), __fmul_rn(-sg, x)};
    const float e2[3] = {b, __fadd_rn(sg, __fmul_rn(__fmul_rn(y, y), a)), -y};
    const float fa = __fmul_rn(st, cp), fb = __fmul_rn(st, sp);
    const float hk[3] = {x, y, z};
#pragma unroll
    for (int k = 0; k < 3; ++k)
        out[k] = __fadd_rn(__fadd_rn(__fmul_rn(fa, e1[k]), __fmul_rn(fb, e2[k])), __fmul_rn(c, hk[k]));
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
        philox4x32_10(j + g.j_off, a.replica_streams ? r : 0u, a.t, make_tag(a.colour, DOM_VECTOR_UPDATE, 0), a.keys, w);
        float sn[NC];
        uint32_t wacc;
        if (NC == 3 && a.rule != 0u) {
            float h3[3] = {h[0], h[1], h[NC - 1]}, s3[3];
            heatbath3(a.beta, h3, w[0], w[1], s3);
#pragma unroll
            for (int c = 0; c < NC; ++c) mine[(size_t)c * g.Nh + j] = s3[c];
            continue;
        }
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

// ---------------------------------------------------------------------------------------------
// Strip kernel (Lx % 8 == 0): one thread owns a quad of 4 consecutive same-colour sites (one 128-bit word per
// component plane) and walks K consecutive rows y, rolling the other colour's rows y-1, y, y+1 through
// registers: every access is a coalesced 128-bit load or store, each other-colour row is loaded (K + 2) / K
// times, and the index arithmetic is paid once per strip.  Same arithmetic, in the same order, as
// vector_halfsweep: the result is bit-identical to it for any K and launch shape.
//   UNITJ: every coupling in use is exactly +1, so J * s is s (exact) and the products are skipped.
template <int NC>
struct Quad {
    float4 c[NC];
};

template <int NC>
__device__ __forceinline__ Quad<NC> load_quad(const float *__restrict__ base, uint32_t Nh, uint32_t off) {
    Quad<NC> q;
#pragma unroll
    for (int c = 0; c < NC; ++c) q.c[c] = __ldg((const float4 *)(base + (size_t)c * Nh + off));
    return q;
}

__device__ __forceinline__ float lane_of(const float4 &v, int i) { return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w)); }

template <bool UNITJ>
__device__ __forceinline__ float add_nb(float h, float J, float s) {
    return UNITJ ? __fadd_rn(h, s) : __fadd_rn(h, __fmul_rn(J, s));
}

template <int NC, int D, bool UNITJ, int K, bool HB = false>
__global__ void __launch_bounds__(128) vector_strip_halfsweep(const __grid_constant__ VectorArgs a) {
    const Geometry &g = a.g;
    const uint32_t RL = g.RL, QX = RL >> 2, Ly = (uint32_t)g.Ly, Lz = (uint32_t)g.Lz, Nh = g.Nh;
    const uint32_t nstrip = (Ly + K - 1) / K;
    const uint32_t per_replica = QX * nstrip * Lz;
    // the replica is blockIdx.y (host: gridDim.y = R), so the plane base pointers are warp-uniform and every access is
    // "uniform 64-bit base + 32-bit offset" (no per-thread 64-bit address arithmetic)
    const uint32_t it = blockIdx.x * blockDim.x + threadIdx.x;
    if (it >= per_replica) return;
    const uint32_t r = blockIdx.y;
    const uint32_t sz = fdiv(it, g.divQX), q = it - sz * QX;       // sz = strip + nstrip * z
    const uint32_t z = sz / nstrip, y0 = (sz - z * nstrip) * K;
    const uint32_t kend = min((uint32_t)K, Ly - y0);
    const float *__restrict__ other = a.s[1 - a.colour] + (size_t)r * NC * Nh;
    float *mine = a.s[a.colour] + (size_t)r * NC * Nh;
    const uint32_t rho = a.replica_streams ? r : 0u;
    const uint32_t tag = make_tag(a.colour, DOM_VECTOR_UPDATE, 0);
    const uint32_t plane = RL * Ly, zoff = z * plane;
    const uint32_t zm_off = (D == 3) ? (z == 0 ? Lz - 1 : z - 1) * plane : 0u;
    const uint32_t zp_off = (D == 3) ? (z == Lz - 1 ? 0u : z + 1) * plane : 0u;
    const uint32_t x4 = 4u * q;
    // position, inside a row, of the one x-neighbour outside this quad: p = 1 -> first site of the next quad,
    // p = 0 -> last site of the previous quad (periodic)
    const uint32_t side_p1 = q + 1 == QX ? 0u : x4 + 4u, side_p0 = q == 0 ? RL - 1u : x4 - 1u;
    const float Jx = a.Jdir[0], Jy = a.Jdir[1], Jz = a.Jdir[2];
    const uint32_t ym0 = y0 == 0 ? Ly - 1 : y0 - 1;
    Quad<NC> o_prev = load_quad<NC>(other, Nh, zoff + ym0 * RL + x4);
    Quad<NC> o_cur = load_quad<NC>(other, Nh, zoff + y0 * RL + x4);
    uint32_t p = (y0 + z + a.colour) & 1u;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        if ((uint32_t)k < kend) {
            const uint32_t y = y0 + k;
            const uint32_t yp = y + 1 == Ly ? 0u : y + 1;
            const uint32_t row = zoff + y * RL, off = row + x4;
            const Quad<NC> o_next = load_quad<NC>(other, Nh, zoff + yp * RL + x4);
            Quad<NC> own;
#pragma unroll
            for (int c = 0; c < NC; ++c) own.c[c] = *(const float4 *)(mine + (size_t)c * Nh + off);
            Quad<NC> o_zm, o_zp;
            if (D == 3) {
                o_zm = load_quad<NC>(other, Nh, zm_off + y * RL + x4);
                o_zp = load_quad<NC>(other, Nh, zp_off + y * RL + x4);
            }
            float side[NC];
#pragma unroll
            for (int c = 0; c < NC; ++c) side[c] = __ldg(other + (size_t)c * Nh + row + (p ? side_p1 : side_p0));
            // local field, order -x, +x, -y, +y, -z, +z, every product and sum rounded separately
            float h[4][NC];
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                // the two x-neighbours are o (same compressed index) and sh (index + 1 if p, index - 1 if not); the
                // first sum J x(-x) + J x(+x) is commutative, so which of the two is "-x" does not matter
                const float4 o = o_cur.c[c];
                const float4 sh = p ? make_float4(o.y, o.z, o.w, side[c]) : make_float4(side[c], o.x, o.y, o.z);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    float v = UNITJ ? __fadd_rn(lane_of(o, i), lane_of(sh, i))
                                    : __fadd_rn(__fmul_rn(Jx, lane_of(o, i)), __fmul_rn(Jx, lane_of(sh, i)));
                    v = add_nb<UNITJ>(v, Jy, lane_of(o_prev.c[c], i));
                    v = add_nb<UNITJ>(v, Jy, lane_of(o_next.c[c], i));
                    if (D == 3) {
                        v = add_nb<UNITJ>(v, Jz, lane_of(o_zm.c[c], i));
                        v = add_nb<UNITJ>(v, Jz, lane_of(o_zp.c[c], i));
                    }
                    h[i][c] = v;
                }
            }
            float res[NC][4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                uint32_t w[4];
                philox4x32_10(off + i + g.j_off, rho, a.t, tag, a.keys, w);
                float sn[NC], so[NC];
                uint32_t wacc;
                if (HB && NC == 3) {
                    float h3[3] = {h[i][0], h[i][1], h[i][NC - 1]}, s3[3];
                    heatbath3(a.beta, h3, w[0], w[1], s3);
#pragma unroll
                    for (int c = 0; c < NC; ++c) res[c][i] = s3[c];
                    continue;
                }
                if (NC == 3) { direction3(w[0], w[1], sn); wacc = w[2]; }
                else { direction2(w[0], sn); wacc = w[1]; }
#pragma unroll
                for (int c = 0; c < NC; ++c) so[c] = lane_of(own.c[c], i);
                float acc = __fmul_rn(__fsub_rn(sn[0], so[0]), h[i][0]);
#pragma unroll
                for (int c = 1; c < NC; ++c) acc = __fadd_rn(acc, __fmul_rn(__fsub_rn(sn[c], so[c]), h[i][c]));
                const float dE = -acc;
                const bool accept = dE <= 0.0f || u24(wacc) < expf(__fmul_rn(-a.beta, dE));
#pragma unroll
                for (int c = 0; c < NC; ++c) res[c][i] = accept ? sn[c] : so[c];
            }
#pragma unroll
            for (int c = 0; c < NC; ++c)
                *(float4 *)(mine + (size_t)c * Nh + off) = make_float4(res[c][0], res[c][1], res[c][2], res[c][3]);
            o_prev = o_cur;
            o_cur = o_next;
            p ^= 1u;
        }
    }
}

}  // namespace spin
