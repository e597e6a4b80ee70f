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
    uint32_t rho_off;     // added to the replica index in the Philox counter (temperature axis: one launch per replica, R = 1)
    float Jdir[3];
    float beta;
    uint32_t rule;        // 0 Metropolis (Eq. (2)), 1 heat bath (n = 3 only)
    uint32_t prefetch;    // strip kernel: L2 prefetch distance in CTAs (0 = off)
    double *part;         // fused E / M of the strip kernel: [R][warps of the grid][1 + NC] partial sums
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
    const float inv = __frcp_rn(hn);   // = 1 / hn correctly rounded (rcp.rn is the IEEE reciprocal: the bits of __fdiv_rn(1, hn), three instructions fewer)
    const float x = __fmul_rn(h[0], inv), y = __fmul_rn(h[1], inv), z = __fmul_rn(h[2], inv);
    const float sg = signbit(z) ? -1.0f : 1.0f;
    const float a = -__frcp_rn(__fadd_rn(sg, z));   // = -1 / (sg + z): round-to-nearest is symmetric, the negation exact
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
    const uint32_t total = g.sw_jn * a.R;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const uint32_t r = idx / g.sw_jn, j = g.sw_j0 + idx - r * g.sw_jn;
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
        {
            // n = 3 Metropolis: a call per site; updates that take two words (n = 2; heat bath): sites 2k, 2k + 1 of a colour
            // share the call of unit k (words 0, 1 / 2, 3; R-16b)
            const uint32_t jg = j + g.j_off;
            const bool pair = NC == 2 || a.rule != 0u;
            philox4x32_10(pair ? jg >> 1 : jg, a.replica_streams ? r + a.rho_off : 0u, a.t, make_tag(a.colour, DOM_VECTOR_UPDATE, 0), a.keys, w);
            if (pair && (jg & 1u)) { w[0] = w[2]; w[1] = w[3]; }
        }
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

// ---------------------------------------------------------------------------------------------
// Packed fp32 arithmetic (sm_100: add / mul / fma.rn.f32x2 -> FADD2 / FMUL2 / FFMA2, two IEEE operations per issued
// instruction).  Each half of a packed operation is the correctly rounded scalar operation, so a pair of sites computed
// this way carries exactly the bits the one-thread-per-site kernel produces with __fadd_rn / __fmul_rn / fmaf; what is
// saved is issue slots, which is what bounds these kernels (profiles/).
__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 f2s(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
// A product that feeds a sum directly: ptxas contracts mul.rn.f32x2 + add.rn.f32x2 into one FFMA2 (measured: CUDA 12.9,
// sm_100a; the scalar _rn intrinsics are never contracted), which would round once instead of twice.  Two scalar products
// feeding a packed sum are not contracted, so where the contract (R-14) wants product and sum rounded separately
// the product is taken with this helper -- every product of such a sum, the first one included: ptxas contracts whichever packed
// product has the sum as its only use (found by reading the SASS: an FFMA2 in the acceptance sum of the XY kernel).
__device__ __forceinline__ float2 mul2s(float2 a, float2 b) { return make_float2(__fmul_rn(a.x, b.x), __fmul_rn(a.y, b.y)); }

// sincospi_u24 for two sites at once: integer range reduction per site, the two polynomials packed
__device__ __forceinline__ void sincospi_u24_x2(uint32_t wa, uint32_t wb, float2 *sn, float2 *cs) {
    const uint32_t ka = wa >> 8, kb = wb >> 8;
    const uint32_t qa = (ka + (1u << 21)) >> 22, qb = (kb + (1u << 21)) >> 22;
    const float2 r = __fmul2_rn(f2((float)(int)(ka - (qa << 22)), (float)(int)(kb - (qb << 22))), f2s(1.1920928955078125e-07f));
    const float2 u = __fmul2_rn(r, r);
    float2 ps = __ffma2_rn(f2s(-0.589078654592815f), u, f2s(2.5497672980581947f));
    ps = __ffma2_rn(ps, u, f2s(-5.167707829131533f));
    ps = __ffma2_rn(ps, u, f2s(3.1415926439336053f));
    const float2 sr = __fmul2_rn(ps, r);
    float2 cr = __ffma2_rn(f2s(0.2313297165900991f), u, f2s(-1.3350445644556512f));
    cr = __ffma2_rn(cr, u, f2s(4.058707263029904f));
    cr = __ffma2_rn(cr, u, f2s(-4.934802162589503f));
    cr = __ffma2_rn(cr, u, f2s(1.0f));
    const float aa = (qa & 1u) ? cr.x : sr.x, ba = (qa & 1u) ? sr.x : cr.x;
    const float ab = (qb & 1u) ? cr.y : sr.y, bb = (qb & 1u) ? sr.y : cr.y;
    sn->x = __uint_as_float(__float_as_uint(aa) ^ ((qa & 2u) << 30));
    cs->x = __uint_as_float(__float_as_uint(ba) ^ (((qa + 1u) & 2u) << 30));
    sn->y = __uint_as_float(__float_as_uint(ab) ^ ((qb & 2u) << 30));
    cs->y = __uint_as_float(__float_as_uint(bb) ^ (((qb + 1u) & 2u) << 30));
}

// direction3 / direction2 for two sites (site a in .x, site b in .y); out[c] = component c of both
__device__ __forceinline__ void direction3_x2(uint32_t w0a, uint32_t w1a, uint32_t w0b, uint32_t w1b, float2 out[3]) {
    // z = 2 u24(w) - 1 = k 2^-23 - 1 with k < 2^24: product and difference are exact, so one fma gives the same float
    const float2 z = __ffma2_rn(f2((float)(w0a >> 8), (float)(w0b >> 8)), f2s(1.1920928955078125e-07f), f2s(-1.0f));
    const float2 om = __fadd2_rn(f2s(1.0f), neg2(mul2s(z, z)));
    const float2 rho = f2(__fsqrt_rn(fmaxf(om.x, 0.0f)), __fsqrt_rn(fmaxf(om.y, 0.0f)));
    float2 sn, cs;
    sincospi_u24_x2(w1a, w1b, &sn, &cs);
    out[0] = mul2s(rho, cs);   // the proposal feeds the difference s' - s: it must not be contracted into it
    out[1] = mul2s(rho, sn);
    out[2] = z;
}
__device__ __forceinline__ void direction2_x2(uint32_t w0a, uint32_t w0b, float2 out[2]) {
    float2 sn, cs;
    sincospi_u24_x2(w0a, w0b, &sn, &cs);
    out[0] = cs;
    out[1] = sn;
}

// heatbath3 for two sites at once (site a in .x, site b in .y; h[c] = component c of both fields): the plain products and
// sums are packed (each half is the scalar operation of heatbath3, in the same order: bit-identical), the square roots,
// divisions, expf, logf stay scalar.  A zero field (H = 0) falls back to the uniform direction, per site.
__device__ __forceinline__ void heatbath3_x2(float beta, const float2 h[3], uint32_t w0a, uint32_t w1a, uint32_t w0b, uint32_t w1b,
                                             float2 out[3]) {
    const float2 hh = __fadd2_rn(__fadd2_rn(mul2s(h[0], h[0]), mul2s(h[1], h[1])), mul2s(h[2], h[2]));
    const float2 hn = f2(__fsqrt_rn(hh.x), __fsqrt_rn(hh.y));
    const float2 H = __fmul2_rn(f2s(beta), hn);
    const float2 u = __fmul2_rn(f2((float)(w0a >> 8), (float)(w0b >> 8)), f2s(5.9604644775390625e-08f));
    const float2 m2H = __fmul2_rn(f2s(-2.0f), H);
    const float2 e2H = f2(expf(m2H.x), expf(m2H.y));
    const float2 arg = __fadd2_rn(f2s(1.0f), neg2(mul2s(u, __fadd2_rn(f2s(1.0f), neg2(e2H)))));
    float2 c = __fadd2_rn(f2s(1.0f), f2(__fdiv_rn(logf(arg.x), H.x), __fdiv_rn(logf(arg.y), H.y)));
    c = f2(fminf(fmaxf(c.x, -1.0f), 1.0f), fminf(fmaxf(c.y, -1.0f), 1.0f));
    const float2 omc = __fadd2_rn(f2s(1.0f), neg2(mul2s(c, c)));
    const float2 st = f2(__fsqrt_rn(fmaxf(omc.x, 0.0f)), __fsqrt_rn(fmaxf(omc.y, 0.0f)));
    float2 sp, cp;
    sincospi_u24_x2(w1a, w1b, &sp, &cp);
    const float2 inv = f2(__frcp_rn(hn.x), __frcp_rn(hn.y));
    const float2 x = __fmul2_rn(h[0], inv), y = __fmul2_rn(h[1], inv), z = mul2s(h[2], inv);   // z feeds the sum sg + z
    const float2 sg = f2(signbit(z.x) ? -1.0f : 1.0f, signbit(z.y) ? -1.0f : 1.0f);
    const float2 sz = __fadd2_rn(sg, z);
    const float2 a = f2(-__frcp_rn(sz.x), -__frcp_rn(sz.y));
    const float2 b = __fmul2_rn(__fmul2_rn(x, y), a);
    const float2 e1[3] = {__fadd2_rn(f2s(1.0f), mul2s(__fmul2_rn(sg, __fmul2_rn(x, x)), a)), __fmul2_rn(sg, b), __fmul2_rn(neg2(sg), x)};
    const float2 e2[3] = {b, __fadd2_rn(sg, mul2s(__fmul2_rn(y, y), a)), neg2(y)};
    const float2 fa = __fmul2_rn(st, cp), fb = __fmul2_rn(st, sp);
    const float2 hk[3] = {x, y, z};
#pragma unroll
    for (int k = 0; k < 3; ++k)
        out[k] = __fadd2_rn(__fadd2_rn(mul2s(fa, e1[k]), mul2s(fb, e2[k])), mul2s(c, hk[k]));
    if (!(H.x > 0.0f) || !(H.y > 0.0f)) {
        float d[3];
        if (!(H.x > 0.0f)) { direction3(w0a, w1a, d); out[0].x = d[0]; out[1].x = d[1]; out[2].x = d[2]; }
        if (!(H.y > 0.0f)) { direction3(w0b, w1b, d); out[0].y = d[0]; out[1].y = d[1]; out[2].y = d[2]; }
    }
}

template <bool UNITJ>
__device__ __forceinline__ float2 add_nb2(float2 h, float J, float sa, float sb) {
    return UNITJ ? __fadd2_rn(h, f2(sa, sb)) : __fadd2_rn(h, mul2s(f2s(J), f2(sa, sb)));
}

// The update of one quad of 4 consecutive same-colour sites of a row, shared by the strip kernel and the TMA-staged
// kernel (vector_tma_kernel.cuh) so that both perform the same fp32 operations in the same order as the one-thread-per-
// site kernel (bit-identical results); the sites are handled as two pairs with packed arithmetic.  o_cur = other colour
// at the same compressed indices, side[c] = the one x-neighbour outside the quad (p = 1: first site of the next quad,
// p = 0: last site of the previous one), o_prev / o_next = rows y -+ 1, o_zm / o_zp = planes z -+ 1 (D = 3), own = the
// quad's spins, ctr0 = GLOBAL compressed index of the quad's first site (Philox counter word 0 of site i is ctr0 + i).
// phase 1: the local fields of the four sites, hp[pr][c] = component c of sites 2 pr and 2 pr + 1
template <int NC, int D, bool UNITJ>
__device__ __forceinline__ void vector_quad_field(float Jx, float Jy, float Jz, uint32_t p, const Quad<NC> &o_cur,
                                                  const float side[NC], const Quad<NC> &o_prev, const Quad<NC> &o_next,
                                                  const Quad<NC> &o_zm, const Quad<NC> &o_zp, float2 hp[2][NC]) {
    // order -x, +x, -y, +y, -z, +z, every product and sum rounded separately
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        // the two x-neighbours are o (same compressed index) and sh (index + 1 if p, index - 1 if not); the
        // first sum J x(-x) + J x(+x) is commutative, so which of the two is "-x" does not matter
        const float4 o = o_cur.c[c];
        const float4 sh = p ? make_float4(o.y, o.z, o.w, side[c]) : make_float4(side[c], o.x, o.y, o.z);
        float2 v01 = UNITJ ? __fadd2_rn(f2(o.x, o.y), f2(sh.x, sh.y))
                           : __fadd2_rn(mul2s(f2s(Jx), f2(o.x, o.y)), mul2s(f2s(Jx), f2(sh.x, sh.y)));
        float2 v23 = UNITJ ? __fadd2_rn(f2(o.z, o.w), f2(sh.z, sh.w))
                           : __fadd2_rn(mul2s(f2s(Jx), f2(o.z, o.w)), mul2s(f2s(Jx), f2(sh.z, sh.w)));
        v01 = add_nb2<UNITJ>(v01, Jy, o_prev.c[c].x, o_prev.c[c].y);
        v23 = add_nb2<UNITJ>(v23, Jy, o_prev.c[c].z, o_prev.c[c].w);
        v01 = add_nb2<UNITJ>(v01, Jy, o_next.c[c].x, o_next.c[c].y);
        v23 = add_nb2<UNITJ>(v23, Jy, o_next.c[c].z, o_next.c[c].w);
        if (D == 3) {
            v01 = add_nb2<UNITJ>(v01, Jz, o_zm.c[c].x, o_zm.c[c].y);
            v23 = add_nb2<UNITJ>(v23, Jz, o_zm.c[c].z, o_zm.c[c].w);
            v01 = add_nb2<UNITJ>(v01, Jz, o_zp.c[c].x, o_zp.c[c].y);
            v23 = add_nb2<UNITJ>(v23, Jz, o_zp.c[c].z, o_zp.c[c].w);
        }
        hp[0][c] = v01;
        hp[1][c] = v23;
    }
}

// phase 2: proposals, acceptance and the new spins res[c][i] of the four sites from their fields and old spins
// MEAS: *eq = sum over the four sites of s'_i . h_i (fp32, sites in order, each product and sum rounded separately)
template <int NC, bool HB, bool MEAS = false>
__device__ __forceinline__ void vector_quad_accept(const VectorArgs &a, const float2 hp[2][NC], const Quad<NC> &own,
                                                   uint32_t ctr0, uint32_t rho, uint32_t tag, float res[NC][4], float *eq = nullptr) {
    [[maybe_unused]] float esum = 0.0f;
    // the two sites of pair pr: esum += s' . h, first site then second
    [[maybe_unused]] const auto add_energy = [&](int pr) {
        float2 dot = mul2s(f2(res[0][2 * pr], res[0][2 * pr + 1]), hp[pr][0]);
#pragma unroll
        for (int c = 1; c < NC; ++c) dot = __fadd2_rn(dot, mul2s(f2(res[c][2 * pr], res[c][2 * pr + 1]), hp[pr][c]));
        esum = __fadd_rn(__fadd_rn(esum, dot.x), dot.y);
    };
#pragma unroll
    for (int pr = 0; pr < 2; ++pr) {
        uint32_t wa[4], wb[4];
        if (NC == 2 || HB) {
            // the two sites of a pair share one call (R-16b; ctr0 is a multiple of 4): words 0, 1 -> first site, 2, 3 -> second
            philox4x32_10((ctr0 >> 1) + pr, rho, a.t, tag, a.keys, wa);
            wb[0] = wa[2]; wb[1] = wa[3];
        } else {
            philox4x32_10(ctr0 + 2 * pr, rho, a.t, tag, a.keys, wa);
            philox4x32_10(ctr0 + 2 * pr + 1, rho, a.t, tag, a.keys, wb);
        }
        if (HB && NC == 3) {
            const float2 h3[3] = {hp[pr][0], hp[pr][1], hp[pr][NC - 1]};
            float2 s3[3];
            heatbath3_x2(a.beta, h3, wa[0], wa[1], wb[0], wb[1], s3);
#pragma unroll
            for (int c = 0; c < NC; ++c) { res[c][2 * pr] = s3[c].x; res[c][2 * pr + 1] = s3[c].y; }
            if (MEAS) add_energy(pr);
            continue;
        }
        float2 sn[NC], so[NC];
        uint32_t wacc_a, wacc_b;
        if (NC == 3) { direction3_x2(wa[0], wa[1], wb[0], wb[1], sn); wacc_a = wa[2]; wacc_b = wb[2]; }
        else { direction2_x2(wa[0], wb[0], sn); wacc_a = wa[1]; wacc_b = wb[1]; }
#pragma unroll
        for (int c = 0; c < NC; ++c) so[c] = pr == 0 ? f2(own.c[c].x, own.c[c].y) : f2(own.c[c].z, own.c[c].w);
        // acc = (s' - s) . h = -dE; accept iff dE <= 0 (acc >= 0) or u < exp(-beta dE) = exp(beta acc)
        float2 acc = mul2s(__fadd2_rn(sn[0], neg2(so[0])), hp[pr][0]);   // every product of the sum, the first one too (mul2s)
#pragma unroll
        for (int c = 1; c < NC; ++c) acc = __fadd2_rn(acc, mul2s(__fadd2_rn(sn[c], neg2(so[c])), hp[pr][c]));
        const float2 arg = __fmul2_rn(f2s(a.beta), acc);
        // branch-free (`|`, not `||`): a short-circuit branch around the exponential diverges inside the warp anyway and its
        // reconvergence barriers keep the two sites' chains from interleaving
        const bool acc_a = (acc.x >= 0.0f) | (u24(wacc_a) < expf(arg.x));
        const bool acc_b = (acc.y >= 0.0f) | (u24(wacc_b) < expf(arg.y));
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            res[c][2 * pr] = acc_a ? sn[c].x : so[c].x;
            res[c][2 * pr + 1] = acc_b ? sn[c].y : so[c].y;
        }
        if (MEAS) add_energy(pr);
    }
    if (MEAS) *eq = esum;
}

template <int NC, int D, bool UNITJ, bool HB>
__device__ __forceinline__ void vector_quad_update(const VectorArgs &a, float Jx, float Jy, float Jz, uint32_t p,
                                                   const Quad<NC> &o_cur, const float side[NC], const Quad<NC> &o_prev,
                                                   const Quad<NC> &o_next, const Quad<NC> &o_zm, const Quad<NC> &o_zp,
                                                   const Quad<NC> &own, uint32_t ctr0, uint32_t rho, uint32_t tag,
                                                   float res[NC][4]) {
    float2 hp[2][NC];
    vector_quad_field<NC, D, UNITJ>(Jx, Jy, Jz, p, o_cur, side, o_prev, o_next, o_zm, o_zp, hp);
    vector_quad_accept<NC, HB>(a, hp, own, ctr0, rho, tag, res);
}

// MEAS (colour-1 half-sweep of spin_sweep_record): every bond joins the two colours, so
// E = -sum_{i in colour 1} s'_i . h_i with the local field this half-sweep has formed anyway, and M = the new colour-1
// spins plus the colour-0 spins at the same compressed indices (already loaded as o_cur).  Per-site terms in fp32 (each
// product and sum rounded separately) summed in fp32 over the 128 sites of a warp (fixed shuffle tree), then in fp64 by
// vector_partials_finalize in a fixed order: deterministic.
template <int NC, int D, bool UNITJ, int K, bool HB = false, bool MEAS = false, bool RANGED = false>
__global__ void __launch_bounds__(128, (HB && !MEAS) ? 7 : 0) vector_strip_halfsweep(const __grid_constant__ VectorArgs a) {
    const Geometry &g = a.g;
    const uint32_t RL = g.RL, QX = RL >> 2, Ly = (uint32_t)g.Ly, Lz = (uint32_t)g.Lz, Nh = g.Nh;
    // RANGED: rows (d = 2) / planes (d = 3) [sw_p0, sw_p0 + sw_pn) of the slowest axis only (slab handles, half-sweeps in pieces)
    const uint32_t ys0 = (RANGED && D == 2) ? g.sw_p0 : 0u, Lys = (RANGED && D == 2) ? g.sw_pn : Ly;
    const uint32_t zs0 = (RANGED && D == 3) ? g.sw_p0 : 0u, Lzs = (RANGED && D == 3) ? g.sw_pn : Lz;
    const uint32_t j_first = RANGED ? g.sw_j0 : 0u;
    const uint32_t nstrip = (Lys + K - 1) / K;
    const uint32_t per_replica = QX * nstrip * Lzs;
    // the replica is blockIdx.y (host: gridDim.y = R), so the plane base pointers are warp-uniform and every access is
    // "uniform 64-bit base + 32-bit offset" (no per-thread 64-bit address arithmetic)
    const uint32_t it = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t r = blockIdx.y;
    if (K == 1 && a.prefetch && threadIdx.x == 0u) {
        // K = 1: quad `it` sits at float offset sw_j0 + 4 it of every component plane, so the CTA `prefetch` places ahead reads two
        // contiguous ranges per component (its own spins and the other colour at the same indices; the rows around them
        // belong to CTAs that run at about the same time).  One thread asks for them now: bulk L2 prefetch, no registers.
        const uint32_t it0 = (blockIdx.x + a.prefetch) * blockDim.x;
        if (it0 < per_replica) {
            const uint32_t bytes = 16u * min(blockDim.x, per_replica - it0);
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                l2_prefetch_bulk(a.s[a.colour] + ((size_t)r * NC + c) * Nh + j_first + 4u * (size_t)it0, bytes);
                l2_prefetch_bulk(a.s[1 - a.colour] + ((size_t)r * NC + c) * Nh + j_first + 4u * (size_t)it0, bytes);
            }
        }
    }
    float e_acc = 0.0f, m_acc[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) m_acc[c] = 0.0f;
    if (it < per_replica) {
    const uint32_t sz = fdiv(it, g.divQX), q = it - sz * QX;       // sz = strip + nstrip * z
    // one row per thread on the whole lattice: nstrip = Ly, whose host-prepared reciprocal replaces the ~20-instruction division
    const uint32_t zl = (K == 1 && !RANGED) ? fdiv(sz, g.divLy) : sz / nstrip, z = zs0 + zl, y0 = ys0 + (sz - zl * nstrip) * K;
    const uint32_t kend = min((uint32_t)K, ys0 + Lys - y0);
    const float *__restrict__ other = a.s[1 - a.colour] + (size_t)r * NC * Nh;
    float *mine = a.s[a.colour] + (size_t)r * NC * Nh;
    const uint32_t rho = a.replica_streams ? r + a.rho_off : 0u;
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
            float res[NC][4];
            float2 hp[2][NC];
            [[maybe_unused]] float osum[NC];   // MEAS: the colour-0 spins at the quad's indices, summed before they die
            if (MEAS) {
#pragma unroll
                for (int c = 0; c < NC; ++c) osum[c] = __fadd_rn(__fadd_rn(o_cur.c[c].x, o_cur.c[c].y), __fadd_rn(o_cur.c[c].z, o_cur.c[c].w));
            }
            vector_quad_field<NC, D, UNITJ>(Jx, Jy, Jz, p, o_cur, side, o_prev, o_next, o_zm, o_zp, hp);
            [[maybe_unused]] float eq = 0.0f;
            vector_quad_accept<NC, HB, MEAS>(a, hp, own, off + g.j_off, rho, tag, res, &eq);
#pragma unroll
            for (int c = 0; c < NC; ++c)
                *(float4 *)(mine + (size_t)c * Nh + off) = make_float4(res[c][0], res[c][1], res[c][2], res[c][3]);
            if (MEAS && off >= g.own_j0 && off < g.own_j1) {
                e_acc = __fsub_rn(e_acc, eq);
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const float mq = __fadd_rn(__fadd_rn(__fadd_rn(res[c][0], res[c][1]), __fadd_rn(res[c][2], res[c][3])), osum[c]);
                    m_acc[c] = __fadd_rn(m_acc[c], mq);
                }
            }
            o_prev = o_cur;
            o_cur = o_next;
            p ^= 1u;
        }
    }
    }
    if (MEAS) {
        // per warp: fp32 shuffle tree over the lanes' quad sums (128 sites: fixed order, dead lanes contribute 0); everything
        // above the warp is summed in fp64: the CTA's warps here, the CTAs in vector_partials_finalize
        float v[1 + NC];
        v[0] = e_acc;
#pragma unroll
        for (int c = 0; c < NC; ++c) v[1 + c] = m_acc[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int c = 0; c < 1 + NC; ++c) v[c] = __fadd_rn(v[c], __shfl_down_sync(0xFFFFFFFFu, v[c], o));
        }
        __shared__ float wsum[4][1 + NC];
        if ((threadIdx.x & 31u) == 0u) {
#pragma unroll
            for (int c = 0; c < 1 + NC; ++c) wsum[threadIdx.x >> 5][c] = v[c];
        }
        __syncthreads();
        if (threadIdx.x < 1 + NC) {
            // the CTA's partial: its warps in order, in fp64
            double t = 0.0;
            for (uint32_t w = 0; w < (blockDim.x >> 5); ++w) t += (double)wsum[w][threadIdx.x];
            a.part[((size_t)r * gridDim.x + blockIdx.x) * (1 + NC) + threadIdx.x] = t;
        }
    }
}

}  // namespace spin
