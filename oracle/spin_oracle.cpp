/*
 * spin_oracle.cpp -- the CPU ORACLE (TEST INFRASTRUCTURE, NOT PRODUCT; see spin_oracle.h).
 *
 * Plain, slow, single-threaded.  One site at a time, in the paper's order:
 *   sweep = for colour c in (0, 1): for every site of colour c: Metropolis update
 * (PAPER.md:42 checkerboard decomposition; Eq. (2)).
 * Nothing here is blocked, fused, vectorised or reordered.  The only memo is the
 * one-entry cache of the 32 Philox words of the current random "unit" (32 sites
 * share them by definition of the bit-plane contract, R-16); the
 * uncached definition is oracle_ising_uniform() and a test checks both agree.
 *
 * Build: g++ -O2 -std=c++17 -ffp-contract=off -fno-fast-math -shared -fPIC
 * (-ffp-contract=off matters: every fp32 operation below is a separately rounded
 *  IEEE operation, in the order written).
 */
#include "spin_oracle.h"

#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

namespace {

/* ---------------------------------------------------------------- Philox -- */
/* Salmon et al., SC'11: 10 rounds of
 *   (hi0, lo0) = M0 * ctr[0];  (hi1, lo1) = M1 * ctr[2]
 *   ctr = (hi1 ^ ctr[1] ^ key[0], lo1, hi0 ^ ctr[3] ^ key[1], lo0)
 * with the key bumped by the Weyl constants between rounds. */
const uint32_t PHILOX_M0 = 0xD2511F53u;
const uint32_t PHILOX_M1 = 0xCD9E8D57u;
const uint32_t PHILOX_W0 = 0x9E3779B9u;
const uint32_t PHILOX_W1 = 0xBB67AE85u;

void philox(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* rand(unit, rho, t, tag); tag = colour + 16 domain + 256 call */
enum { DOMAIN_ISING_UPDATE = 0, DOMAIN_INIT = 1, DOMAIN_BONDS = 2, DOMAIN_VECTOR_UPDATE = 3 };

void rand4(uint64_t seed, uint32_t unit, uint32_t rho, uint32_t t, uint32_t tag, uint32_t out[4]) {
    const uint32_t ctr[4] = {unit, rho, t, tag};
    const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
    philox(ctr, key, out);
}

uint32_t make_tag(int colour, int domain, int call) { return (uint32_t)colour + 16u * (uint32_t)domain + 256u * (uint32_t)call; }

/* Words of the n >= 2 update of the site with compressed same-colour index j (R-16b):
 * the Metropolis update of n = 3 takes three words, so every site has its own call rand(j, ...);
 * n = 2 (angle, acceptance) and the heat bath of n = 3 (polar cosine, azimuth) take two, so sites 2k and 2k + 1 of a
 * colour share the call rand(k, ...): the even one takes words 0 and 1, the odd one words 2 and 3 (returned as w[0], w[1]). */
void vector_site_words(uint64_t seed, int n, int rule, uint64_t j, uint32_t rho, uint32_t t, int colour, uint32_t w[4]) {
    if (n == 2 || rule == ORACLE_RULE_HEATBATH) {
        uint32_t c[4];
        rand4(seed, (uint32_t)(j >> 1), rho, t, make_tag(colour, DOMAIN_VECTOR_UPDATE, 0), c);
        const int o = (int)(j & 1u) * 2;
        w[0] = c[o]; w[1] = c[o + 1]; w[2] = 0u; w[3] = 0u;
    } else {
        rand4(seed, (uint32_t)j, rho, t, make_tag(colour, DOMAIN_VECTOR_UPDATE, 0), w);
    }
}

/* Bit-plane contract (R-16): the 32-bit acceptance uniform of lane `lane` of a
 * unit has digit k (k = 0 is the most significant) equal to bit `lane` of word
 * (k & 3) of Philox call (k >> 2). */
void unit_words(uint64_t seed, uint32_t unit, uint32_t rho, uint32_t t, int colour, uint32_t words[32]) {
    for (int call = 0; call < 8; ++call)
        rand4(seed, unit, rho, t, make_tag(colour, DOMAIN_ISING_UPDATE, call), &words[4 * call]);
}

uint32_t lane_uniform(const uint32_t words[32], int lane) {
    uint32_t U = 0;
    for (int k = 0; k < 32; ++k) U = (U << 1) | ((words[k] >> lane) & 1u);
    return U;
}

/* ------------------------------------------------------------ thresholds -- */
/* T(dE) = floor(exp(-beta dE) * 2^32) in double; 2^32 when the factor is 1. */
uint64_t threshold(double beta, int dE) {
    const double p = std::exp(-beta * (double)dE);
    const double scaled = std::ldexp(p, 32);
    if (!(scaled < 4294967296.0)) return 4294967296ull; /* p >= 1 (or NaN guard) */
    if (!(scaled > 0.0)) return 0ull;
    return (uint64_t)std::floor(scaled);
}

/* -------------------------------------------------- continuous-spin maths -- */
float u24(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-08f; /* 2^-24, exact */ }

/* sin(pi x), cos(pi x) for x in [0, 2), in double with exact quadrant
 * reduction, rounded once to fp32 by the caller. */
void sincospi_double(double x, double *s, double *c) {
    const double two_x = 2.0 * x;
    const double nq = std::floor(two_x + 0.5);     /* nearest half-integer index */
    const double r = x - 0.5 * nq;                 /* exact, |r| <= 1/4          */
    const double PI = 3.14159265358979323846264338327950288;
    const double sr = std::sin(PI * r), cr = std::cos(PI * r);
    const int q = ((int)nq) & 3;
    switch (q) {
        case 0: *s = sr;  *c = cr;  break;
        case 1: *s = cr;  *c = -sr; break;
        case 2: *s = -sr; *c = -cr; break;
        default: *s = -cr; *c = sr; break;
    }
}

/* direction(a, b): uniform point on the unit sphere (R-12):
 * z = 2 u24(a) - 1; rho = sqrt(max(0, 1 - z z)); phi/pi = 2 u24(b). */
void direction3(uint32_t a, uint32_t b, float out[3]) {
    const float z = 2.0f * u24(a) - 1.0f;
    const float zz = z * z;
    float one_minus = 1.0f - zz;
    if (one_minus < 0.0f) one_minus = 0.0f;
    const float rho = std::sqrt(one_minus);
    const float phi2 = 2.0f * u24(b);
    double sd, cd;
    sincospi_double((double)phi2, &sd, &cd);
    const float sf = (float)sd, cf = (float)cd;
    out[0] = rho * cf;
    out[1] = rho * sf;
    out[2] = z;
}

void direction2(uint32_t a, float out[2]) {
    const float phi2 = 2.0f * u24(a);
    double sd, cd;
    sincospi_double((double)phi2, &sd, &cd);
    out[0] = (float)cd;
    out[1] = (float)sd;
}

int vector_accept(float beta_f, float dE, uint32_t w) {
    if (dE <= 0.0f) return 1;
    const float arg = (-beta_f) * dE;                 /* one fp32 rounding   */
    const float p = (float)std::exp((double)arg);     /* exp, rounded once   */
    return u24(w) < p ? 1 : 0;
}

/* ------------------------------------------------------------ heat bath -- */
/* PAPER.md:40 "updates according to the heat-bath prescription": the new value of
 * the spin is drawn from its conditional Boltzmann distribution in the local field
 * h = sum_j J_ij s_j, whatever the old value was.
 *   n = 1: P(s = +1) = e^{beta h} / (e^{beta h} + e^{-beta h}) = 1 / (1 + e^{-2 beta h});
 *          tabulated like the Metropolis factors: T_hb(h) = floor(P 2^32), s = +1 iff U < T_hb(h). */
uint64_t heatbath_threshold(double beta, int h) {
    const double p = 1.0 / (1.0 + std::exp(-2.0 * beta * (double)h));
    const double scaled = std::ldexp(p, 32);
    if (!(scaled < 4294967296.0)) return 4294967296ull;
    if (!(scaled > 0.0)) return 0ull;
    return (uint64_t)std::floor(scaled);
}

/*   n = 3: with H = beta |h| the cosine c of the angle between the new spin and h has density
 *          proportional to e^{H c} on [-1, 1]; inverting its distribution function with a uniform u:
 *          c = 1 + ln(1 - u (1 - e^{-2H})) / H.  The azimuth about h is uniform.  H = 0: uniform direction.
 *   Frame: hhat = h / |h| and the branch-free orthonormal basis (e1, e2) of Duff et al. (JCGT 2017):
 *          sg = copysign(1, hz), a = -1 / (sg + hz), b = hx hy a,
 *          e1 = (1 + sg hx hx a, sg b, -sg hx), e2 = (b, sg + hy hy a, -hy).
 *   s' = st (cp e1 + sp e2) + c hhat, st = sqrt(max(0, 1 - c c)), (sp, cp) = sincospi(2 u24(w1)).
 *   fp32 throughout, every operation rounded separately in the order written; exp, log and sincospi are
 *   evaluated in double and rounded once (as for the Metropolis proposal). */
void heatbath3(float beta_f, const float h[3], uint32_t w0, uint32_t w1, float out[3]) {
    const float hh = (h[0] * h[0] + h[1] * h[1]) + h[2] * h[2];
    const float hn = std::sqrt(hh);
    const float H = beta_f * hn;
    if (!(H > 0.0f)) { direction3(w0, w1, out); return; }
    const float u = u24(w0);
    const float e2H = (float)std::exp((double)(-2.0f * H));
    const float arg = 1.0f - u * (1.0f - e2H);          /* in (e^{-2H}, 1] */
    const float lg = (float)std::log((double)arg);
    float c = 1.0f + lg / H;
    if (c < -1.0f) c = -1.0f;
    if (c > 1.0f) c = 1.0f;
    float omc = 1.0f - c * c;
    if (omc < 0.0f) omc = 0.0f;
    const float st = std::sqrt(omc);
    double sd, cd;
    sincospi_double((double)(2.0f * u24(w1)), &sd, &cd);
    const float sp = (float)sd, cp = (float)cd;
    const float inv = 1.0f / hn;
    const float x = h[0] * inv, y = h[1] * inv, z = h[2] * inv;
    const float sg = std::signbit(z) ? -1.0f : 1.0f;
    const float a = -1.0f / (sg + z);
    const float b = (x * y) * a;
    const float e1[3] = {1.0f + (sg * (x * x)) * a, sg * b, (-sg) * x};
    const float e2[3] = {b, sg + (y * y) * a, -y};
    const float fa = st * cp, fb = st * sp;
    for (int k = 0; k < 3; ++k) {
        const float hk = (k == 0) ? x : (k == 1 ? y : z);
        out[k] = (fa * e1[k] + fb * e2[k]) + c * hk;
    }
}

}  // namespace

/* ---------------------------------------------------------------- system -- */
struct oracle_system {
    int Lx, Ly, Lz, d, n;
    int coupling_kind;
    double J[3];
    int R, replica_streams;
    int rule; /* ORACLE_RULE_METROPOLIS (Eq. (2)) or ORACLE_RULE_HEATBATH */
    uint64_t seed;
    uint64_t t; /* sweeps done so far = Philox sweep counter */
    int64_t N;
    std::vector<int8_t> s1;    /* n = 1 : [r][i]          */
    std::vector<float> sv;     /* n >= 2: [r][i][n]       */
    std::vector<int8_t> bonds; /* BOND_PM1: [r][mu][i]    */
    /* bookkeeping only (the accepted move changes H by dE): sum over the last sweep, all replicas, of
     * the dE of every accepted Metropolis move, as the sweep itself computed it; never read by the update */
    double dE_accepted = 0.0;

    int64_t site(int x, int y, int z) const { return (int64_t)x + (int64_t)Lx * ((int64_t)y + (int64_t)Ly * (int64_t)z); }
    int64_t compressed(int x, int y, int z) const { return (int64_t)(x >> 1) + (int64_t)(Lx / 2) * ((int64_t)y + (int64_t)Ly * (int64_t)z); }

    /* coupling of the bond that leaves site i in direction +mu, replica r */
    double forward_J(int r, int mu, int64_t i) const {
        if (coupling_kind == ORACLE_J_UNIFORM) return J[0];
        if (coupling_kind == ORACLE_J_PER_DIRECTION) return J[mu];
        return (double)bonds[((size_t)r * d + mu) * (size_t)N + (size_t)i];
    }
};

namespace {

struct Neighbour { int64_t i; double J; };

/* the 2d neighbours of (x, y, z) in the fixed order -x, +x, -y, +y, -z, +z with
 * the coupling of the connecting bond; periodic in every direction (R-7).  A
 * dimension of size 2 has -mu and +mu neighbour equal: both bonds count. */
int neighbours(const oracle_system &S, int r, int x, int y, int z, Neighbour nb[6]) {
    const int L[3] = {S.Lx, S.Ly, S.Lz};
    const int p[3] = {x, y, z};
    int count = 0;
    for (int mu = 0; mu < S.d; ++mu) {
        int q[3] = {x, y, z};
        q[mu] = (p[mu] == 0) ? L[mu] - 1 : p[mu] - 1;            /* (x - 1) mod L */
        const int64_t im = S.site(q[0], q[1], q[2]);
        nb[count].i = im;
        nb[count].J = S.forward_J(r, mu, im); /* bond from the -mu neighbour to us */
        ++count;
        q[mu] = (p[mu] == L[mu] - 1) ? 0 : p[mu] + 1;            /* (x + 1) mod L */
        nb[count].i = S.site(q[0], q[1], q[2]);
        nb[count].J = S.forward_J(r, mu, S.site(x, y, z)); /* our own forward bond */
        ++count;
    }
    return count;
}

int64_t sweep_ising(oracle_system &S, double beta) {
    int64_t accepted = 0;
    S.dE_accepted = 0.0;
    /* table of the Boltzmann factors that can occur: dE = 2 s h, |h| <= 2d */
    uint64_t T[13], Thb[13];
    for (int dE = 0; dE <= 12; ++dE) T[dE] = threshold(beta, dE);
    for (int h = -6; h <= 6; ++h) Thb[h + 6] = heatbath_threshold(beta, h);
    const uint32_t t32 = (uint32_t)S.t;
    for (int colour = 0; colour < 2; ++colour) {
        for (int r = 0; r < S.R; ++r) {
            const uint32_t rho = S.replica_streams ? (uint32_t)r : 0u;
            int8_t *s = &S.s1[(size_t)r * (size_t)S.N];
            uint32_t words[32];
            int64_t cached_unit = -1;
            for (int z = 0; z < S.Lz; ++z)
                for (int y = 0; y < S.Ly; ++y)
                    for (int x = 0; x < S.Lx; ++x) {
                        if (((x + y + z) & 1) != colour) continue;
                        const int64_t i = S.site(x, y, z);
                        const int64_t j = S.compressed(x, y, z);
                        const int64_t unit = j >> 5;
                        if (unit != cached_unit) {
                            unit_words(S.seed, (uint32_t)unit, rho, t32, colour, words);
                            cached_unit = unit;
                        }
                        const uint32_t U = lane_uniform(words, (int)(j & 31));
                        Neighbour nb[6];
                        const int q = neighbours(S, r, x, y, z, nb);
                        int h = 0;
                        for (int k = 0; k < q; ++k) h += (int)nb[k].J * (int)s[nb[k].i];
                        if (S.rule == ORACLE_RULE_HEATBATH) {
                            const int8_t snew = ((uint64_t)U < Thb[h + 6]) ? (int8_t)1 : (int8_t)-1;
                            if (snew != s[i]) ++accepted;
                            s[i] = snew;
                            continue;
                        }
                        const int dE = 2 * (int)s[i] * h;
                        if (dE <= 0 || (uint64_t)U < T[dE]) {
                            s[i] = (int8_t)(-s[i]);
                            ++accepted;
                            S.dE_accepted += (double)dE;
                        }
                    }
        }
    }
    S.t += 1;
    return accepted;
}

int64_t sweep_vector(oracle_system &S, double beta) {
    int64_t accepted = 0;
    S.dE_accepted = 0.0;
    const float beta_f = (float)beta;
    const uint32_t t32 = (uint32_t)S.t;
    const int n = S.n;
    for (int colour = 0; colour < 2; ++colour) {
        for (int r = 0; r < S.R; ++r) {
            const uint32_t rho = S.replica_streams ? (uint32_t)r : 0u;
            float *s = &S.sv[(size_t)r * (size_t)S.N * (size_t)n];
            for (int z = 0; z < S.Lz; ++z)
                for (int y = 0; y < S.Ly; ++y)
                    for (int x = 0; x < S.Lx; ++x) {
                        if (((x + y + z) & 1) != colour) continue;
                        const int64_t i = S.site(x, y, z);
                        const int64_t j = S.compressed(x, y, z);
                        uint32_t w[4];
                        vector_site_words(S.seed, n, S.rule, (uint64_t)j, rho, t32, colour, w);
                        float snew[3] = {0.0f, 0.0f, 0.0f};
                        uint32_t w_accept;
                        if (n == 3) { direction3(w[0], w[1], snew); w_accept = w[2]; }
                        else        { direction2(w[0], snew);       w_accept = w[1]; }
                        Neighbour nb[6];
                        const int q = neighbours(S, r, x, y, z, nb);
                        float h[3] = {0.0f, 0.0f, 0.0f};
                        for (int k = 0; k < q; ++k) {
                            const float Jf = (float)nb[k].J;
                            for (int a = 0; a < n; ++a) {
                                const float term = Jf * s[(size_t)nb[k].i * n + a];
                                h[a] = h[a] + term;
                            }
                        }
                        if (S.rule == ORACLE_RULE_HEATBATH) {
                            /* n = 3 only (oracle_set_update_rule refuses n = 2) */
                            heatbath3(beta_f, h, w[0], w[1], snew);
                            for (int a = 0; a < n; ++a) s[(size_t)i * n + a] = snew[a];
                            ++accepted;
                            continue;
                        }
                        float acc = 0.0f;
                        for (int a = 0; a < n; ++a) {
                            const float diff = snew[a] - s[(size_t)i * n + a];
                            const float prod = diff * h[a];
                            acc = (a == 0) ? prod : acc + prod;
                        }
                        const float dE = -acc;
                        if (vector_accept(beta_f, dE, w_accept)) {
                            for (int a = 0; a < n; ++a) s[(size_t)i * n + a] = snew[a];
                            ++accepted;
                            S.dE_accepted += (double)dE;
                        }
                    }
        }
    }
    S.t += 1;
    return accepted;
}

}  // namespace

/* ------------------------------------------------------------- C interface -- */
extern "C" {

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox(ctr, key, out); }

void oracle_rand(uint64_t seed, uint32_t unit, uint32_t rho, uint32_t t, uint32_t tag, uint32_t out[4]) {
    rand4(seed, unit, rho, t, tag, out);
}

void oracle_vector_site_words(uint64_t seed, int n, int rule, uint64_t j, uint32_t rho, uint32_t t, int colour, uint32_t out[4]) {
    vector_site_words(seed, n, rule, j, rho, t, colour, out);
}

uint32_t oracle_ising_uniform(uint64_t seed, uint64_t j, uint32_t rho, uint32_t t, int colour) {
    uint32_t words[32];
    unit_words(seed, (uint32_t)(j >> 5), rho, t, colour, words);
    return lane_uniform(words, (int)(j & 31));
}

uint64_t oracle_threshold(double beta, int dE) { return threshold(beta, dE); }

int oracle_ising_accept(double beta, int dE, uint32_t U) {
    if (dE <= 0) return 1;
    return (uint64_t)U < threshold(beta, dE) ? 1 : 0;
}

float oracle_u24(uint32_t w) { return u24(w); }
void oracle_direction3(uint32_t a, uint32_t b, float out[3]) { direction3(a, b, out); }
void oracle_direction2(uint32_t a, float out[2]) { direction2(a, out); }
int oracle_vector_accept(double beta, float dE, uint32_t w) { return vector_accept((float)beta, dE, w); }

oracle_system *oracle_create(const int32_t dims[3], int32_t n, int32_t coupling_kind, const double J[3],
                             const int8_t *bonds, int32_t n_replicas, int32_t replica_streams, int32_t init,
                             uint64_t seed) {
    if (!dims || !J) return nullptr;
    if (n < 1 || n > 3 || n_replicas < 1) return nullptr;
    if (dims[0] < 2 || dims[1] < 2 || dims[2] < 1) return nullptr;
    if ((dims[0] & 1) || (dims[1] & 1) || (dims[2] > 1 && (dims[2] & 1))) return nullptr;
    if (coupling_kind < 0 || coupling_kind > 2) return nullptr;
    if (init != ORACLE_INIT_HOT && init != ORACLE_INIT_COLD) return nullptr;
    oracle_system *S = new (std::nothrow) oracle_system();
    if (!S) return nullptr;
    S->Lx = dims[0]; S->Ly = dims[1]; S->Lz = dims[2];
    S->d = (dims[2] == 1) ? 2 : 3;
    S->n = n;
    S->coupling_kind = coupling_kind;
    for (int mu = 0; mu < 3; ++mu) S->J[mu] = J[mu];
    if (n == 1 && coupling_kind != ORACLE_J_BOND_PM1) {
        /* the integer table covers J in {-1, 0, +1} only (R-6) */
        const int used = (coupling_kind == ORACLE_J_UNIFORM) ? 1 : S->d;
        for (int mu = 0; mu < used; ++mu)
            if (!(J[mu] == -1.0 || J[mu] == 0.0 || J[mu] == 1.0)) { delete S; return nullptr; }
    }
    S->R = n_replicas;
    S->replica_streams = replica_streams ? 1 : 0;
    S->rule = ORACLE_RULE_METROPOLIS;
    S->seed = seed;
    S->t = 0;
    S->N = (int64_t)dims[0] * dims[1] * dims[2];
    const size_t N = (size_t)S->N, R = (size_t)S->R;

    if (coupling_kind == ORACLE_J_BOND_PM1) {
        S->bonds.resize(R * (size_t)S->d * N);
        if (bonds) {
            for (size_t k = 0; k < S->bonds.size(); ++k) {
                if (bonds[k] != 1 && bonds[k] != -1) { delete S; return nullptr; }
                S->bonds[k] = bonds[k];
            }
        } else {
            /* J[r][mu][i] = bit (i & 31) of word mu of rand(i >> 5, r, 0, BONDS) ? -1 : +1 */
            for (size_t r = 0; r < R; ++r)
                for (size_t i = 0; i < N; ++i) {
                    uint32_t w[4];
                    rand4(seed, (uint32_t)(i >> 5), (uint32_t)r, 0u, make_tag(0, DOMAIN_BONDS, 0), w);
                    for (int mu = 0; mu < S->d; ++mu)
                        S->bonds[(r * S->d + mu) * N + i] = ((w[mu] >> (i & 31)) & 1u) ? (int8_t)-1 : (int8_t)1;
                }
        }
    }

    if (n == 1) {
        S->s1.resize(R * N);
        for (size_t r = 0; r < R; ++r)
            for (size_t i = 0; i < N; ++i) {
                if (init == ORACLE_INIT_COLD) { S->s1[r * N + i] = 1; continue; }
                /* s = bit (i & 31) of word ((i >> 5) & 3) of rand(i >> 7, r, 0, INIT) ? -1 : +1 */
                uint32_t w[4];
                rand4(seed, (uint32_t)(i >> 7), (uint32_t)r, 0u, make_tag(0, DOMAIN_INIT, 0), w);
                S->s1[r * N + i] = ((w[(i >> 5) & 3] >> (i & 31)) & 1u) ? (int8_t)-1 : (int8_t)1;
            }
    } else {
        S->sv.resize(R * N * (size_t)n);
        for (size_t r = 0; r < R; ++r)
            for (size_t i = 0; i < N; ++i) {
                float v[3] = {0.0f, 0.0f, 0.0f};
                if (init == ORACLE_INIT_COLD) {
                    if (n == 3) v[2] = 1.0f; else v[0] = 1.0f;
                } else {
                    uint32_t w[4];
                    rand4(seed, (uint32_t)i, (uint32_t)r, 0u, make_tag(0, DOMAIN_INIT, 0), w);
                    if (n == 3) direction3(w[0], w[1], v); else direction2(w[0], v);
                }
                for (int a = 0; a < n; ++a) S->sv[(r * N + i) * n + a] = v[a];
            }
    }
    return S;
}

void oracle_destroy(oracle_system *S) { delete S; }

int oracle_set_update_rule(oracle_system *S, int32_t rule) {
    if (!S || (rule != ORACLE_RULE_METROPOLIS && rule != ORACLE_RULE_HEATBATH)) return 1;
    if (rule == ORACLE_RULE_HEATBATH && S->n == 2) return 1; /* no closed-form inverse for the von Mises law */
    S->rule = rule;
    return 0;
}

uint64_t oracle_heatbath_threshold(double beta, int h) { return heatbath_threshold(beta, h); }
void oracle_heatbath3(double beta, const float h[3], uint32_t w0, uint32_t w1, float out[3]) {
    heatbath3((float)beta, h, w0, w1, out);
}

int oracle_sweep_count(oracle_system *S, double beta, int64_t n_sweeps, int64_t *accepted) {
    if (!S || n_sweeps < 0 || !(beta >= 0.0)) return 1;
    for (int64_t k = 0; k < n_sweeps; ++k) {
        if (S->t > 0xFFFFFFFFull) return 2; /* 32-bit sweep counter (R-19) */
        const int64_t acc = (S->n == 1) ? sweep_ising(*S, beta) : sweep_vector(*S, beta);
        if (accepted) accepted[k] = acc;
    }
    return 0;
}

double oracle_last_sweep_dE(const oracle_system *S) { return S ? S->dE_accepted : 0.0; }

int oracle_sweep(oracle_system *S, double beta, int64_t n_sweeps) { return oracle_sweep_count(S, beta, n_sweeps, nullptr); }

int oracle_measure(const oracle_system *S, double *E, double *M) {
    if (!S || !E || !M) return 1;
    const int L[3] = {S->Lx, S->Ly, S->Lz};
    const size_t N = (size_t)S->N;
    for (int r = 0; r < S->R; ++r) {
        if (S->n == 1) {
            const int8_t *s = &S->s1[(size_t)r * N];
            int64_t e = 0, m = 0;
            for (int z = 0; z < S->Lz; ++z)
                for (int y = 0; y < S->Ly; ++y)
                    for (int x = 0; x < S->Lx; ++x) {
                        const int64_t i = S->site(x, y, z);
                        m += s[i];
                        for (int mu = 0; mu < S->d; ++mu) {
                            int q[3] = {x, y, z};
                            q[mu] = (q[mu] + 1) % L[mu];
                            const int64_t ip = S->site(q[0], q[1], q[2]);
                            e -= (int64_t)S->forward_J(r, mu, i) * s[i] * s[ip];
                        }
                    }
            E[r] = (double)e;
            M[r] = (double)m;
        } else {
            const int n = S->n;
            const float *s = &S->sv[(size_t)r * N * n];
            double e = 0.0, m[3] = {0.0, 0.0, 0.0};
            for (int z = 0; z < S->Lz; ++z)
                for (int y = 0; y < S->Ly; ++y)
                    for (int x = 0; x < S->Lx; ++x) {
                        const int64_t i = S->site(x, y, z);
                        for (int a = 0; a < n; ++a) m[a] += (double)s[(size_t)i * n + a];
                        for (int mu = 0; mu < S->d; ++mu) {
                            int q[3] = {x, y, z};
                            q[mu] = (q[mu] + 1) % L[mu];
                            const int64_t ip = S->site(q[0], q[1], q[2]);
                            double dot = 0.0;
                            for (int a = 0; a < n; ++a) dot += (double)s[(size_t)i * n + a] * (double)s[(size_t)ip * n + a];
                            e -= (double)(float)S->forward_J(r, mu, i) * dot;
                        }
                    }
            E[r] = e;
            for (int a = 0; a < n; ++a) M[(size_t)r * n + a] = m[a];
        }
    }
    return 0;
}

int oracle_get_spins(const oracle_system *S, void *out, uint64_t bytes) {
    if (!S || !out) return 1;
    if (S->n == 1) {
        if (bytes != S->s1.size()) return 1;
        std::memcpy(out, S->s1.data(), S->s1.size());
    } else {
        if (bytes != S->sv.size() * sizeof(float)) return 1;
        std::memcpy(out, S->sv.data(), S->sv.size() * sizeof(float));
    }
    return 0;
}

int oracle_set_spins(oracle_system *S, const void *in, uint64_t bytes) {
    if (!S || !in) return 1;
    if (S->n == 1) {
        if (bytes != S->s1.size()) return 1;
        const int8_t *p = (const int8_t *)in;
        for (size_t k = 0; k < S->s1.size(); ++k)
            if (p[k] != 1 && p[k] != -1) return 1;
        std::memcpy(S->s1.data(), in, S->s1.size());
    } else {
        if (bytes != S->sv.size() * sizeof(float)) return 1;
        std::memcpy(S->sv.data(), in, S->sv.size() * sizeof(float));
    }
    return 0;
}

int oracle_get_bonds(const oracle_system *S, int8_t *out, uint64_t bytes) {
    if (!S || !out || S->coupling_kind != ORACLE_J_BOND_PM1 || bytes != S->bonds.size()) return 1;
    std::memcpy(out, S->bonds.data(), S->bonds.size());
    return 0;
}

uint64_t oracle_get_sweep_count(const oracle_system *S) { return S ? S->t : 0; }
void oracle_set_sweep_count(oracle_system *S, uint64_t t) { if (S) S->t = t; }

}  /* extern "C" */
