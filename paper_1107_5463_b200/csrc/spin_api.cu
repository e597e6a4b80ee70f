// spin_api.cu -- host side of libspin: the C ABI of include/spin.h (argument checks, workspace carving,
// Boltzmann table, kernel selection and launches).  No torch types, no CPU fallback: every step of the
// sweep and of the measurement runs in the kernels of this directory.
#include "../../include/spin.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "ising_int8_kernel.cuh"
#include "ising_kernels.cuh"
#include "ising_msc_kernel.cuh"
#include "ising_pmj_own_kernel.cuh"
#include "ising_resident_kernel.cuh"
#include "ising_resident_pmj_kernel.cuh"
#include "ising_tblock_kernel.cuh"
#include "measure_kernels.cuh"
#include "setup_kernels.cuh"
#include "vector_kernels.cuh"
#include "vector_tma_kernel.cuh"

using namespace spin;

// ------------------------------------------------------------------------------- errors ------
static thread_local char g_err[512] = "";

static spin_status fail(spin_status st, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return st;
}

#define CUDA_TRY(expr)                                                                                    \
    do {                                                                                                  \
        cudaError_t e_ = (expr);                                                                          \
        if (e_ != cudaSuccess) return fail(SPIN_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_));       \
    } while (0)

// ------------------------------------------------------------------------------- handle ------
enum Path { PATH_ISING_GENERIC, PATH_ISING_INT8, PATH_ISING_BITPACK, PATH_VECTOR, PATH_ISING_MSC };

struct Layout {
    size_t off_s[2], bytes_s;   // one colour array
    size_t off_alt[2];          // temporal blocking: the second pair of colour arrays (bytes_s each), or off_s when not offered
    size_t off_bonds, bytes_bonds;
    size_t off_acc, bytes_acc;  // n = 1: int64 [R][2]; n >= 2: double [R][partials][1 + n], then the two below
    size_t off_mid, off_cnt;    // n >= 2: double [R][FINALIZE_BLOCKS][1 + n] and unsigned [R] of vector_partials_finalize
    size_t off_res, bytes_res;  // double [R] E then [R][n] M
    size_t total;
};

struct spin_system {
    spin_config cfg;
    Geometry g;
    PhiloxKeys keys;
    Path path;
    int d, n;
    uint32_t R;
    uint64_t N;
    Layout lay;
    char *ws;
    uint64_t t;          // sweeps done = Philox sweep index of the next sweep
    uint64_t launches;
    int sm_count;
    int block;           // threads per CTA
    int strip_rows;      // strip kernels: rows per thread (1, 2, 4, 8, 16)
    int strip_rows_set;  // the caller chose strip_rows (otherwise each kernel family uses its own default)
    int axis, own_planes; // slab decomposition: axis (2 z, 1 y, -1 none) and owned planes along it
    uint32_t next_colour; // spin_halfsweep: colour expected next
    int vector_generic;  // n >= 2: force the one-thread-per-site kernel (test knob)
    int tblock;          // SPIN_OPT_TEMPORAL_BLOCKING: -1 auto (lattices beyond the CUDA-graph regime), 0 off, 1 wherever offered
    int tblock_rows;     // SPIN_OPT_TBLOCK_ROWS: rows per stripe, 0 = one wave of resident CTAs
    int tblock_ok;       // this handle has the second pair of arrays
    int variant;         // SPIN_OPT_KERNEL_VARIANT: 0 = the default kernel of each family, > 0 = a named alternative (A/B knob)
    int defer_cap;       // SPIN_OPT_DEFER_CAP: queue entries per warp of the deferred digit comparison (default DEFER_CAP)
    int l2_keep;         // SPIN_OPT_L2_KEEP: -1 automatic, -2 no L2 eviction hints, >= 0 replicas whose coupling words are kept in L2
    int l2_bytes;        // L2 size of the device
    int l2_prefetch;     // SPIN_OPT_L2_PREFETCH: -1 each kernel's own distance (default), 0 off, > 0 that distance
    int grid_num, grid_den;
    uint32_t mblocks;    // CTAs (per replica) of the measurement kernels
    double table_beta;   // beta the cached table was built for (NaN = none)
    IsingTable tab;
    HeatBathTable hb;    // n = 1 heat bath: built with the table above
    cudaGraphExec_t gexec;      // GRAPH_SWEEPS sweeps for (g_beta, launch shape); NULL until first used
    cudaGraph_t graph;          // the captured graph (its node handles address the kernel nodes of gexec)
    struct GraphNode *gnodes;   // its kernel nodes with host copies of their argument blocks
    size_t n_gnodes;
    cudaStream_t cap_stream;    // capture-only stream (nothing ever runs on it)
    double g_beta;
    int g_block, g_rows, g_rows_set, g_num, g_den;
    int set_pending;     // a spin_set_spins_async whose +-1 check has not been read yet
    void *staging;       // device buffer for canonical arrays (get / set calls), kept until spin_destroy
    size_t staging_bytes;
    void *h_res;         // pinned host doubles for spin_measure's result (made by the first call)
    // n >= 2, d = 3: TMA-staged kernel (vector_tma_kernel.cuh)
    int tma_ok;          // tensor maps encoded (rows of <= 256 sites per colour, driver entry point found)
    int use_tma;         // SPIN_OPT_TMA_KERNELS: 1 every half-sweep, 0 never, -1 (default) only where its fused E / M pays
    uint32_t tma_ty;     // rows per tile
    CUtensorMap tma_main[2], tma_row[2];
};

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

static FastDiv make_fastdiv(uint32_t d) {
    FastDiv f;
    f.div = d;
    if (d <= 1) { f.mul = 0; f.shift = 0; return f; }
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;                       // l = ceil(log2 d) >= 1
    const unsigned __int128 one = 1;
    const unsigned __int128 num = one << (31 + l);
    f.mul = (uint32_t)((num + d - 1) / d);             // ceil(2^(31+l) / d) <= 2^32 - 1 for d not a power of two
    if (((uint64_t)d & ((uint64_t)d - 1)) == 0) f.mul = 0x80000000u;  // power of two: exact
    f.shift = l - 1;
    return f;
}

struct Derived {
    int d;
    uint64_t N;        // sites of the local arrays (with the ghost planes of a slab)
    uint64_t Nown;     // owned sites (= N when the handle holds the whole lattice)
    int32_t pad[3];    // dims of the local arrays
    int axis;          // slab axis (2: z, 1: y) or -1
    Path path;
};

static spin_status derive(const spin_config *c, Derived *out) {
    if (!c) return fail(SPIN_ERR_INVALID_ARG, "config is NULL");
    const int32_t *L = c->dims;
    if (L[0] < 2 || L[1] < 2 || L[2] < 1) return fail(SPIN_ERR_INVALID_ARG, "dims must be >= 2 (Lz >= 1)");
    if ((L[0] & 1) || (L[1] & 1) || (L[2] > 1 && (L[2] & 1)))
        return fail(SPIN_ERR_INVALID_ARG, "every lattice dimension must be even (checkerboard + periodic)");
    if (c->n < 1 || c->n > 3) return fail(SPIN_ERR_INVALID_ARG, "n must be 1, 2 or 3");
    if (c->n_replicas < 1) return fail(SPIN_ERR_INVALID_ARG, "n_replicas must be >= 1");
    if (c->storage == SPIN_STORE_MSC ? c->n_replicas > 32 * 65535 : c->n_replicas > 65535)
        return fail(SPIN_ERR_UNSUPPORTED, "at most 65535 replicas (MSC: groups of 32 replicas) per handle (they map to a grid dimension)");
    if (c->coupling_kind < SPIN_J_UNIFORM || c->coupling_kind > SPIN_J_BOND_PM1)
        return fail(SPIN_ERR_INVALID_ARG, "bad coupling_kind");
    if (c->init != SPIN_INIT_HOT && c->init != SPIN_INIT_COLD) return fail(SPIN_ERR_INVALID_ARG, "bad init");
    if (c->update_rule != SPIN_UPDATE_METROPOLIS && c->update_rule != SPIN_UPDATE_HEATBATH)
        return fail(SPIN_ERR_INVALID_ARG, "bad update_rule");
    if (c->update_rule == SPIN_UPDATE_HEATBATH && c->n == 2)
        return fail(SPIN_ERR_UNSUPPORTED, "heat bath is offered for n = 1 and n = 3 (no closed-form inverse for n = 2)");
    if (c->storage < SPIN_STORE_INT8 || c->storage > SPIN_STORE_MSC) return fail(SPIN_ERR_INVALID_ARG, "bad storage");
    if (c->n == 1 && c->storage == SPIN_STORE_FP32) return fail(SPIN_ERR_INVALID_ARG, "n = 1 needs INT8 or BITPACK storage");
    if (c->n > 1 && c->storage != SPIN_STORE_FP32) return fail(SPIN_ERR_INVALID_ARG, "n >= 2 needs FP32 storage");
    out->d = L[2] == 1 ? 2 : 3;
    out->Nown = (uint64_t)L[0] * (uint64_t)L[1] * (uint64_t)L[2];
    out->pad[0] = L[0]; out->pad[1] = L[1]; out->pad[2] = L[2];
    out->axis = -1;
    if (c->slab_global != 0) {
        // slab of a larger lattice along the slowest axis: two ghost planes on either side (even, so colours keep
        // their parity); the update sequence is that of the global lattice (global indices feed Philox)
        const int ax = out->d == 3 ? 2 : 1;
        if (c->slab_global < L[ax] || (c->slab_global & 1) || c->slab_offset < 0 || (c->slab_offset & 1) ||
            c->slab_offset + L[ax] > c->slab_global)
            return fail(SPIN_ERR_INVALID_ARG, "slab: need even global extent >= local, even offset, offset + local <= global");
        if (c->coupling_kind == SPIN_J_BOND_PM1) return fail(SPIN_ERR_UNSUPPORTED, "slab decomposition with per-bond couplings");
        if ((uint64_t)L[0] * L[1] * (out->d == 3 ? (uint64_t)c->slab_global : 1ull) >= (1ull << 32) ||
            (out->d == 2 && (uint64_t)L[0] * c->slab_global >= (1ull << 32)))
            return fail(SPIN_ERR_UNSUPPORTED, "slab: the global lattice must have fewer than 2^32 sites");
        out->axis = ax;
        out->pad[ax] = L[ax] + 4;
    }
    out->N = (uint64_t)out->pad[0] * (uint64_t)out->pad[1] * (uint64_t)out->pad[2];
    if (out->N * (uint64_t)c->n_replicas >= (1ull << 31))
        return fail(SPIN_ERR_UNSUPPORTED, "N * n_replicas must stay below 2^31");
    const int used = c->coupling_kind == SPIN_J_UNIFORM ? 1 : (c->coupling_kind == SPIN_J_PER_DIRECTION ? out->d : 0);
    for (int mu = 0; mu < used; ++mu)
        if (!std::isfinite(c->J[mu])) return fail(SPIN_ERR_INVALID_ARG, "J must be finite");
    if (c->n == 1) {
        for (int mu = 0; mu < used; ++mu)
            if (!(c->J[mu] == -1.0 || c->J[mu] == 0.0 || c->J[mu] == 1.0))
                return fail(SPIN_ERR_UNSUPPORTED, "n = 1 supports couplings in {-1, 0, +1} only (integer table)");
        const bool unit_uniform = c->coupling_kind == SPIN_J_UNIFORM && c->J[0] != 0.0;
        if (c->storage == SPIN_STORE_MSC) {
            // replica-per-bit multi-spin coding: 32 realisations per word, one random number per site for all
            if (c->coupling_kind != SPIN_J_BOND_PM1 || c->replica_streams != 0)
                return fail(SPIN_ERR_UNSUPPORTED, "MSC storage is for per-bond +-1 couplings with a shared update stream (replica_streams = 0)");
            if (c->n_replicas % 32) return fail(SPIN_ERR_UNSUPPORTED, "MSC storage needs n_replicas %% 32 == 0");
            if ((out->N / 2) % 32) return fail(SPIN_ERR_UNSUPPORTED, "MSC storage needs N / 2 %% 32 == 0");
            out->path = PATH_ISING_MSC;
        } else if (c->storage == SPIN_STORE_BITPACK) {
            if (L[0] % 64) return fail(SPIN_ERR_UNSUPPORTED, "BITPACK storage needs Lx %% 64 == 0");
            if (!(unit_uniform || c->coupling_kind == SPIN_J_BOND_PM1))
                return fail(SPIN_ERR_UNSUPPORTED, "BITPACK storage needs uniform J = +-1 or per-bond +-1 couplings");
            out->path = PATH_ISING_BITPACK;
        } else {
            out->path = (L[0] % 64 == 0 && unit_uniform) ? PATH_ISING_INT8 : PATH_ISING_GENERIC;
        }
    } else {
        if (c->coupling_kind == SPIN_J_BOND_PM1) return fail(SPIN_ERR_UNSUPPORTED, "per-bond couplings are n = 1 only");
        out->path = PATH_VECTOR;
    }
    return SPIN_OK;
}

static uint32_t measure_blocks(uint64_t work_items) {
    uint64_t b = (work_items + 255) / 256;
    if (b > 592) b = 592;  // 4 CTAs per SM on 148 SMs
    if (b < 1) b = 1;
    return (uint32_t)b;
}

// TMA-staged kernel of the n >= 2 models: rows per tile, and CTAs per replica for S steps, R replicas and room for `cap` CTAs
static uint32_t tma_tile_rows(uint32_t RL) { return RL <= 128 ? 8u : 4u; }
static uint32_t tma_grid_x(uint64_t S, uint64_t R, uint64_t cap) {
    uint64_t gx = cap / R;
    if (gx < 1) gx = 1;
    if (gx > S) gx = S;
    return (uint32_t)gx;
}
constexpr uint64_t TMA_MAX_CTAS = 512;
constexpr uint32_t FINALIZE_BLOCKS = 128;   // first-level blocks of vector_partials_finalize

// Exact temporal blocking (two sweeps per pass, ising_tblock_kernel.cuh) is offered for the 2D Ising int8 fast layout with uniform
// couplings and the Metropolis rule when a row of one colour is 32 .. 512 words; it needs a second pair of colour arrays.
static bool tblock_offered(const spin_config *c, const Derived &dv) {
    if (c->n != 1 || dv.d != 2 || dv.axis >= 0) return false;
    // int8 storage only: the bit-packed lattices are L2-resident and gain nothing (measured 55.2 vs 55.6 us at L = 16384)
    if (dv.path != PATH_ISING_INT8 || c->coupling_kind != SPIN_J_UNIFORM) return false;
    if (c->n_replicas > 1 && !c->replica_streams) return false;   // shared-stream replicas take the mask-reuse kernels
    const int32_t WX = dv.pad[0] / 64;
    return WX >= 32 && WX <= 512 && WX % 32 == 0;
}

// slots of the n = 1 accumulators: as many as 64, fewer when there are many replicas (8192 / R rounded down to a power of two)
static uint32_t acc_slots_for(uint64_t R) {
    uint32_t k = 64;
    while (k > 1 && (uint64_t)k * R > 8192) k >>= 1;
    return k;
}

static void make_layout(const spin_config *c, const Derived &dv, Layout *l, uint32_t *mblocks) {
    const uint64_t Nh = dv.N / 2, R = (uint64_t)c->n_replicas;
    size_t off = 0;
    if (dv.path == PATH_ISING_BITPACK || dv.path == PATH_ISING_MSC) l->bytes_s = (size_t)(R * Nh / 8);
    else if (dv.path == PATH_VECTOR) l->bytes_s = (size_t)(R * Nh * c->n * sizeof(float));
    else l->bytes_s = (size_t)(R * Nh);
    for (int k = 0; k < 2; ++k) { l->off_s[k] = off; off += align_up(l->bytes_s); }
    for (int k = 0; k < 2; ++k) {
        l->off_alt[k] = l->off_s[k];
        if (tblock_offered(c, dv)) { l->off_alt[k] = off; off += align_up(l->bytes_s); }
    }
    l->bytes_bonds = 0;
    if (c->coupling_kind == SPIN_J_BOND_PM1)
        l->bytes_bonds = dv.path == PATH_ISING_BITPACK ? (size_t)(2 * R * 3 * (Nh / 32) * 4)
                       : dv.path == PATH_ISING_MSC ? (size_t)(2 * (R / 32) * dv.d * Nh * 4) : (size_t)(R * dv.d * dv.N);
    l->off_bonds = off; off += align_up(l->bytes_bonds);
    *mblocks = measure_blocks(dv.path == PATH_ISING_BITPACK || dv.path == PATH_ISING_INT8 ? Nh / 32 : Nh);
    uint64_t pblocks = *mblocks;   // n >= 2: per-CTA partials of the measurement pass or of the fused TMA half-sweep
    if (c->n > 1 && dv.d == 3) {
        const uint32_t ty = tma_tile_rows((uint32_t)dv.pad[0] / 2);
        const uint64_t S = (uint64_t)((dv.pad[1] + ty - 1) / ty) * dv.pad[2];
        const uint64_t gx = tma_grid_x(S, R, TMA_MAX_CTAS);
        if (gx > pblocks) pblocks = gx;
    }
    // n >= 2, rows of whole quads: the fused strip kernel leaves one partial per CTA (at least 32 quads each)
    if (c->n > 1 && (dv.pad[0] / 2) % 4 == 0 && Nh / 128 + 4 > pblocks) pblocks = Nh / 128 + 4;   // CTAs of >= 32 quads
    const size_t part_bytes = c->n == 1 ? (size_t)(acc_slots_for(R) * R * 2 * sizeof(long long)) : (size_t)(R * pblocks * (1 + c->n) * sizeof(double));
    l->off_acc = off;
    l->off_mid = off + align_up(part_bytes);
    l->off_cnt = l->off_mid + (c->n == 1 ? 0 : align_up((size_t)(R * FINALIZE_BLOCKS * (1 + c->n) * sizeof(double))));
    l->bytes_acc = (l->off_cnt - off) + (c->n == 1 ? 0 : align_up((size_t)(R * sizeof(unsigned))));
    off += align_up(l->bytes_acc);
    l->bytes_res = (size_t)(R * (1 + c->n) * sizeof(double));
    l->off_res = off; off += align_up(l->bytes_res);
    l->total = off;
}

static SetupArgs setup_args(const spin_system *s) {
    SetupArgs a;
    a.g = s->g; a.keys = s->keys; a.R = s->R;
    a.bitpack = s->path == PATH_ISING_BITPACK;
    a.int8perm = s->path == PATH_ISING_INT8;
    a.nc = s->n;
    return a;
}

static int grid_for(const spin_system *s, uint64_t work_items) {
    uint64_t need = (work_items + s->block - 1) / s->block;
    uint64_t cap = (uint64_t)s->sm_count * (2048 / s->block) * (uint64_t)s->grid_num / (uint64_t)s->grid_den;
    if (cap < 1) cap = 1;
    if (need > cap) need = cap;
    if (need < 1) need = 1;
    return (int)need;
}

// ------------------------------------------------------------------- Boltzmann table ---------
// T(dE) = floor(exp(-beta dE) 2^32), 0 <= T <= 2^32, in double (R-4, R-5).
static void build_table(double beta, IsingTable *tab) {
    std::memset(tab, 0, sizeof *tab);
    for (int dE = 0; dE <= 12; ++dE) {
        const double scaled = std::ldexp(std::exp(-beta * (double)dE), 32);
        uint64_t T;
        if (!(scaled < 4294967296.0)) T = 4294967296ull;
        else if (!(scaled > 0.0)) T = 0ull;
        else T = (uint64_t)std::floor(scaled);
        if (T >= 4294967296ull) { tab->Talways |= 1u << dE; tab->T[dE] = 0xFFFFFFFFu; }
        else tab->T[dE] = (uint32_t)T;
    }
    for (int th = 0; th < 3; ++th) {
        const int dE = 4 * (th + 1);
        tab->always[th] = ((tab->Talways >> dE) & 1u) ? 0xFFFFFFFFu : 0u;
        for (int k = 0; k < 32; ++k) tab->digit[th][k] = ((tab->T[dE] >> (31 - k)) & 1u) ? 0xFFFFFFFFu : 0u;
    }
}

// Heat-bath probabilities: T_hb(h) = floor(2^32 / (1 + exp(-2 beta h))), h = -6 .. 6, in double.
// digit[k] / always[k] serve the bit-sliced kernels, indexed by the number k of neighbour terms equal to -1
// (h = q - 2 k, q = 2 d neighbours).
static void build_hb_table(double beta, int q, HeatBathTable *hb) {
    std::memset(hb, 0, sizeof *hb);
    uint64_t T[13];
    for (int h = -6; h <= 6; ++h) {
        const double scaled = std::ldexp(1.0 / (1.0 + std::exp(-2.0 * beta * (double)h)), 32);
        uint64_t v;
        if (!(scaled < 4294967296.0)) v = 4294967296ull;
        else if (!(scaled > 0.0)) v = 0ull;
        else v = (uint64_t)std::floor(scaled);
        T[h + 6] = v;
        if (v >= 4294967296ull) { hb->Talways |= 1u << (h + 6); hb->T[h + 6] = 0xFFFFFFFFu; }
        else hb->T[h + 6] = (uint32_t)v;
    }
    for (int k = 0; k <= q && k < 7; ++k) {
        const int h = q - 2 * k;
        hb->always[k] = T[h + 6] >= 4294967296ull ? 0xFFFFFFFFu : 0u;
        for (int dg = 0; dg < 32; ++dg) hb->digit[k][dg] = ((hb->T[h + 6] >> (31 - dg)) & 1u) ? 0xFFFFFFFFu : 0u;
    }
}

static IsingArgs ising_args(const spin_system *s) {
    IsingArgs a;
    a.g = s->g; a.keys = s->keys; a.tab = s->tab;
    a.s[0] = s->ws + s->lay.off_s[0];
    a.s[1] = s->ws + s->lay.off_s[1];
    a.bonds = s->lay.bytes_bonds ? s->ws + s->lay.off_bonds : nullptr;
    a.R = s->R; a.replica_streams = s->cfg.replica_streams ? 1u : 0u;
    a.t = (uint32_t)s->t; a.colour = 0; a.rho_off = 0;
    a.coupling_kind = s->cfg.coupling_kind;
    for (int mu = 0; mu < 3; ++mu)
        a.Jdir[mu] = s->cfg.coupling_kind == SPIN_J_UNIFORM ? (int)s->cfg.J[0]
                   : (s->cfg.coupling_kind == SPIN_J_PER_DIRECTION ? (mu < s->d ? (int)s->cfg.J[mu] : 0) : 0);
    a.jneg = (s->cfg.coupling_kind == SPIN_J_UNIFORM && s->cfg.J[0] < 0.0) ? 1u : 0u;
    a.rule = s->cfg.update_rule == SPIN_UPDATE_HEATBATH ? 1u : 0u;
    a.prefetch = s->l2_prefetch < 0 ? 0u : (uint32_t)s->l2_prefetch;   // +-J quad kernel: replicas ahead (no gain measured: off)
    a.hb = s->hb;
    a.acc = (long long *)(s->ws + s->lay.off_acc);
    a.acc_slots = acc_slots_for(s->R);
    // +-J quad kernel: L2 eviction hints when spins + coupling words do not fit in L2 anyway: keep the spins and the coupling words
    // of as many replicas as fit in two thirds of L2 (measured at 256^3 x 16: 4 .. 8 replicas 28.8 us, 0 30.8, 12 32.4, no hints 32.9)
    a.defer_cap = (uint32_t)s->defer_cap;
    a.l2_keep = 0xFFFFFFFFu;
    if (s->l2_keep >= 0) a.l2_keep = (uint32_t)s->l2_keep;
    else if (s->l2_keep == -1 && s->lay.bytes_bonds && s->l2_bytes > 0) {
        const double budget = 0.66 * (double)s->l2_bytes, spins = 2.0 * (double)s->lay.bytes_s, per_rep = (double)s->lay.bytes_bonds / s->R;
        if (spins + (double)s->lay.bytes_bonds > 0.6 * (double)s->l2_bytes && spins < budget) {
            double k = (budget - spins) / per_rep;
            a.l2_keep = k >= (double)s->R ? s->R : (uint32_t)k;
        }
    }
    a.alt[0] = s->ws + s->lay.off_alt[0];
    a.alt[1] = s->ws + s->lay.off_alt[1];
    a.tb_rows = 0;
    return a;
}

static VectorArgs vector_args(const spin_system *s, double beta) {
    VectorArgs a;
    a.g = s->g; a.keys = s->keys;
    a.s[0] = (float *)(s->ws + s->lay.off_s[0]);
    a.s[1] = (float *)(s->ws + s->lay.off_s[1]);
    a.R = s->R; a.replica_streams = s->cfg.replica_streams ? 1u : 0u;
    a.t = (uint32_t)s->t; a.colour = 0; a.rho_off = 0;
    for (int mu = 0; mu < 3; ++mu)
        a.Jdir[mu] = s->cfg.coupling_kind == SPIN_J_UNIFORM ? (float)s->cfg.J[0] : (mu < s->d ? (float)s->cfg.J[mu] : 0.0f);
    a.beta = (float)beta;
    a.rule = s->cfg.update_rule == SPIN_UPDATE_HEATBATH ? 1u : 0u;
    // strip kernel: CTAs ahead; default = one wave of resident CTAs (9 of 128 threads per SM at 52 registers)
    a.prefetch = s->l2_prefetch < 0 ? (uint32_t)s->sm_count * 9u : (uint32_t)s->l2_prefetch;
    a.part = (double *)(s->ws + s->lay.off_acc);
    return a;
}

// rows and planes a launch with geometry g updates (Geometry::sw_*): the strips of the fast kernels are cut from these
static uint32_t sweep_rows(const Geometry &g) { return g.d == 2 ? g.sw_pn : (uint32_t)g.Ly; }
static uint32_t sweep_planes(const Geometry &g) { return g.d == 3 ? g.sw_pn : (uint32_t)g.Lz; }
// does the launch update less than the whole local lattice (slab handle, half-sweep in pieces)?  Then the RANGED instances of
// the strip kernels run (rows per thread 1 or 4 only); the whole-lattice instances carry no offsets (4 % faster at 512^3)
static bool is_ranged(const Geometry &g) { return g.sw_p0 != 0u || g.sw_pn != (uint32_t)(g.d == 3 ? g.Lz : g.Ly); }

// ----------------------------------------------------------------------------- launches ------
// fused: NULL, or (colour 1 only) ask for E / M to be accumulated into a.acc by the half-sweep itself;
// *fused tells whether the kernel that ran could do it (the strip kernels with 1 or 4 rows per thread).
static spin_status launch_halfsweep_ising(spin_system *s, const IsingArgs &a, cudaStream_t st, bool *fused = nullptr) {
    const bool bonds = s->cfg.coupling_kind == SPIN_J_BOND_PM1;
    const bool shared = s->R > 1 && !s->cfg.replica_streams;
    const int B = s->path == PATH_ISING_INT8 && s->block > 128 ? 128 : s->block;   // the int8 kernel is built for <= 128 threads
    if (fused) *fused = false;
    if (s->path == PATH_ISING_MSC) {
        // replica-per-bit words: thread = site, lanes of a warp = the 32 sites of a Philox unit; the groups of 32 realisations
        // are cut into chunks over gridDim.y so that the GPU is full, but not below 8 groups per thread (the site's uniform is
        // assembled once per thread)
        const uint32_t G = s->R / 32;
        const int Bm = s->g.Nh < 128u ? (int)s->g.Nh : 128;
        uint64_t Gy = (uint64_t)s->sm_count * 1024 * (uint64_t)s->grid_num / ((uint64_t)s->grid_den * s->g.Nh);
        if (Gy > G / 8) Gy = G / 8;
        if (Gy < 1) Gy = 1;
        const dim3 Gm((s->g.Nh + Bm - 1) / Bm, (unsigned)Gy);
        const bool hb = s->cfg.update_rule == SPIN_UPDATE_HEATBATH;
        if (s->d == 2) { if (hb) ising_msc_halfsweep<2, true><<<Gm, Bm, 0, st>>>(a); else ising_msc_halfsweep<2, false><<<Gm, Bm, 0, st>>>(a); }
        else { if (hb) ising_msc_halfsweep<3, true><<<Gm, Bm, 0, st>>>(a); else ising_msc_halfsweep<3, false><<<Gm, Bm, 0, st>>>(a); }
    } else if (s->path == PATH_ISING_GENERIC) {
        ising_generic_halfsweep<<<grid_for(s, (uint64_t)a.g.sw_jn * s->R), B, 0, st>>>(a);
    } else if (s->path == PATH_ISING_INT8) {
        // one thread per (replica, z, strip of K rows, unit column)
        const bool hb = s->cfg.update_rule == SPIN_UPDATE_HEATBATH;
        // rows per thread: the caller's choice, else 4 when that still leaves every SM several CTAs and 1 otherwise
        // (a thread walks its rows one after the other: on small grids more threads beat fewer halo loads);
        // the heat-bath kernel is instantiated for K = 4 only
        int K = s->strip_rows;
        if (!s->strip_rows_set) {
            const uint64_t threads4 = (uint64_t)s->g.WX * ((sweep_rows(a.g) + 3) / 4) * sweep_planes(a.g) * s->R;
            K = threads4 >= (uint64_t)s->sm_count * 2048 ? 4 : 1;
        }
        if (hb) K = 4;
        const bool ranged = is_ranged(a.g);
        if (ranged) K = K >= 4 ? 4 : 1;
        const uint64_t items = (uint64_t)s->g.WX * ((sweep_rows(a.g) + K - 1) / K) * sweep_planes(a.g) * s->R;
        const int G = (int)((items + B - 1) / B);
        if (ranged) {
#define I8R(D_, K_, HB_) ising_int8_halfsweep<D_, K_, HB_, false, true><<<G, B, 0, st>>>(a)
            if (hb) { if (s->d == 2) I8R(2, 4, true); else I8R(3, 4, true); }
            else if (s->d == 2) { if (K == 1) I8R(2, 1, false); else I8R(2, 4, false); }
            else { if (K == 1) I8R(3, 1, false); else I8R(3, 4, false); }
#undef I8R
        } else
        if (fused && (K == 1 || K == 4) && a.colour == 1u) {
            *fused = true;
#define I8M(D_, K_, HB_) ising_int8_halfsweep<D_, K_, HB_, true><<<G, B, 0, st>>>(a)
            if (hb) { if (s->d == 2) I8M(2, 4, true); else I8M(3, 4, true); }
            else if (s->d == 2) { if (K == 1) I8M(2, 1, false); else I8M(2, 4, false); }
            else { if (K == 1) I8M(3, 1, false); else I8M(3, 4, false); }
#undef I8M
        } else
#define I8(D_, K_) ising_int8_halfsweep<D_, K_><<<G, B, 0, st>>>(a)
        if (hb) { if (s->d == 2) ising_int8_halfsweep<2, 4, true><<<G, B, 0, st>>>(a); else ising_int8_halfsweep<3, 4, true><<<G, B, 0, st>>>(a); }
        else if (s->d == 2) { if (K == 1) I8(2, 1); else if (K == 2) I8(2, 2); else if (K == 4) I8(2, 4); else if (K == 8) I8(2, 8); else I8(2, 16); }
        else { if (K == 1) I8(3, 1); else if (K == 2) I8(3, 2); else if (K == 4) I8(3, 4); else if (K == 8) I8(3, 8); else I8(3, 16); }
#undef I8
    } else if (!bonds && !shared && !s->vector_generic) {
        // uniform couplings, own random numbers per word: the strip kernel (K rows per thread, as for int8;
        // measured at L = 16384: 65.7 / 61.6 / 58.4 / 65.8 / 71.9 us for K = 1 / 2 / 4 / 8 / 16)
        int K = s->strip_rows_set ? s->strip_rows : 0;
        if (!K) {
            const uint64_t threads4 = (uint64_t)s->g.WX * ((sweep_rows(a.g) + 3) / 4) * sweep_planes(a.g) * s->R;
            K = threads4 >= (uint64_t)s->sm_count * 2048 ? 4 : 1;
        }
        if (K > 4) K = 4;
        const bool ranged = is_ranged(a.g);
        if (ranged && K == 2) K = 1;
        const int Bs = B > 128 ? 128 : B;
        const uint64_t items = (uint64_t)s->g.WX * ((sweep_rows(a.g) + K - 1) / K) * sweep_planes(a.g) * s->R;
        const int G = (int)((items + Bs - 1) / Bs);
        const bool hb = s->cfg.update_rule == SPIN_UPDATE_HEATBATH;
#define BS3(D_, K_) do { if (hb) ising_bitpack_strip_halfsweep<D_, K_, true><<<G, Bs, 0, st>>>(a); else ising_bitpack_strip_halfsweep<D_, K_, false><<<G, Bs, 0, st>>>(a); } while (0)
#define BS2(D_) do { if (K == 1) BS3(D_, 1); else if (K == 2) BS3(D_, 2); else BS3(D_, 4); } while (0)
#define BM3(D_, K_) do { if (hb) ising_bitpack_strip_halfsweep<D_, K_, true, true><<<G, Bs, 0, st>>>(a); else ising_bitpack_strip_halfsweep<D_, K_, false, true><<<G, Bs, 0, st>>>(a); } while (0)
#define BR3(D_, K_) do { if (hb) ising_bitpack_strip_halfsweep<D_, K_, true, false, true><<<G, Bs, 0, st>>>(a); else ising_bitpack_strip_halfsweep<D_, K_, false, false, true><<<G, Bs, 0, st>>>(a); } while (0)
        if (ranged) {
            if (s->d == 2) { if (K == 1) BR3(2, 1); else BR3(2, 4); } else { if (K == 1) BR3(3, 1); else BR3(3, 4); }
        } else
#undef BR3
        if (fused && (K == 1 || K == 4) && a.colour == 1u) {
            *fused = true;
            if (s->d == 2) { if (K == 1) BM3(2, 1); else BM3(2, 4); } else { if (K == 1) BM3(3, 1); else BM3(3, 4); }
        } else
        if (s->d == 2) BS2(2); else BS2(3);
#undef BM3
#undef BS2
#undef BS3
    } else if (bonds && !shared && s->g.WX % 4 == 0 && !s->vector_generic && s->variant != 1 && s->cfg.update_rule != SPIN_UPDATE_HEATBATH &&
               !(fused && a.colour == 1u)) {
        // per-bond couplings, own update stream per replica (or one replica), Lx % 256 == 0: one thread per quad, deferred digit tails
        const int Bq = 128;
        const uint64_t quads = (uint64_t)s->g.NW / 4;
        unsigned Gy = 1;
        if (quads < (uint64_t)s->sm_count * 512) {
            uint64_t want = ((uint64_t)s->sm_count * 512 + quads - 1) / quads;   // replica chunks that fill the GPU
            if (want > s->R) want = s->R;
            Gy = (unsigned)(want < 1 ? 1 : want);
        }
        const dim3 G((unsigned)((quads + Bq - 1) / Bq), Gy);
        if (s->d == 2) ising_pmj_quad_own_halfsweep<2><<<G, Bq, 0, st>>>(a); else ising_pmj_quad_own_halfsweep<3><<<G, Bq, 0, st>>>(a);
    } else if (bonds && shared && s->g.WX % 4 == 0 && !s->vector_generic) {
        // Lx % 256 == 0: one thread per quad of four words, 128-bit accesses (ising_pmj_quad_halfsweep).
        // All replicas in one thread when the quads alone give every SM >= 256 threads (measured at 256^3, R = 16:
        // 35.2 / 37.1 / 35.2 / 47.4 / 78.1 us for 1 / 2 / 4 / 8 / 16 replica chunks), else chunks of >= 4 replicas
        const uint64_t quads = (uint64_t)s->g.NW / 4;
        const bool hb = s->cfg.update_rule == SPIN_UPDATE_HEATBATH;
        if (s->variant != 1 && s->R >= 2) {
            // cooperative kernel (default; with the L2 eviction hints 26.8 vs 28.8 us at 256^3 x 16, and faster on small lattices):
            // a CTA of CH warps per 32 quads, warp c serves replica chunk c
            int CH = (s->block > 128 ? 128 : s->block) / 32;
            while (CH > 1 && (uint32_t)CH > s->R) CH /= 2;
            const dim3 G((unsigned)((quads + 31) / 32));
            const int Bc = 32 * CH;
            const bool meas = fused && a.colour == 1u;   // row a7: E and M from the bond masks of the colour-1 half-sweep
            if (meas) *fused = true;
#define PC(D_, HB_) do { if (meas) ising_pmj_quad_coop_halfsweep<D_, HB_, true><<<G, Bc, 0, st>>>(a); else ising_pmj_quad_coop_halfsweep<D_, HB_, false><<<G, Bc, 0, st>>>(a); } while (0)
            if (s->d == 2) { if (hb) PC(2, true); else PC(2, false); }
            else { if (hb) PC(3, true); else PC(3, false); }
#undef PC
        } else {
        const int Bq = s->block < 128 ? s->block : 128;
        unsigned Gy = 1;
        if (quads < (uint64_t)s->sm_count * 256) {
            uint64_t want = ((uint64_t)s->sm_count * 256 + quads - 1) / quads;   // chunks that would fill the GPU
            const uint64_t most = (s->R + 3) / 4;
            if (want > most) want = most;
            Gy = (unsigned)(want < 1 ? 1 : want);
        }
        const dim3 G((unsigned)((quads + Bq - 1) / Bq), Gy);
        if (fused && a.colour == 1u) {
            // colour-1 half-sweep of a recorded sweep: E and M from the bond masks it forms anyway (row a7)
            *fused = true;
            if (s->d == 2) { if (hb) ising_pmj_quad_halfsweep<2, true, true><<<G, Bq, 0, st>>>(a); else ising_pmj_quad_halfsweep<2, false, true><<<G, Bq, 0, st>>>(a); }
            else { if (hb) ising_pmj_quad_halfsweep<3, true, true><<<G, Bq, 0, st>>>(a); else ising_pmj_quad_halfsweep<3, false, true><<<G, Bq, 0, st>>>(a); }
        } else
        if (s->d == 2) { if (hb) ising_pmj_quad_halfsweep<2, true><<<G, Bq, 0, st>>>(a); else ising_pmj_quad_halfsweep<2, false><<<G, Bq, 0, st>>>(a); }
        else { if (hb) ising_pmj_quad_halfsweep<3, true><<<G, Bq, 0, st>>>(a); else ising_pmj_quad_halfsweep<3, false><<<G, Bq, 0, st>>>(a); }
        }
    } else {
        // shared update stream: chunks of >= 16 replicas per thread (the masks of a word are built once per chunk);
        // more chunks only when the lattice alone cannot fill the GPU (many realisations of a small lattice)
        int Bq = B;
        const uint32_t NWs = a.g.sw_jn >> 5;   // words this launch updates
        while (Bq > 32 && (uint32_t)(Bq / 2) >= NWs) Bq /= 2;   // small lattices: no dead threads
        const int Gx = (int)((NWs + Bq - 1) / Bq) < grid_for(s, NWs) ? (int)((NWs + Bq - 1) / Bq) : grid_for(s, NWs);
        int Gy = 1;
        if (shared && s->R > 16) {
            // replicas per thread: 16 when the lattice fills the GPU, down to 4 when it is the replicas that must
            uint64_t per = (uint64_t)s->g.NW * s->R / ((uint64_t)s->sm_count * 1024);
            if (per > 16) per = 16;
            if (per < 4) per = 4;
            Gy = (int)((s->R + per - 1) / per);
            if (Gy > 65535) Gy = 65535;
        }
        const dim3 G(Gx, Gy);
        const bool meas = fused && a.colour == 1u && s->cfg.update_rule != SPIN_UPDATE_HEATBATH;   // row a7, Metropolis kernels
        if (meas) *fused = true;
#define BP(D_, BONDS_, SH_)                                                                      \
    do {                                                                                         \
        if (s->cfg.update_rule == SPIN_UPDATE_HEATBATH) ising_bitpack_halfsweep_hb<D_, BONDS_, SH_><<<G, Bq, 0, st>>>(a); \
        else if (meas) ising_bitpack_halfsweep<D_, BONDS_, SH_, true><<<G, Bq, 0, st>>>(a);     \
        else ising_bitpack_halfsweep<D_, BONDS_, SH_><<<G, Bq, 0, st>>>(a);                     \
    } while (0)
        if (s->d == 2) {
            if (bonds) { if (shared) BP(2, true, true); else BP(2, true, false); }
            else { if (shared) BP(2, false, true); else BP(2, false, false); }
        } else {
            if (bonds) { if (shared) BP(3, true, true); else BP(3, true, false); }
            else { if (shared) BP(3, false, true); else BP(3, false, false); }
        }
#undef BP
    }
    s->launches += 1;
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

// cuTensorMapEncodeTiled through the runtime (no link against libcuda); NULL if the driver does not offer it
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// Tensor maps of the two colour arrays float [R][NC][Lz][Ly][RL] for the TMA-staged kernel: a box of TY rows and a
// box of one row, each over all NC components.  Leaves tma_ok = 0 (strip kernel) when the shape does not qualify.
static void tma_prepare(spin_system *s) {
    s->tma_ok = 0;
    const Geometry &g = s->g;
    if (s->path != PATH_VECTOR || s->d != 3 || g.RL % 4 != 0 || g.RL > 256 || s->R > 65535) return;
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return;
    s->tma_ty = tma_tile_rows(g.RL);
    const cuuint64_t dims[5] = {g.RL, (cuuint64_t)g.Ly, (cuuint64_t)g.Lz, (cuuint64_t)s->n, s->R};
    const cuuint64_t strides[4] = {(cuuint64_t)g.RL * 4, (cuuint64_t)g.RL * g.Ly * 4, (cuuint64_t)g.Nh * 4, (cuuint64_t)g.Nh * 4 * s->n};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    for (int c = 0; c < 2; ++c) {
        void *base = s->ws + s->lay.off_s[c];
        const cuuint32_t box_main[5] = {g.RL, s->tma_ty, 1, (cuuint32_t)s->n, 1};
        const cuuint32_t box_row[5] = {g.RL, 1, 1, (cuuint32_t)s->n, 1};
        if (enc(&s->tma_main[c], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, base, dims, strides, box_main, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return;
        if (enc(&s->tma_row[c], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, base, dims, strides, box_row, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return;
    }
    s->tma_ok = 1;
}

template <int NC, bool UNITJ, bool HB, bool MEAS>
static cudaError_t launch_tma(const VectorTmaArgs &ta, dim3 G, size_t smem, cudaStream_t st) {
    static size_t configured = 0;   // dynamic shared memory this instantiation has been allowed so far
    if (configured < smem) {
        cudaError_t e = cudaFuncSetAttribute(vector_tma_halfsweep<NC, UNITJ, HB, MEAS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    vector_tma_halfsweep<NC, UNITJ, HB, MEAS><<<G, TMA_THREADS, smem, st>>>(ta);
    return cudaGetLastError();
}

// CTAs per replica of the TMA-staged kernel on this device
static uint32_t tma_ctas(const spin_system *s, bool hb, bool meas) {
    const uint64_t S = (uint64_t)((s->g.Ly + s->tma_ty - 1) / s->tma_ty) * s->g.Lz;
    uint64_t cap = (uint64_t)s->sm_count * tma_ctas_per_sm(hb, meas) * (uint64_t)s->grid_num / (uint64_t)s->grid_den;
    if (cap > TMA_MAX_CTAS) cap = TMA_MAX_CTAS;
    if (cap < 1) cap = 1;
    return tma_grid_x(S, s->R, cap);
}

// n >= 2.  d = 3 with rows of at most 256 sites per colour: the TMA-staged kernel (tiles + halo in shared memory, ring over
// z); otherwise the strip kernel (128-bit accesses, K rows per thread) when a row holds whole quads of 4 sites, else the
// one-thread-per-site kernel.  fused: NULL, or (colour 1) ask for E / M partials from the half-sweep itself (row a7);
// *fused = number of per-replica partials written (0: this kernel cannot, run the measurement pass).
static spin_status launch_halfsweep_vector(spin_system *s, const VectorArgs &a, cudaStream_t st, bool allow_tma = true,
                                           uint32_t *fused = nullptr, bool *two_level = nullptr) {
    const Geometry &g = s->g;
    const bool hb = s->cfg.update_rule == SPIN_UPDATE_HEATBATH;
    const bool strip_ok = g.RL % 4 == 0 && !s->vector_generic && s->R <= 65535;
    if (fused) *fused = 0;
    // the staged kernel serves (a) every half-sweep when SPIN_OPT_TMA_KERNELS is on, (b) by default only the colour-1 half-sweep
    // of a recorded sweep, whose fused E / M saves the measurement pass (the strip kernel is faster otherwise: profiles/)
    const bool want_fused = fused && a.colour == 1u;
    if (two_level) *two_level = false;
    if (want_fused && strip_ok && s->use_tma != 1 && two_level) {
        // colour-1 half-sweep of a recorded sweep: the strip kernel (one row per thread) with E / M fused, one partial per warp
        bool unitj = true;
        for (int mu = 0; mu < s->d; ++mu) unitj = unitj && a.Jdir[mu] == 1.0f;
        const int B = s->block > 128 ? 128 : s->block;
        const uint64_t items = (uint64_t)(g.RL / 4) * sweep_rows(a.g) * sweep_planes(a.g);
        const dim3 G((unsigned)((items + B - 1) / B), s->R);
#define VM4(NC_, D_, U_, HB_) vector_strip_halfsweep<NC_, D_, U_, 1, HB_, true><<<G, B, 0, st>>>(a)
#define VM3(NC_, D_, HB_) do { if (unitj) VM4(NC_, D_, true, HB_); else VM4(NC_, D_, false, HB_); } while (0)
        if (s->n == 2) { if (s->d == 2) VM3(2, 2, false); else VM3(2, 3, false); }
        else if (hb) { if (s->d == 2) VM3(3, 2, true); else VM3(3, 3, true); }
        else { if (s->d == 2) VM3(3, 2, false); else VM3(3, 3, false); }
#undef VM3
#undef VM4
        CUDA_TRY(cudaGetLastError());
        *fused = G.x;
        *two_level = true;
        s->launches += 1;
        return SPIN_OK;
    }
    if (allow_tma && s->tma_ok && (s->use_tma == 1 || (s->use_tma < 0 && want_fused)) && !s->vector_generic) {
        bool unitj = true;
        for (int mu = 0; mu < s->d; ++mu) unitj = unitj && a.Jdir[mu] == 1.0f;
        VectorTmaArgs ta;
        ta.v = a;
        for (int c = 0; c < 2; ++c) { ta.main_map[c] = s->tma_main[c]; ta.row_map[c] = s->tma_row[c]; }
        ta.TY = s->tma_ty;
        ta.nyb = ((uint32_t)g.Ly + s->tma_ty - 1) / s->tma_ty;
        ta.part = (double *)(s->ws + s->lay.off_acc);
        const bool meas = fused && a.colour == 1u;
        const dim3 G(tma_ctas(s, hb, meas), s->R);
        const size_t smem = tma_smem_bytes(s->n, (int)s->tma_ty, g.RL);
        cudaError_t e;
#define TM4(NC_, U_, HB_, M_) e = launch_tma<NC_, U_, HB_, M_>(ta, G, smem, st)
#define TM3(NC_, U_, HB_) do { if (meas) TM4(NC_, U_, HB_, true); else TM4(NC_, U_, HB_, false); } while (0)
#define TM2(NC_, HB_) do { if (unitj) TM3(NC_, true, HB_); else TM3(NC_, false, HB_); } while (0)
        if (s->n == 2) TM2(2, false);
        else if (hb) TM2(3, true);
        else TM2(3, false);
#undef TM2
#undef TM3
#undef TM4
        if (e != cudaSuccess) return fail(SPIN_ERR_CUDA, "TMA half-sweep launch: %s", cudaGetErrorString(e));
        if (meas) *fused = G.x;
        s->launches += 1;
        return SPIN_OK;
    }
    if (strip_ok && hb) {
        // heat bath (n = 3): the strip kernel with one row per thread
        bool unitj = true;
        for (int mu = 0; mu < s->d; ++mu) unitj = unitj && a.Jdir[mu] == 1.0f;
        const int B = s->block > 128 ? 128 : s->block;
        const uint64_t items = (uint64_t)(g.RL / 4) * sweep_rows(a.g) * sweep_planes(a.g);
        const dim3 G((unsigned)((items + B - 1) / B), s->R);
#define VH(D_, U_) do { if (is_ranged(a.g)) vector_strip_halfsweep<3, D_, U_, 1, true, false, true><<<G, B, 0, st>>>(a); else vector_strip_halfsweep<3, D_, U_, 1, true><<<G, B, 0, st>>>(a); } while (0)
        if (s->d == 2) { if (unitj) VH(2, true); else VH(2, false); }
        else { if (unitj) VH(3, true); else VH(3, false); }
#undef VH
    } else if (strip_ok) {
        bool unitj = true;
        for (int mu = 0; mu < s->d; ++mu) unitj = unitj && a.Jdir[mu] == 1.0f;
        int K = s->strip_rows_set ? (s->strip_rows >= 4 ? 4 : s->strip_rows) : 1;  // default 1 (measured fastest)
        const bool ranged = is_ranged(a.g);
        if (ranged) K = 1;
        const int B = s->block > 128 ? 128 : s->block;
        const uint64_t items = (uint64_t)(g.RL / 4) * ((sweep_rows(a.g) + K - 1) / K) * sweep_planes(a.g);
        const dim3 G((unsigned)((items + B - 1) / B), s->R);
#define VS4(NC_, D_, U_, K_) vector_strip_halfsweep<NC_, D_, U_, K_><<<G, B, 0, st>>>(a)
#define VS3(NC_, D_, U_) do { if (ranged) vector_strip_halfsweep<NC_, D_, U_, 1, false, false, true><<<G, B, 0, st>>>(a); \
                              else if (K == 1) VS4(NC_, D_, U_, 1); else if (K == 2) VS4(NC_, D_, U_, 2); else VS4(NC_, D_, U_, 4); } while (0)
#define VS2(NC_, D_) do { if (unitj) VS3(NC_, D_, true); else VS3(NC_, D_, false); } while (0)
        if (s->n == 2) { if (s->d == 2) VS2(2, 2); else VS2(2, 3); }
        else { if (s->d == 2) VS2(3, 2); else VS2(3, 3); }
#undef VS2
#undef VS3
#undef VS4
    } else {
        const int G = grid_for(s, (uint64_t)a.g.sw_jn * s->R);
        if (s->n == 2) vector_halfsweep<2><<<G, s->block, 0, st>>>(a);
        else vector_halfsweep<3><<<G, s->block, 0, st>>>(a);
    }
    s->launches += 1;
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

// ------------------------------------------------------------------- temporal blocking -------
static bool graph_ok(const spin_system *s, int64_t n_sweeps);
static void graph_drop(spin_system *s);
static bool tblock_use(const spin_system *s, int64_t n_sweeps) {
    if (!s->tblock_ok || s->tblock == 0 || s->vector_generic || n_sweeps < 2) return false;
    if (s->tblock == 1) return true;
    // auto: int8 storage (where it cuts the HBM traffic to a third; the bit-packed lattices are L2-resident and gain nothing:
    // 55.2 vs 55.6 us at L = 16384) and only where a half-sweep outlasts its launch
    // (the heat-bath instance is ALU-bound either way: 84.3 vs 82.3 us for the strip kernel at L = 16384, so it runs on request only)
    return s->path == PATH_ISING_INT8 && s->cfg.update_rule == SPIN_UPDATE_METROPOLIS && !graph_ok(s, 1 << 20);
}

template <bool INT8, int MAXT, bool HB>
static cudaError_t tblock_launch(const IsingArgs &a, dim3 G, int B, size_t smem, cudaStream_t st) {
    static size_t configured = 0;
    if (configured < smem) {
        cudaError_t e = cudaFuncSetAttribute(ising_tblock2_sweeps<INT8, MAXT, HB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    ising_tblock2_sweeps<INT8, MAXT, HB><<<G, B, smem, st>>>(a);
    return cudaGetLastError();
}

// pairs of sweeps through the temporal-blocking kernel; the colour arrays swap roles after every launch
static spin_status tblock_sweeps(spin_system *s, int64_t pairs, cudaStream_t st) {
    const int B = (int)s->g.WX;
    const size_t smem = tblock_smem_bytes(s->g.WX);
    const bool hb = s->cfg.update_rule == SPIN_UPDATE_HEATBATH;
    // rows per stripe: one wave of resident CTAs (a stripe costs 3 / H redundant row updates; a second wave would idle)
    uint32_t H = (uint32_t)s->tblock_rows;
    if (H == 0) {
        int per_sm = 1;
        cudaError_t e;
        if (B <= 256) e = hb ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ising_tblock2_sweeps<true, 256, true>, B, smem)
                             : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ising_tblock2_sweeps<true, 256, false>, B, smem);
        else e = hb ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ising_tblock2_sweeps<true, 512, true>, B, smem)
                    : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ising_tblock2_sweeps<true, 512, false>, B, smem);
        if (e != cudaSuccess || per_sm < 1) per_sm = 1;
        uint64_t stripes = (uint64_t)s->sm_count * per_sm / s->R;
        if (stripes < 1) stripes = 1;
        H = (uint32_t)(((uint64_t)s->g.Ly + stripes - 1) / stripes);
        if (H < 8) H = 8;
    }
    const dim3 G((unsigned)((s->g.Ly + H - 1) / H), s->R);
    for (int64_t k = 0; k < pairs; ++k) {
        IsingArgs a = ising_args(s);
        a.tb_rows = H;
        cudaError_t e;
        if (B <= 256) e = hb ? tblock_launch<true, 256, true>(a, G, B, smem, st) : tblock_launch<true, 256, false>(a, G, B, smem, st);
        else e = hb ? tblock_launch<true, 512, true>(a, G, B, smem, st) : tblock_launch<true, 512, false>(a, G, B, smem, st);
        if (e != cudaSuccess) return fail(SPIN_ERR_CUDA, "temporal-blocking launch: %s", cudaGetErrorString(e));
        for (int c = 0; c < 2; ++c) { const size_t t = s->lay.off_s[c]; s->lay.off_s[c] = s->lay.off_alt[c]; s->lay.off_alt[c] = t; }
        s->t += 2;
        s->launches += 1;
    }
    graph_drop(s);   // a captured graph holds the array pointers of before the swap
    return SPIN_OK;
}

// One sweep at sweep index t_override (graph capture: the handle is not advanced) or at the handle's counter.
static spin_status enqueue_sweep(spin_system *s, double beta, cudaStream_t st, bool capture = false, uint32_t t_override = 0) {
    if (s->n == 1) {
        IsingArgs a = ising_args(s);
        if (capture) a.t = t_override;
        for (uint32_t colour = 0; colour < 2; ++colour) {
            a.colour = colour;
            spin_status rc = launch_halfsweep_ising(s, a, st);
            if (rc != SPIN_OK) return rc;
        }
    } else {
        VectorArgs a = vector_args(s, beta);
        if (capture) a.t = t_override;
        for (uint32_t colour = 0; colour < 2; ++colour) {
            a.colour = colour;
            // graph replay patches the sweep index into VectorArgs-sized argument blocks: strip kernel only
            spin_status rc = launch_halfsweep_vector(s, a, st, !capture);
            if (rc != SPIN_OK) return rc;
        }
    }
    if (!capture) s->t += 1;
    return SPIN_OK;
}

// ------------------------------------------------------------------------- CUDA graphs -------
// Lattices between the resident kernel's limit and a few million sites are launch-bound: a half-sweep takes less
// time than its launch (the argument block with the tables is ~3 KB).  spin_sweep then replays a graph of
// GRAPH_SWEEPS sweeps.  The kernels are the ordinary ones (the sweep index is an ordinary kernel argument, so the large
// lattices pay nothing for this): before each replay the host rewrites that one argument of every kernel node
// (cudaGraphExecKernelNodeSetParams), which costs about a microsecond per node and runs ahead of the GPU.
constexpr int GRAPH_SWEEPS = 16;

struct GraphNode {
    cudaGraphNode_t node;
    cudaKernelNodeParams params;   // kernelParams is re-pointed at `args` before every update
    uint32_t k;                    // sweep offset of this launch inside the graph
    union { IsingArgs ising; VectorArgs vec; } args;
    GraphNode() {}
};

static void graph_drop(spin_system *s);
static bool graph_ok(const spin_system *s, int64_t n_sweeps) {
    if (s->vector_generic || s->axis >= 0 || n_sweeps < 2 * GRAPH_SWEEPS) return false;
    // threads of a half-sweep launch; beyond a few full waves the kernel outlasts its launch
    const uint64_t per_thread = s->n == 1 ? 32 : 4;
    return s->N * s->R / 2 / per_thread <= (uint64_t)s->sm_count * 2048 * 2;
}

static void graph_drop(spin_system *s) {
    if (s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }
    if (s->graph) { cudaGraphDestroy(s->graph); s->graph = nullptr; }
    delete[] s->gnodes; s->gnodes = nullptr; s->n_gnodes = 0; s->graph = nullptr;
}

static spin_status graph_prepare(spin_system *s, double beta) {
    const bool same = s->gexec && s->g_beta == beta && s->g_block == s->block && s->g_rows == s->strip_rows &&
                      s->g_rows_set == s->strip_rows_set && s->g_num == s->grid_num && s->g_den == s->grid_den;
    if (same) return SPIN_OK;
    graph_drop(s);
    if (!s->cap_stream) CUDA_TRY(cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking));
    const uint64_t launches0 = s->launches;
    CUDA_TRY(cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
    spin_status rc = SPIN_OK;
    for (int k = 0; k < GRAPH_SWEEPS && rc == SPIN_OK; ++k) rc = enqueue_sweep(s, beta, s->cap_stream, true, (uint32_t)k);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(s->cap_stream, &graph);
    s->launches = launches0;   // capturing launched nothing
    if (rc != SPIN_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(SPIN_ERR_CUDA, "graph capture: %s", cudaGetErrorString(e));
    // every kernel node with a copy of its argument block; the captured sweep offset is read back from that block
    size_t n_nodes = 0;
    e = cudaGraphGetNodes(graph, nullptr, &n_nodes);
    cudaGraphNode_t *nodes = (e == cudaSuccess && n_nodes) ? new (std::nothrow) cudaGraphNode_t[n_nodes] : nullptr;
    s->gnodes = nodes ? new (std::nothrow) GraphNode[n_nodes] : nullptr;
    if (e == cudaSuccess && (!nodes || !s->gnodes)) e = cudaErrorMemoryAllocation;
    if (e == cudaSuccess) e = cudaGraphGetNodes(graph, nodes, &n_nodes);
    for (size_t i = 0; e == cudaSuccess && i < n_nodes; ++i) {
        cudaGraphNodeType type;
        e = cudaGraphNodeGetType(nodes[i], &type);
        if (e != cudaSuccess || type != cudaGraphNodeTypeKernel) continue;
        GraphNode &gn = s->gnodes[s->n_gnodes];
        gn.node = nodes[i];
        e = cudaGraphKernelNodeGetParams(nodes[i], &gn.params);
        if (e != cudaSuccess) break;
        if (s->n == 1) { std::memcpy(&gn.args.ising, gn.params.kernelParams[0], sizeof(IsingArgs)); gn.k = gn.args.ising.t; }
        else { std::memcpy(&gn.args.vec, gn.params.kernelParams[0], sizeof(VectorArgs)); gn.k = gn.args.vec.t; }
        s->n_gnodes += 1;
    }
    delete[] nodes;
    if (e == cudaSuccess && s->n_gnodes != 2 * GRAPH_SWEEPS) e = cudaErrorUnknown;
    if (e == cudaSuccess) e = cudaGraphInstantiate(&s->gexec, graph, 0);
    s->graph = graph;   // kept: node handles stay valid as long as it lives
    if (e != cudaSuccess) { s->gexec = nullptr; graph_drop(s); return fail(SPIN_ERR_CUDA, "graph build: %s", cudaGetErrorString(e)); }
    s->g_beta = beta; s->g_block = s->block; s->g_rows = s->strip_rows; s->g_rows_set = s->strip_rows_set;
    s->g_num = s->grid_num; s->g_den = s->grid_den;
    return SPIN_OK;
}

// as many whole graphs as fit into n_sweeps; returns the sweeps done
static spin_status graph_sweeps(spin_system *s, double beta, int64_t n_sweeps, cudaStream_t st, int64_t *done) {
    *done = 0;
    spin_status rc = graph_prepare(s, beta);
    if (rc != SPIN_OK) return rc;
    while (n_sweeps - *done >= GRAPH_SWEEPS) {
        for (size_t i = 0; i < s->n_gnodes; ++i) {
            GraphNode &gn = s->gnodes[i];
            void *argp[1];
            if (s->n == 1) { gn.args.ising.t = (uint32_t)s->t + gn.k; argp[0] = &gn.args.ising; }
            else { gn.args.vec.t = (uint32_t)s->t + gn.k; argp[0] = &gn.args.vec; }
            gn.params.kernelParams = argp;
            gn.params.extra = nullptr;
            CUDA_TRY(cudaGraphExecKernelNodeSetParams(s->gexec, gn.node, &gn.params));
        }
        CUDA_TRY(cudaGraphLaunch(s->gexec, st));
        s->t += GRAPH_SWEEPS;
        s->launches += 2 * GRAPH_SWEEPS;
        *done += GRAPH_SWEEPS;
    }
    return SPIN_OK;
}

// E, M of every replica into device doubles dE[R], dM[R][n]
static spin_status enqueue_measure(spin_system *s, double *dE, double *dM, cudaStream_t st) {
    const dim3 grid(s->mblocks, s->R);
    if (s->n == 1) {
        IsingArgs a = ising_args(s);
        long long *acc = (long long *)(s->ws + s->lay.off_acc);
        const bool bonds = s->cfg.coupling_kind == SPIN_J_BOND_PM1;
        if (s->path == PATH_ISING_MSC) {
            const uint32_t spt = 64;   // sites per thread (bit-sliced counters hold 4095)
            const dim3 gm((unsigned)(((s->g.Nh + spt - 1) / spt + 127) / 128), s->R / 32);
            if (s->d == 2) ising_msc_measure<2><<<gm, 128, 0, st>>>(a, spt); else ising_msc_measure<3><<<gm, 128, 0, st>>>(a, spt);
        } else if (s->path == PATH_ISING_BITPACK) {
            if (s->d == 2) { if (bonds) ising_bitpack_measure<2, true><<<grid, 256, 0, st>>>(a); else ising_bitpack_measure<2, false><<<grid, 256, 0, st>>>(a); }
            else { if (bonds) ising_bitpack_measure<3, true><<<grid, 256, 0, st>>>(a); else ising_bitpack_measure<3, false><<<grid, 256, 0, st>>>(a); }
        } else if (s->path == PATH_ISING_INT8) {
            if (s->d == 2) ising_int8_measure<2><<<grid, 256, 0, st>>>(a);
            else ising_int8_measure<3><<<grid, 256, 0, st>>>(a);
        } else {
            ising_generic_measure<<<grid, 256, 0, st>>>(a);
        }
        CUDA_TRY(cudaGetLastError());
        ising_measure_finalize<<<(s->R + 3) / 4, 128, 0, st>>>(acc, s->R, a.acc_slots, dE, dM);
    } else {
        VectorArgs a = vector_args(s, 0.0);
        double *part = (double *)(s->ws + s->lay.off_acc);
        if (s->n == 2) vector_measure<2><<<grid, 256, 0, st>>>(a, part);
        else vector_measure<3><<<grid, 256, 0, st>>>(a, part);
        CUDA_TRY(cudaGetLastError());
        vector_measure_finalize<<<s->R, 256, 0, st>>>(part, s->mblocks, s->n, dE, dM);
    }
    s->launches += 2;
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

// Small uniform-coupling Ising systems (at most RESIDENT_MAX_WORDS 32-site words per colour over all replicas):
// all n_sweeps sweeps, and the per-sweep E and M if asked for, in ONE launch of the shared-memory-resident kernel.
static bool resident_ok(const spin_system *s, bool record) {
    if (s->vector_generic || s->n != 1 || s->axis >= 0) return false;
    if (!(s->path == PATH_ISING_INT8 || s->path == PATH_ISING_BITPACK)) return false;
    if (s->cfg.coupling_kind != SPIN_J_UNIFORM) return false;
    if ((uint64_t)s->g.NW * s->R > (uint64_t)RESIDENT_MAX_WORDS) return false;
    return !record || s->R <= 32;
}

static spin_status enqueue_resident(spin_system *s, int64_t n_sweeps, double *d_E, double *d_M, cudaStream_t st) {
    const int words = (int)(s->g.NW * s->R), B = (words + 31) / 32 * 32;
    // up to AHEAD_MAX_WORDS words (and R <= 32 replica slots): the kernel whose spare warps build the random masks ahead of the state;
    // up to 128 words with 512 threads (88 registers, nothing spilled in the consumers' chain: 0.42 against 0.47 us per recorded sweep
    // at 64 x 64; 256 threads leave too few producers: 0.50 us), beyond that with 1024 threads (64 registers)
    const bool ahead = s->variant != 1 && words <= AHEAD_MAX_WORDS && s->R <= 32 &&
                       2 * (s->cfg.update_rule == SPIN_UPDATE_HEATBATH ? 2 * s->d + 1 : s->d) * words * 2 <= AHEAD_SMEM_WORDS;
    while (n_sweeps > 0) {
        const uint32_t chunk = (uint32_t)(n_sweeps > (1 << 20) ? (1 << 20) : n_sweeps);
        const IsingArgs a = ising_args(s);
        const bool i8 = s->path == PATH_ISING_INT8;
        const bool hb = s->cfg.update_rule == SPIN_UPDATE_HEATBATH;
#define RS(D_, I8_, HB_) do { if (ahead && words <= 128) ising_resident_ahead_sweeps<D_, I8_, HB_, 512><<<1, 512, 0, st>>>(a, chunk, d_E, d_M); \
                              else if (ahead) ising_resident_ahead_sweeps<D_, I8_, HB_, 1024><<<1, 1024, 0, st>>>(a, chunk, d_E, d_M); \
                              else ising_resident_sweeps<D_, I8_, HB_><<<1, B, 0, st>>>(a, chunk, d_E, d_M); } while (0)
#define RS2(D_, I8_) do { if (hb) RS(D_, I8_, true); else RS(D_, I8_, false); } while (0)
        if (s->d == 2) { if (i8) RS2(2, true); else RS2(2, false); }
        else { if (i8) RS2(3, true); else RS2(3, false); }
#undef RS2
#undef RS
        CUDA_TRY(cudaGetLastError());
        s->launches += 1;
        s->t += chunk;
        n_sweeps -= chunk;
        if (d_E) { d_E += (size_t)chunk * s->R; d_M += (size_t)chunk * s->R; }
    }
    return SPIN_OK;
}

static spin_status check_sweep_args(spin_system *s, double beta, int64_t n_sweeps) {
    if (!s) return fail(SPIN_ERR_INVALID_ARG, "handle is NULL");
    if (!(beta >= 0.0) || !std::isfinite(beta)) return fail(SPIN_ERR_INVALID_ARG, "beta must be finite and >= 0");
    if (n_sweeps < 0) return fail(SPIN_ERR_INVALID_ARG, "n_sweeps must be >= 0");
    if (s->t + (uint64_t)n_sweeps > 0x100000000ull) return fail(SPIN_ERR_STATE, "sweep counter would pass 2^32");
    if (s->n == 1 && !(beta == s->table_beta)) {
        build_table(beta, &s->tab);
        if (s->cfg.update_rule == SPIN_UPDATE_HEATBATH) build_hb_table(beta, 2 * s->d, &s->hb);
        s->table_beta = beta;
    }
    return SPIN_OK;
}

// ------------------------------------------------------------------- no-allocation measurement ------
// spin_measure_noalloc (include/spin.h): for callers that may not allocate -- code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  The scratch of the measurement kernels (per-CTA partial sums for n >= 2, the int64
// accumulator slots for n = 1; normally carved from the caller's workspace) lives in this file-scope device array instead:
// SPIN_NOALLOC_SCRATCH_BYTES = 1 MiB, held by every GPU that loads the library until the process exits.
// In HOST code the name g_noalloc_scratch is a host-side stand-in, not a device address (a kernel given it would fault, or, where
// the GPU can reach host memory, silently use the wrong memory): the device address comes from cudaGetSymbolAddress, once per
// device, with that device current, and it is that pointer the kernels receive.
static __device__ __align__(256) unsigned char g_noalloc_scratch[SPIN_NOALLOC_SCRATCH_BYTES];

constexpr int NOALLOC_MAX_DEVICES = 64;
static void *g_noalloc_ptr[NOALLOC_MAX_DEVICES];   // device address of g_noalloc_scratch per device ordinal, NULL until looked up

// device address of the scratch array on the CURRENT device (looked up on first use; no allocation)
static spin_status noalloc_scratch(void **out) {
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(SPIN_ERR_UNSUPPORTED, "device ordinal %d beyond %d", dev, NOALLOC_MAX_DEVICES);
    if (!g_noalloc_ptr[dev]) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess || !ptr) return fail(SPIN_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch): %s", cudaGetErrorString(e));
        g_noalloc_ptr[dev] = ptr;
    }
    *out = g_noalloc_ptr[dev];
    return SPIN_OK;
}

// ------------------------------------------------------------------------------ C ABI --------
extern "C" {

const char *spin_last_error(void) { return g_err; }
const char *spin_version(void) { return "libspin 0.2 sm_100a"; }

spin_status spin_workspace_bytes(const spin_config *cfg, size_t *bytes) {
    if (!bytes) return fail(SPIN_ERR_INVALID_ARG, "bytes is NULL");
    Derived dv;
    spin_status rc = derive(cfg, &dv);
    if (rc != SPIN_OK) return rc;
    Layout l;
    uint32_t mb;
    make_layout(cfg, dv, &l, &mb);
    *bytes = l.total;
    return SPIN_OK;
}

spin_status spin_create(const spin_config *cfg, void *d_workspace, size_t bytes, void *stream, spin_system **out) {
    if (!out) return fail(SPIN_ERR_INVALID_ARG, "out is NULL");
    Derived dv;
    spin_status rc = derive(cfg, &dv);
    if (rc != SPIN_OK) return rc;
    if (!d_workspace) return fail(SPIN_ERR_INVALID_ARG, "d_workspace is NULL");
    if (((uintptr_t)d_workspace & 255) != 0) return fail(SPIN_ERR_INVALID_ARG, "d_workspace must be 256-byte aligned");
    if (cfg->coupling_kind == SPIN_J_BOND_PM1 && cfg->bonds) {
        const size_t nb = (size_t)cfg->n_replicas * dv.d * dv.N;
        for (size_t k = 0; k < nb; ++k)
            if (cfg->bonds[k] != 1 && cfg->bonds[k] != -1) return fail(SPIN_ERR_INVALID_ARG, "bonds must be +-1");
    }
    spin_system *s = new (std::nothrow) spin_system();
    if (!s) return fail(SPIN_ERR_INVALID_ARG, "out of host memory");
    s->cfg = *cfg;
    s->cfg.bonds = nullptr;  // host array is read here only
    s->d = dv.d; s->n = cfg->n; s->R = (uint32_t)cfg->n_replicas; s->N = dv.Nown; s->path = dv.path;
    s->axis = dv.axis; s->own_planes = dv.axis >= 0 ? cfg->dims[dv.axis] : 0; s->next_colour = 0;
    make_layout(cfg, dv, &s->lay, &s->mblocks);
    if (bytes < s->lay.total) {
        const size_t need = s->lay.total;
        delete s;
        return fail(SPIN_ERR_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, %zu needed", bytes, need);
    }
    s->ws = (char *)d_workspace;
    s->tma_ok = 0; s->use_tma = -1; s->tma_ty = 0;
    s->t = 0; s->launches = 0; s->staging = nullptr; s->staging_bytes = 0; s->set_pending = 0; s->h_res = nullptr; s->gexec = nullptr; s->cap_stream = nullptr; s->gnodes = nullptr; s->n_gnodes = 0;
    // 128 threads per CTA for the Ising fast paths (measured: +-J R = 16 39.1 vs 40.4 us with 256)
    s->block = (dv.path == PATH_ISING_INT8 || dv.path == PATH_ISING_BITPACK || dv.path == PATH_ISING_MSC) ? 128 : 256; s->grid_num = 1; s->grid_den = 1; s->strip_rows = 4; s->strip_rows_set = 0; s->vector_generic = 0; s->l2_prefetch = -1; s->l2_keep = -1; s->defer_cap = DEFER_CAP; s->l2_bytes = 0; s->variant = 0; s->tblock = -1; s->tblock_rows = 0; s->tblock_ok = tblock_offered(cfg, dv) ? 1 : 0;
    s->table_beta = std::nan("");
    Geometry &g = s->g;
    g.Lx = dv.pad[0]; g.Ly = dv.pad[1]; g.Lz = dv.pad[2]; g.d = dv.d;
    g.RL = (uint32_t)(g.Lx / 2); g.rows = (uint32_t)(g.Ly * g.Lz); g.Nh = (uint32_t)(dv.N / 2);
    g.WX = g.RL / 32; g.NW = g.Nh / 32;
    g.divRL = make_fastdiv(g.RL); g.divWX = make_fastdiv(g.WX ? g.WX : 1); g.divLy = make_fastdiv((uint32_t)g.Ly);
    g.divQX = make_fastdiv(g.RL / 4 ? g.RL / 4 : 1);
    g.divQW = make_fastdiv(g.WX / 4 ? g.WX / 4 : 1);
    g.j_off = 0; g.unit_off = 0; g.i_off = 0; g.own_j0 = 0; g.own_j1 = g.Nh; g.own_i0 = 0; g.own_in = (uint32_t)dv.N;
    if (dv.axis >= 0) {
        const int64_t plane_sites = dv.axis == 2 ? (int64_t)g.Lx * g.Ly : (int64_t)g.Lx, plane_h = plane_sites / 2;
        const int64_t shift = (int64_t)cfg->slab_offset - 2;   // local plane p is global plane p + shift
        g.j_off = (uint32_t)(shift * plane_h);
        g.unit_off = (uint32_t)(shift * plane_h / 32);        // exact for the fast layouts (plane_h % 32 == 0)
        g.i_off = (uint32_t)(shift * plane_sites);
        g.own_j0 = (uint32_t)(2 * plane_h); g.own_j1 = (uint32_t)((2 + cfg->dims[dv.axis]) * plane_h);
        g.own_i0 = (uint32_t)(2 * plane_sites); g.own_in = (uint32_t)dv.Nown;
    }
    {
        // what a half-sweep updates: everything, or the owned planes of a slab (the ghost planes are only read)
        const uint32_t plane_h = g.d == 3 ? g.RL * (uint32_t)g.Ly : g.RL;
        g.sw_p0 = dv.axis >= 0 ? 2u : 0u;
        g.sw_pn = dv.axis >= 0 ? (uint32_t)cfg->dims[dv.axis] : (uint32_t)(g.d == 3 ? g.Lz : g.Ly);
        g.sw_j0 = g.sw_p0 * plane_h; g.sw_jn = g.sw_pn * plane_h;
    }
    for (int r = 0; r < 10; ++r) {
        s->keys.k0[r] = (uint32_t)(cfg->seed & 0xFFFFFFFFull) + (uint32_t)r * 0x9E3779B9u;
        s->keys.k1[r] = (uint32_t)(cfg->seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&s->sm_count, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&s->l2_bytes, cudaDevAttrL2CacheSize, dev)) != cudaSuccess) {
        delete s;
        return fail(SPIN_ERR_CUDA, "no usable CUDA device: %s", cudaGetErrorString(e));
    }
    tma_prepare(s);
#define CREATE_TRY(expr)                                                                              \
    do {                                                                                              \
        cudaError_t e2_ = (expr);                                                                     \
        if (e2_ != cudaSuccess) {                                                                     \
            if (staging) cudaFree(staging);                                                           \
            delete s;                                                                                 \
            return fail(SPIN_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e2_));                     \
        }                                                                                             \
    } while (0)
    void *staging = nullptr;
    const SetupArgs sa = setup_args(s);
    const int B = 256;
    const int G = grid_for(s, 2ull * s->R * g.Nh);
    CREATE_TRY(cudaMemsetAsync(s->ws + s->lay.off_acc, 0, s->lay.bytes_acc, st));
    if (cfg->coupling_kind == SPIN_J_BOND_PM1) {
        const size_t nb = (size_t)s->R * s->d * s->N;
        if (s->path == PATH_ISING_MSC) {
            if (cfg->bonds) {
                CREATE_TRY(cudaMalloc(&staging, nb));
                CREATE_TRY(cudaMemcpyAsync(staging, cfg->bonds, nb, cudaMemcpyHostToDevice, st));
            }
            msc_bonds_pack<<<G, B, 0, st>>>(sa, (const int8_t *)staging, (uint32_t *)(s->ws + s->lay.off_bonds));
        } else if (s->path == PATH_ISING_BITPACK) {
            if (cfg->bonds) {
                CREATE_TRY(cudaMalloc(&staging, nb));
                CREATE_TRY(cudaMemcpyAsync(staging, cfg->bonds, nb, cudaMemcpyHostToDevice, st));
            }
            bonds_pack<<<G, B, 0, st>>>(sa, (const int8_t *)staging, (uint32_t *)(s->ws + s->lay.off_bonds));
        } else if (cfg->bonds) {
            CREATE_TRY(cudaMemcpyAsync(s->ws + s->lay.off_bonds, cfg->bonds, nb, cudaMemcpyHostToDevice, st));
        } else {
            bonds_draw_canonical<<<grid_for(s, (uint64_t)s->R * s->N), B, 0, st>>>(sa, (int8_t *)(s->ws + s->lay.off_bonds));
        }
        CREATE_TRY(cudaGetLastError());
    }
    const int mode = cfg->init == SPIN_INIT_HOT ? 1 : 0;
    if (s->path == PATH_ISING_MSC) msc_fill<<<G, B, 0, st>>>(sa, mode, nullptr, (uint32_t *)(s->ws + s->lay.off_s[0]), (uint32_t *)(s->ws + s->lay.off_s[1]));
    else if (s->n == 1) ising_fill<<<G, B, 0, st>>>(sa, mode, nullptr, s->ws + s->lay.off_s[0], s->ws + s->lay.off_s[1]);
    else if (s->n == 2) vector_fill<2><<<G, B, 0, st>>>(sa, mode, nullptr, (float *)(s->ws + s->lay.off_s[0]), (float *)(s->ws + s->lay.off_s[1]));
    else vector_fill<3><<<G, B, 0, st>>>(sa, mode, nullptr, (float *)(s->ws + s->lay.off_s[0]), (float *)(s->ws + s->lay.off_s[1]));
    CREATE_TRY(cudaGetLastError());
    CREATE_TRY(cudaStreamSynchronize(st));
    if (staging) cudaFree(staging);
#undef CREATE_TRY
    *out = s;
    return SPIN_OK;
}

spin_status spin_destroy(spin_system *s) {
    if (s && s->staging) cudaFree(s->staging);
    if (s && s->h_res) cudaFreeHost(s->h_res);
    if (s) graph_drop(s);
    if (s && s->cap_stream) cudaStreamDestroy(s->cap_stream);
    delete s;
    return SPIN_OK;
}

// Many +-J realisations of a small lattice with a shared update stream (bit-packed, both update rules): groups of realisations stay in
// shared memory for all n_sweeps sweeps of the call (ising_resident_pmj_kernel.cuh).  G = realisations per CTA: two CTAs per SM, within
// RPMJ_SMEM_MAX bytes of shared memory each.
constexpr size_t RPMJ_SMEM_MAX = 100 * 1024;
static uint32_t resident_pmj_group(const spin_system *s) {
    const uint32_t NW = (uint32_t)s->g.NW;
    if (NW == 0 || NW > (uint32_t)RPMJ_THREADS || RPMJ_THREADS % NW != 0) return 0;
    // an even share of the replicas for each of the 2 sm_count CTAs that are resident at once (measured at 4096 x 64^2: groups of 14,
    // 293 CTAs, against groups of 16 = a multiple of RG, 256 CTAs of which 108 SMs hold two and 40 one)
    uint64_t G = (s->R + 2 * (uint64_t)s->sm_count - 1) / (2 * (uint64_t)s->sm_count);
    while (G > 1 && 4 * rpmj_smem_words((uint32_t)G, NW, s->d, s->cfg.update_rule == SPIN_UPDATE_HEATBATH) > RPMJ_SMEM_MAX) G -= 1;
    if (4 * rpmj_smem_words((uint32_t)G, NW, s->d, s->cfg.update_rule == SPIN_UPDATE_HEATBATH) > RPMJ_SMEM_MAX) return 0;
    return (uint32_t)G;
}
static bool resident_pmj_ok(const spin_system *s) {
    if (s->variant == 1) return false;   // A/B: one launch per half-sweep (ising_bitpack_halfsweep / the quad kernels)
    if (s->vector_generic || s->n != 1 || s->axis >= 0 || s->path != PATH_ISING_BITPACK) return false;
    if (s->cfg.coupling_kind != SPIN_J_BOND_PM1) return false;
    if (!(s->R > 1 && !s->cfg.replica_streams)) return false;
    return resident_pmj_group(s) != 0;
}
static spin_status enqueue_resident_pmj(spin_system *s, int64_t n_sweeps, cudaStream_t st) {
    const uint32_t G = resident_pmj_group(s);
    const bool hb = s->cfg.update_rule == SPIN_UPDATE_HEATBATH;
    const size_t smem = 4 * rpmj_smem_words(G, (uint32_t)s->g.NW, s->d, hb);
    const unsigned grid = (unsigned)((s->R + G - 1) / G);
#define RPMJ(D_, HB_) do { CUDA_TRY(cudaFuncSetAttribute(ising_resident_pmj_sweeps<D_, HB_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
                           ising_resident_pmj_sweeps<D_, HB_><<<grid, RPMJ_THREADS, smem, st>>>(a, chunk, G); } while (0)
    while (n_sweeps > 0) {
        const uint32_t chunk = (uint32_t)(n_sweeps > (1 << 20) ? (1 << 20) : n_sweeps);
        const IsingArgs a = ising_args(s);
        if (s->d == 2) { if (hb) RPMJ(2, true); else RPMJ(2, false); }
        else { if (hb) RPMJ(3, true); else RPMJ(3, false); }
        CUDA_TRY(cudaGetLastError());
        s->launches += 1;
        s->t += chunk;
        n_sweeps -= chunk;
    }
#undef RPMJ
    return SPIN_OK;
}

spin_status spin_sweep(spin_system *s, double beta, int64_t n_sweeps, void *stream) {
    spin_status rc = check_sweep_args(s, beta, n_sweeps);
    if (rc != SPIN_OK) return rc;
    if (s->axis >= 0) return fail(SPIN_ERR_STATE, "slab handle: drive it with spin_halfsweep and the halo calls");
    if (s->next_colour != 0) return fail(SPIN_ERR_STATE, "a spin_halfsweep of colour 1 is pending");
    if (tblock_use(s, n_sweeps)) {
        // two sweeps per pass over the lattice; an odd last sweep goes through the plain kernels below
        rc = tblock_sweeps(s, n_sweeps / 2, (cudaStream_t)stream);
        if (rc != SPIN_OK) return rc;
        n_sweeps &= 1;
    } else if (resident_ok(s, false)) return enqueue_resident(s, n_sweeps, nullptr, nullptr, (cudaStream_t)stream);
    else if (resident_pmj_ok(s)) return enqueue_resident_pmj(s, n_sweeps, (cudaStream_t)stream);
    if (graph_ok(s, n_sweeps)) {
        int64_t done = 0;
        rc = graph_sweeps(s, beta, n_sweeps, (cudaStream_t)stream, &done);
        if (rc != SPIN_OK) return rc;
        n_sweeps -= done;
    }
    for (int64_t k = 0; k < n_sweeps; ++k) {
        rc = enqueue_sweep(s, beta, (cudaStream_t)stream);
        if (rc != SPIN_OK) return rc;
    }
    return SPIN_OK;
}

// Temperature axis: replica r at betas[r].  One launch per replica and half-sweep with the
// ordinary kernels: the launch sees a one-replica system whose arrays start at replica r and whose Philox replica word is r
// (rho_off), so replica r follows exactly the chain it has in a handle swept at betas[r] throughout.
spin_status spin_sweep_betas(spin_system *s, const double *betas, int64_t n_sweeps, void *stream) {
    if (!s || !betas) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    for (uint32_t r = 0; r < s->R; ++r)
        if (!(betas[r] >= 0.0) || !std::isfinite(betas[r])) return fail(SPIN_ERR_INVALID_ARG, "beta must be finite and >= 0");
    spin_status rc = check_sweep_args(s, betas[0], n_sweeps);
    if (rc != SPIN_OK) return rc;
    if (s->axis >= 0) return fail(SPIN_ERR_STATE, "slab handle: drive it with spin_halfsweep and the halo calls");
    if (s->next_colour != 0) return fail(SPIN_ERR_STATE, "a spin_halfsweep of colour 1 is pending");
    if (s->R > 1 && !s->cfg.replica_streams) return fail(SPIN_ERR_UNSUPPORTED, "a temperature axis needs replica_streams = 1 (a shared update stream ties the acceptance masks of the replicas together)");
    if (s->path == PATH_ISING_MSC || (s->path == PATH_ISING_BITPACK && s->cfg.coupling_kind == SPIN_J_BOND_PM1))
        return fail(SPIN_ERR_UNSUPPORTED, "temperature axis with bit-packed per-bond couplings (use INT8 storage)");
    cudaStream_t st = (cudaStream_t)stream;
    const uint32_t R = s->R;
    IsingTable *tabs = nullptr;
    HeatBathTable *hbs = nullptr;
    if (s->n == 1) {
        tabs = new (std::nothrow) IsingTable[R];
        hbs = s->cfg.update_rule == SPIN_UPDATE_HEATBATH ? new (std::nothrow) HeatBathTable[R] : nullptr;
        if (!tabs || (s->cfg.update_rule == SPIN_UPDATE_HEATBATH && !hbs)) { delete[] tabs; delete[] hbs; return fail(SPIN_ERR_INVALID_ARG, "out of host memory"); }
        for (uint32_t r = 0; r < R; ++r) {
            build_table(betas[r], &tabs[r]);
            if (hbs) build_hb_table(betas[r], 2 * s->d, &hbs[r]);
        }
    }
    // bytes of one replica in a colour array / in the canonical per-bond array of the generic kernel
    const size_t rep_bytes = s->lay.bytes_s / R;
    const size_t bond_bytes = s->lay.bytes_bonds / R;
    rc = SPIN_OK;
    for (int64_t k = 0; k < n_sweeps && rc == SPIN_OK; ++k) {
        for (uint32_t colour = 0; colour < 2 && rc == SPIN_OK; ++colour) {
            for (uint32_t r = 0; r < R && rc == SPIN_OK; ++r) {
                s->R = 1;   // the launch helpers size their grids from the handle
                if (s->n == 1) {
                    IsingArgs a = ising_args(s);
                    a.tab = tabs[r];
                    if (hbs) a.hb = hbs[r];
                    a.colour = colour; a.rho_off = r;
                    a.s[0] = (char *)a.s[0] + r * rep_bytes; a.s[1] = (char *)a.s[1] + r * rep_bytes;
                    if (a.bonds) a.bonds = (const char *)a.bonds + r * bond_bytes;
                    rc = launch_halfsweep_ising(s, a, st);
                } else {
                    VectorArgs a = vector_args(s, betas[r]);
                    a.colour = colour; a.rho_off = r;
                    a.s[0] = (float *)((char *)a.s[0] + r * rep_bytes); a.s[1] = (float *)((char *)a.s[1] + r * rep_bytes);
                    rc = launch_halfsweep_vector(s, a, st, false);
                }
                s->R = R;
            }
        }
        if (rc == SPIN_OK) s->t += 1;
    }
    s->table_beta = std::nan("");   // the cached table belongs to no single beta now
    delete[] tabs;
    delete[] hbs;
    return rc;
}

spin_status spin_sweep_record(spin_system *s, double beta, int64_t n_sweeps, double *d_E, double *d_M, void *stream) {
    spin_status rc = check_sweep_args(s, beta, n_sweeps);
    if (rc != SPIN_OK) return rc;
    if (!d_E || !d_M) return fail(SPIN_ERR_INVALID_ARG, "d_E / d_M is NULL");
    if (s->axis >= 0) return fail(SPIN_ERR_STATE, "slab handle: drive it with spin_halfsweep and the halo calls");
    if (s->next_colour != 0) return fail(SPIN_ERR_STATE, "a spin_halfsweep of colour 1 is pending");
    if (resident_ok(s, true)) return enqueue_resident(s, n_sweeps, d_E, d_M, (cudaStream_t)stream);
    cudaStream_t st = (cudaStream_t)stream;
    for (int64_t k = 0; k < n_sweeps; ++k) {
        double *oE = d_E + (size_t)k * s->R, *oM = d_M + (size_t)k * s->R * s->n;
        if (s->n == 1 && !s->vector_generic) {
            // E and M for free inside the colour-1 half-sweep where the kernel can (strip kernels), else a measurement pass
            IsingArgs a = ising_args(s);
            bool fused = false;
            a.colour = 0;
            rc = launch_halfsweep_ising(s, a, st);
            if (rc != SPIN_OK) return rc;
            a.colour = 1;
            rc = launch_halfsweep_ising(s, a, st, &fused);
            if (rc != SPIN_OK) return rc;
            s->t += 1;
            if (fused) {
                ising_measure_finalize<<<(s->R + 3) / 4, 128, 0, st>>>(a.acc, s->R, a.acc_slots, oE, oM);
                s->launches += 1;
                CUDA_TRY(cudaGetLastError());
                continue;
            }
        } else if (s->n > 1) {
            // n >= 2: the TMA-staged colour-1 half-sweep leaves per-CTA partial sums of E and M (row a7)
            VectorArgs a = vector_args(s, beta);
            uint32_t parts = 0;
            bool two_level = false;
            a.colour = 0;
            rc = launch_halfsweep_vector(s, a, st);
            if (rc != SPIN_OK) return rc;
            a.colour = 1;
            rc = launch_halfsweep_vector(s, a, st, true, &parts, &two_level);
            if (rc != SPIN_OK) return rc;
            s->t += 1;
            if (parts) {
                const double *part = (const double *)(s->ws + s->lay.off_acc);
                if (two_level) {
                    const uint32_t F = parts / 256 + 1 < FINALIZE_BLOCKS ? parts / 256 + 1 : FINALIZE_BLOCKS;
                    vector_partials_finalize<<<dim3(F, s->R), 256, 0, st>>>(part, parts, s->n, (double *)(s->ws + s->lay.off_mid),
                                                                             (unsigned *)(s->ws + s->lay.off_cnt), oE, oM);
                } else
                vector_measure_finalize<<<s->R, 256, 0, st>>>(part, parts, s->n, oE, oM);
                s->launches += 1;
                CUDA_TRY(cudaGetLastError());
                continue;
            }
        } else {
            rc = enqueue_sweep(s, beta, st);
            if (rc != SPIN_OK) return rc;
        }
        rc = enqueue_measure(s, oE, oM, st);
        if (rc != SPIN_OK) return rc;
    }
    return SPIN_OK;
}

// planes [plane0, plane0 + n_planes) of the swept range (whole lattice: along its slowest axis; slab: its owned planes)
static void restrict_range(Geometry &g, int32_t plane0, int32_t n_planes) {
    const uint32_t plane_h = g.d == 3 ? g.RL * (uint32_t)g.Ly : g.RL;
    g.sw_p0 += (uint32_t)plane0;
    g.sw_pn = (uint32_t)n_planes;
    g.sw_j0 = g.sw_p0 * plane_h;
    g.sw_jn = g.sw_pn * plane_h;
}

static spin_status halfsweep_impl(spin_system *s, double beta, int32_t colour, int32_t plane0, int32_t n_planes, bool ranged, bool last,
                                  cudaStream_t st) {
    // either colour needs a sweep index below 2^32 (colour 0 at t = 2^32 would silently reuse the numbers of sweep 0)
    spin_status rc = check_sweep_args(s, beta, 1);
    if (rc != SPIN_OK) return rc;
    if (colour != 0 && colour != 1) return fail(SPIN_ERR_INVALID_ARG, "colour must be 0 or 1");
    if ((uint32_t)colour != s->next_colour) return fail(SPIN_ERR_STATE, "half-sweeps alternate: colour %u is next", s->next_colour);
    if (ranged && (plane0 < 0 || n_planes < 0 || (uint32_t)plane0 + (uint32_t)n_planes > s->g.sw_pn))
        return fail(SPIN_ERR_INVALID_ARG, "plane range [%d, %d) outside the %u planes this handle updates", plane0, plane0 + n_planes, s->g.sw_pn);
    if (!ranged || n_planes > 0) {
        if (s->n == 1) {
            IsingArgs a = ising_args(s);
            a.colour = (uint32_t)colour;
            if (ranged) restrict_range(a.g, plane0, n_planes);
            rc = launch_halfsweep_ising(s, a, st);
        } else {
            VectorArgs a = vector_args(s, beta);
            a.colour = (uint32_t)colour;
            if (ranged) restrict_range(a.g, plane0, n_planes);
            rc = launch_halfsweep_vector(s, a, st, !ranged);
        }
        if (rc != SPIN_OK) return rc;
    }
    if (last) {
        s->next_colour = 1u - (uint32_t)colour;
        if (colour == 1) s->t += 1;
    }
    return SPIN_OK;
}

spin_status spin_halfsweep(spin_system *s, double beta, int32_t colour, void *stream) {
    return halfsweep_impl(s, beta, colour, 0, 0, false, true, (cudaStream_t)stream);
}

spin_status spin_halfsweep_range(spin_system *s, double beta, int32_t colour, int32_t plane0, int32_t n_planes, int32_t last, void *stream) {
    return halfsweep_impl(s, beta, colour, plane0, n_planes, true, last != 0, (cudaStream_t)stream);
}

// one face of one colour: per (replica, component) one contiguous plane of the colour array
struct Face {
    size_t plane_bytes, stride_bytes, rows;
};
static Face face_of(const spin_system *s) {
    const Geometry &g = s->g;
    const size_t plane_h = s->axis == 2 ? (size_t)g.RL * g.Ly : (size_t)g.RL;
    Face f;
    if (s->path == PATH_ISING_BITPACK) { f.plane_bytes = plane_h / 8; f.stride_bytes = (size_t)g.NW * 4; f.rows = s->R; }
    else if (s->path == PATH_VECTOR) { f.plane_bytes = plane_h * 4; f.stride_bytes = (size_t)g.Nh * 4; f.rows = (size_t)s->R * s->n; }
    else { f.plane_bytes = plane_h; f.stride_bytes = g.Nh; f.rows = s->R; }
    return f;
}

spin_status spin_halo_bytes(const spin_system *s, size_t *bytes) {
    if (!s || !bytes) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (s->axis < 0) return fail(SPIN_ERR_STATE, "not a slab handle");
    const Face f = face_of(s);
    *bytes = f.plane_bytes * f.rows;
    return SPIN_OK;
}

static spin_status halo_copy(spin_system *s, int32_t colour, int32_t side, void *d_buf, bool get, cudaStream_t st) {
    if (!s || !d_buf) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (s->axis < 0) return fail(SPIN_ERR_STATE, "not a slab handle");
    if ((colour != 0 && colour != 1) || (side != 0 && side != 1)) return fail(SPIN_ERR_INVALID_ARG, "colour and side must be 0 or 1");
    const Face f = face_of(s);
    // local planes: 0, 1 low ghosts (1 is read), 2 .. own + 1 owned, own + 2, own + 3 high ghosts (own + 2 is read)
    const size_t plane = get ? (side == 0 ? 2 : (size_t)s->own_planes + 1) : (side == 0 ? 1 : (size_t)s->own_planes + 2);
    char *arr = s->ws + s->lay.off_s[colour] + plane * f.plane_bytes;
    if (get) CUDA_TRY(cudaMemcpy2DAsync(d_buf, f.plane_bytes, arr, f.stride_bytes, f.plane_bytes, f.rows, cudaMemcpyDeviceToDevice, st));
    else CUDA_TRY(cudaMemcpy2DAsync(arr, f.stride_bytes, d_buf, f.plane_bytes, f.plane_bytes, f.rows, cudaMemcpyDeviceToDevice, st));
    return SPIN_OK;
}

spin_status spin_halo_get(spin_system *s, int32_t colour, int32_t side, void *d_buf, void *stream) {
    return halo_copy(s, colour, side, d_buf, true, (cudaStream_t)stream);
}

spin_status spin_halo_put(spin_system *s, int32_t colour, int32_t side, const void *d_buf, void *stream) {
    return halo_copy(s, colour, side, const_cast<void *>(d_buf), false, (cudaStream_t)stream);
}

// both faces of one colour with one kernel: pack = owned boundary planes -> d_buf [low][high], unpack = d_buf [from below][from above] -> ghosts
static spin_status halo_faces(spin_system *s, int32_t colour, void *d_buf, bool pack, cudaStream_t st) {
    if (!s || !d_buf) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (s->axis < 0) return fail(SPIN_ERR_STATE, "not a slab handle");
    if (colour != 0 && colour != 1) return fail(SPIN_ERR_INVALID_ARG, "colour must be 0 or 1");
    const Face f = face_of(s);
    // local planes: 0, 1 low ghosts (1 is read), 2 .. own + 1 owned, own + 2, own + 3 high ghosts (own + 2 is read)
    const uint32_t lo = pack ? 2u : 1u, hi = pack ? (uint32_t)s->own_planes + 1u : (uint32_t)s->own_planes + 2u;
    char *arr = s->ws + s->lay.off_s[colour];
    const size_t bytes = 2 * f.plane_bytes * f.rows;
    const bool wide = f.plane_bytes % 16 == 0 && f.stride_bytes % 16 == 0 && ((uintptr_t)d_buf & 15) == 0;
    const size_t elems = wide ? bytes / 16 : bytes;
    const int G = (int)((elems + 255) / 256 > 1184 ? 1184 : (elems + 255) / 256);
    if (wide) halo_faces_copy<uint4><<<G, 256, 0, st>>>((uint4 *)arr, (uint4 *)d_buf, f.plane_bytes / 16, f.stride_bytes / 16, (uint32_t)f.rows, lo, hi, pack);
    else halo_faces_copy<uint8_t><<<G, 256, 0, st>>>((uint8_t *)arr, (uint8_t *)d_buf, f.plane_bytes, f.stride_bytes, (uint32_t)f.rows, lo, hi, pack);
    CUDA_TRY(cudaGetLastError());
    s->launches += 1;
    return SPIN_OK;
}

spin_status spin_halo_wrap(spin_system *s, int32_t colour, void *stream) {
    if (!s) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (s->axis < 0) return fail(SPIN_ERR_STATE, "not a slab handle");
    if (colour != 0 && colour != 1) return fail(SPIN_ERR_INVALID_ARG, "colour must be 0 or 1");
    const Face f = face_of(s);
    char *arr = s->ws + s->lay.off_s[colour];
    const bool wide = f.plane_bytes % 16 == 0 && f.stride_bytes % 16 == 0;
    const size_t elems = 2 * f.plane_bytes * f.rows / (wide ? 16 : 1);
    const int G = (int)((elems + 255) / 256 > 1184 ? 1184 : (elems + 255) / 256);
    cudaStream_t st = (cudaStream_t)stream;
    if (wide) halo_faces_wrap<uint4><<<G, 256, 0, st>>>((uint4 *)arr, f.plane_bytes / 16, f.stride_bytes / 16, (uint32_t)f.rows, (uint32_t)s->own_planes);
    else halo_faces_wrap<uint8_t><<<G, 256, 0, st>>>((uint8_t *)arr, f.plane_bytes, f.stride_bytes, (uint32_t)f.rows, (uint32_t)s->own_planes);
    CUDA_TRY(cudaGetLastError());
    s->launches += 1;
    return SPIN_OK;
}

spin_status spin_colour_array(spin_system *s, int32_t colour, void **d_ptr, size_t *bytes) {
    if (!s || !d_ptr) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (colour != 0 && colour != 1) return fail(SPIN_ERR_INVALID_ARG, "colour must be 0 or 1");
    *d_ptr = s->ws + s->lay.off_s[colour];
    if (bytes) *bytes = s->lay.bytes_s;
    return SPIN_OK;
}

spin_status spin_halo_push(spin_system *s, int32_t colour, void *d_peer_below, void *d_peer_above, void *stream) {
    if (!s || !d_peer_below || !d_peer_above) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (s->axis < 0) return fail(SPIN_ERR_STATE, "not a slab handle");
    if (colour != 0 && colour != 1) return fail(SPIN_ERR_INVALID_ARG, "colour must be 0 or 1");
    const Face f = face_of(s);
    const char *arr = s->ws + s->lay.off_s[colour];
    const bool wide = f.plane_bytes % 16 == 0 && f.stride_bytes % 16 == 0 && (((uintptr_t)d_peer_below | (uintptr_t)d_peer_above) & 15) == 0;
    const size_t elems = 2 * f.plane_bytes * f.rows / (wide ? 16 : 1);
    const int G = (int)((elems + 255) / 256 > 1184 ? 1184 : (elems + 255) / 256);
    cudaStream_t st = (cudaStream_t)stream;
    if (wide) halo_faces_push<uint4><<<G, 256, 0, st>>>((const uint4 *)arr, (uint4 *)d_peer_below, (uint4 *)d_peer_above, f.plane_bytes / 16, f.stride_bytes / 16, (uint32_t)f.rows, (uint32_t)s->own_planes);
    else halo_faces_push<uint8_t><<<G, 256, 0, st>>>((const uint8_t *)arr, (uint8_t *)d_peer_below, (uint8_t *)d_peer_above, f.plane_bytes, f.stride_bytes, (uint32_t)f.rows, (uint32_t)s->own_planes);
    CUDA_TRY(cudaGetLastError());
    s->launches += 1;
    return SPIN_OK;
}

spin_status spin_halo_pack(spin_system *s, int32_t colour, void *d_buf, void *stream) {
    return halo_faces(s, colour, d_buf, true, (cudaStream_t)stream);
}

spin_status spin_halo_unpack(spin_system *s, int32_t colour, const void *d_buf, void *stream) {
    return halo_faces(s, colour, const_cast<void *>(d_buf), false, (cudaStream_t)stream);
}

spin_status spin_measure(spin_system *s, double *E, double *M, void *stream) {
    if (!s || !E || !M) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    double *res = (double *)(s->ws + s->lay.off_res);
    spin_status rc = enqueue_measure(s, res, res + s->R, st);
    if (rc != SPIN_OK) return rc;
    // small result: staged through the handle's pinned host buffer (made once) so outputs are written only on success
    const size_t nE = s->R, nM = (size_t)s->R * s->n;
    if (!s->h_res && cudaMallocHost(&s->h_res, (nE + nM) * sizeof(double)) != cudaSuccess) {
        s->h_res = nullptr;
        return fail(SPIN_ERR_CUDA, "measure: no pinned host memory");
    }
    double *tmp = (double *)s->h_res;
    cudaError_t e = cudaMemcpyAsync(tmp, res, (nE + nM) * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(SPIN_ERR_CUDA, "measure copy: %s", cudaGetErrorString(e));
    std::memcpy(E, tmp, nE * sizeof(double));
    std::memcpy(M, tmp + nE, nM * sizeof(double));
    return SPIN_OK;
}

// E and M of every replica into DEVICE doubles d_E[R], d_M[R * n] of the caller's, enqueued on `stream`: the measurement kernels of
// spin_measure with their scratch in g_noalloc_scratch.  Calls no cudaMalloc / cudaFree / cudaMallocHost and does not synchronise.
spin_status spin_measure_noalloc(spin_system *s, double *d_E, double *d_M, void *stream) {
    if (!s || !d_E || !d_M) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    const size_t need = s->n == 1 ? (size_t)acc_slots_for(s->R) * s->R * 2 * sizeof(long long)
                                  : (size_t)s->R * s->mblocks * (1 + s->n) * sizeof(double);
    if (need > (size_t)SPIN_NOALLOC_SCRATCH_BYTES)
        return fail(SPIN_ERR_UNSUPPORTED, "spin_measure_noalloc: this system needs %zu bytes of scratch, the built-in array holds %d "
                                          "(fewer replicas, or spin_measure with the workspace)", need, (int)SPIN_NOALLOC_SCRATCH_BYTES);
    void *scratch = nullptr;
    spin_status rc = noalloc_scratch(&scratch);
    if (rc != SPIN_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const dim3 grid(s->mblocks, s->R);
    if (s->n == 1) {
        // the accumulators must start at zero, and the array keeps what the last call (of any handle) left
        CUDA_TRY(cudaMemsetAsync(scratch, 0, need, st));
        IsingArgs a = ising_args(s);
        a.acc = (long long *)scratch;
        const bool bonds = s->cfg.coupling_kind == SPIN_J_BOND_PM1;
        if (s->path == PATH_ISING_MSC) {
            const uint32_t spt = 64;
            const dim3 gm((unsigned)(((s->g.Nh + spt - 1) / spt + 127) / 128), s->R / 32);
            if (s->d == 2) ising_msc_measure<2><<<gm, 128, 0, st>>>(a, spt); else ising_msc_measure<3><<<gm, 128, 0, st>>>(a, spt);
        } else if (s->path == PATH_ISING_BITPACK) {
            if (s->d == 2) { if (bonds) ising_bitpack_measure<2, true><<<grid, 256, 0, st>>>(a); else ising_bitpack_measure<2, false><<<grid, 256, 0, st>>>(a); }
            else { if (bonds) ising_bitpack_measure<3, true><<<grid, 256, 0, st>>>(a); else ising_bitpack_measure<3, false><<<grid, 256, 0, st>>>(a); }
        } else if (s->path == PATH_ISING_INT8) {
            if (s->d == 2) ising_int8_measure<2><<<grid, 256, 0, st>>>(a); else ising_int8_measure<3><<<grid, 256, 0, st>>>(a);
        } else {
            ising_generic_measure<<<grid, 256, 0, st>>>(a);
        }
        CUDA_TRY(cudaGetLastError());
        ising_measure_finalize<<<(s->R + 3) / 4, 128, 0, st>>>(a.acc, s->R, a.acc_slots, d_E, d_M);
    } else {
        // every partial is written by its CTA before the finalize reads it: nothing to clear
        VectorArgs a = vector_args(s, 0.0);
        double *part = (double *)scratch;
        if (s->n == 2) vector_measure<2><<<grid, 256, 0, st>>>(a, part); else vector_measure<3><<<grid, 256, 0, st>>>(a, part);
        CUDA_TRY(cudaGetLastError());
        vector_measure_finalize<<<s->R, 256, 0, st>>>(part, s->mblocks, s->n, d_E, d_M);
    }
    CUDA_TRY(cudaGetLastError());
    s->launches += 2;
    return SPIN_OK;
}

// the handle's staging buffer, grown on demand (cudaMalloc / cudaFree cost milliseconds at these sizes)
static cudaError_t ensure_staging(spin_system *s, size_t bytes) {
    if (s->staging && s->staging_bytes >= bytes) return cudaSuccess;
    if (s->staging) { cudaFree(s->staging); s->staging = nullptr; s->staging_bytes = 0; }
    cudaError_t e = cudaMalloc(&s->staging, bytes);
    if (e == cudaSuccess) s->staging_bytes = bytes;
    return e;
}

static size_t canonical_spin_bytes(const spin_system *s) {
    return s->n == 1 ? (size_t)s->R * s->N : (size_t)s->R * s->N * s->n * sizeof(float);
}

// canonical spins <-> the colour arrays, everything on `st`; d_canon is device memory (the caller's or the staging buffer)
static spin_status canonical_from_arrays(spin_system *s, void *d_canon, cudaStream_t st) {
    const SetupArgs sa = setup_args(s);
    const int G = grid_for(s, 2ull * s->R * s->g.Nh);
    void *s0 = s->ws + s->lay.off_s[0], *s1 = s->ws + s->lay.off_s[1];
    if (s->path == PATH_ISING_MSC) msc_to_canonical<<<G, 256, 0, st>>>(sa, (const uint32_t *)s0, (const uint32_t *)s1, (int8_t *)d_canon);
    else if (s->n == 1) ising_to_canonical<<<G, 256, 0, st>>>(sa, s0, s1, (int8_t *)d_canon);
    else if (s->n == 2) vector_to_canonical<2><<<G, 256, 0, st>>>(sa, (const float *)s0, (const float *)s1, (float *)d_canon);
    else vector_to_canonical<3><<<G, 256, 0, st>>>(sa, (const float *)s0, (const float *)s1, (float *)d_canon);
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

// d_bad: device int, nonzero = the canonical array holds a value that is not +-1; the fill kernels then leave the arrays alone
static spin_status arrays_from_canonical(spin_system *s, const void *d_canon, const int *d_bad, cudaStream_t st) {
    const SetupArgs sa = setup_args(s);
    const int G = grid_for(s, 2ull * s->R * s->g.Nh);
    void *s0 = s->ws + s->lay.off_s[0], *s1 = s->ws + s->lay.off_s[1];
    if (s->path == PATH_ISING_MSC) msc_fill<<<G, 256, 0, st>>>(sa, 2, (const int8_t *)d_canon, (uint32_t *)s0, (uint32_t *)s1, d_bad);
    else if (s->n == 1) ising_fill<<<G, 256, 0, st>>>(sa, 2, (const int8_t *)d_canon, s0, s1, d_bad);
    else if (s->n == 2) vector_fill<2><<<G, 256, 0, st>>>(sa, 2, (const float *)d_canon, (float *)s0, (float *)s1);
    else vector_fill<3><<<G, 256, 0, st>>>(sa, 2, (const float *)d_canon, (float *)s0, (float *)s1);
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

spin_status spin_get_spins_device(spin_system *s, void *d_canon, size_t bytes, void *stream) {
    if (!s || !d_canon) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    const size_t need = canonical_spin_bytes(s);
    if (bytes != need) return fail(SPIN_ERR_INVALID_ARG, "spins need exactly %zu bytes, got %zu", need, bytes);
    return canonical_from_arrays(s, d_canon, (cudaStream_t)stream);
}

// Ising spins are checked on the device (d_flag: one int of the caller's, set nonzero if a value is not +-1, in which case nothing
// is overwritten); the caller reads the flag when it wants to know (spin_set_spins does, after synchronising)
spin_status spin_set_spins_device(spin_system *s, const void *d_canon, size_t bytes, int32_t *d_flag, void *stream) {
    if (!s || !d_canon) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    const size_t need = canonical_spin_bytes(s);
    if (bytes != need) return fail(SPIN_ERR_INVALID_ARG, "spins need exactly %zu bytes, got %zu", need, bytes);
    cudaStream_t st = (cudaStream_t)stream;
    if (s->n == 1) {
        if (!d_flag) return fail(SPIN_ERR_INVALID_ARG, "n = 1 needs d_flag (device int that receives the +-1 check)");
        CUDA_TRY(cudaMemsetAsync(d_flag, 0, sizeof(int), st));
        ising_validate_canonical<<<grid_for(s, need / 16 + 1), 256, 0, st>>>((const int8_t *)d_canon, need, d_flag);
        CUDA_TRY(cudaGetLastError());
    }
    return arrays_from_canonical(s, d_canon, s->n == 1 ? d_flag : nullptr, st);
}

// canonical bit arrays (n = 1): an eighth of the bytes over PCIe, nothing to validate
static spin_status bits_check(spin_system *s, const void *p, size_t bytes, size_t *need) {
    if (!s || !p) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (s->n != 1 || s->path == PATH_ISING_MSC || s->axis >= 0 || s->g.Lx % 8)
        return fail(SPIN_ERR_UNSUPPORTED, "bit arrays: n = 1, INT8 or BITPACK storage, whole-lattice handle, Lx %% 8 == 0");
    *need = (size_t)s->R * s->N / 8;
    if (bytes != *need) return fail(SPIN_ERR_INVALID_ARG, "spin bits need exactly %zu bytes, got %zu", *need, bytes);
    return SPIN_OK;
}

spin_status spin_set_spins_bits_async(spin_system *s, const void *host_bits, size_t bytes, void *stream) {
    size_t need = 0;
    spin_status rc = bits_check(s, host_bits, bytes, &need);
    if (rc != SPIN_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(ensure_staging(s, need));
    CUDA_TRY(cudaMemcpyAsync(s->staging, host_bits, need, cudaMemcpyHostToDevice, st));
    void *s0 = s->ws + s->lay.off_s[0], *s1 = s->ws + s->lay.off_s[1];
    if (s->path == PATH_ISING_BITPACK) {   // bits are OR-ed in
        CUDA_TRY(cudaMemsetAsync(s0, 0, s->lay.bytes_s, st));
        CUDA_TRY(cudaMemsetAsync(s1, 0, s->lay.bytes_s, st));
    }
    ising_bits_convert<<<grid_for(s, need), 256, 0, st>>>(setup_args(s), (uint8_t *)s->staging, s0, s1, true);
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

spin_status spin_get_spins_bits(spin_system *s, void *host_bits, size_t bytes, void *stream) {
    size_t need = 0;
    spin_status rc = bits_check(s, host_bits, bytes, &need);
    if (rc != SPIN_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(ensure_staging(s, need));
    ising_bits_convert<<<grid_for(s, need), 256, 0, st>>>(setup_args(s), (uint8_t *)s->staging, s->ws + s->lay.off_s[0], s->ws + s->lay.off_s[1], false);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(host_bits, s->staging, need, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return SPIN_OK;
}

spin_status spin_get_spins(spin_system *s, void *host, size_t bytes) {
    if (!s || !host) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    const size_t need = canonical_spin_bytes(s);
    if (bytes != need) return fail(SPIN_ERR_INVALID_ARG, "spins need exactly %zu bytes, got %zu", need, bytes);
    CUDA_TRY(cudaDeviceSynchronize());   // work enqueued on any stream of the caller's has to be in the arrays
    CUDA_TRY(ensure_staging(s, need));
    spin_status rc = canonical_from_arrays(s, s->staging, 0);
    if (rc != SPIN_OK) return rc;
    CUDA_TRY(cudaMemcpy(host, s->staging, need, cudaMemcpyDeviceToHost));
    return SPIN_OK;
}

// Host array -> arrays on `stream`, without a device-wide synchronisation: the upload goes in chunks, each followed by the
// +-1 check of that chunk (so the check runs under the remaining copies), then ONE fill kernel that reads the flag on the
// device and leaves the arrays alone if the check failed.  Returns after enqueueing; a failed check is reported by the
// next spin_set_spins_status (or by the blocking spin_set_spins).
spin_status spin_set_spins_async(spin_system *s, const void *host, size_t bytes, void *stream) {
    if (!s || !host) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    const size_t need = canonical_spin_bytes(s);
    if (bytes != need) return fail(SPIN_ERR_INVALID_ARG, "spins need exactly %zu bytes, got %zu", need, bytes);
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(ensure_staging(s, need + 512));
    char *staging = (char *)s->staging;
    int *d_bad = (int *)(staging + need + (256 - need % 256) % 256);  // 4 aligned bytes after the spins
    CUDA_TRY(cudaMemsetAsync(d_bad, 0, sizeof(int), st));
    const size_t chunk = (size_t)32 << 20;
    for (size_t o = 0; o < need; o += chunk) {
        const size_t n = need - o < chunk ? need - o : chunk;
        CUDA_TRY(cudaMemcpyAsync(staging + o, (const char *)host + o, n, cudaMemcpyHostToDevice, st));
        if (s->n == 1) {
            ising_validate_canonical<<<grid_for(s, n / 16 + 1), 256, 0, st>>>((const int8_t *)staging + o, n, d_bad);
            CUDA_TRY(cudaGetLastError());
        }
    }
    s->set_pending = s->n == 1;
    return arrays_from_canonical(s, staging, s->n == 1 ? d_bad : nullptr, st);
}

// the +-1 check of the last spin_set_spins_async (synchronises `stream`)
spin_status spin_set_spins_status(spin_system *s, void *stream) {
    if (!s) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (!s->set_pending) return SPIN_OK;
    const size_t need = canonical_spin_bytes(s);
    const int *d_bad = (const int *)((char *)s->staging + need + (256 - need % 256) % 256);
    int bad = 0;
    CUDA_TRY(cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
    s->set_pending = 0;
    if (bad) return fail(SPIN_ERR_INVALID_ARG, "Ising spins must be +-1 (the arrays were left as they were)");
    return SPIN_OK;
}

spin_status spin_set_spins(spin_system *s, const void *host, size_t bytes) {
    if (!s || !host) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    CUDA_TRY(cudaDeviceSynchronize());   // sweeps enqueued on any stream of the caller's come first
    spin_status rc = spin_set_spins_async(s, host, bytes, nullptr);
    if (rc != SPIN_OK) return rc;
    rc = spin_set_spins_status(s, nullptr);
    if (rc != SPIN_OK) return rc;
    CUDA_TRY(cudaStreamSynchronize(0));
    return SPIN_OK;
}

spin_status spin_get_bonds(spin_system *s, int8_t *host, size_t bytes) {
    if (!s || !host) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    if (s->cfg.coupling_kind != SPIN_J_BOND_PM1) return fail(SPIN_ERR_INVALID_ARG, "system has no per-bond couplings");
    const size_t need = (size_t)s->R * s->d * s->N;
    if (bytes != need) return fail(SPIN_ERR_INVALID_ARG, "bonds need exactly %zu bytes, got %zu", need, bytes);
    CUDA_TRY(cudaDeviceSynchronize());
    if (s->path != PATH_ISING_BITPACK && s->path != PATH_ISING_MSC) {
        CUDA_TRY(cudaMemcpy(host, s->ws + s->lay.off_bonds, need, cudaMemcpyDeviceToHost));
        return SPIN_OK;
    }
    CUDA_TRY(ensure_staging(s, need));
    void *staging = s->staging;
    if (s->path == PATH_ISING_MSC) msc_bonds_unpack<<<grid_for(s, 2ull * s->R * s->g.Nh), 256>>>(setup_args(s), (const uint32_t *)(s->ws + s->lay.off_bonds), (int8_t *)staging);
    else
    bonds_unpack<<<grid_for(s, 2ull * s->R * s->g.Nh), 256>>>(setup_args(s), (const uint32_t *)(s->ws + s->lay.off_bonds), (int8_t *)staging);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpy(host, staging, need, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail(SPIN_ERR_CUDA, "get_bonds: %s", cudaGetErrorString(e));
    return SPIN_OK;
}

spin_status spin_get_sweep_count(const spin_system *s, uint64_t *t) {
    if (!s || !t) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    *t = s->t;
    return SPIN_OK;
}

spin_status spin_set_sweep_count(spin_system *s, uint64_t t) {
    if (!s) return fail(SPIN_ERR_INVALID_ARG, "handle is NULL");
    if (t > 0x100000000ull) return fail(SPIN_ERR_INVALID_ARG, "sweep counter is 32 bits wide");
    s->t = t;
    return SPIN_OK;
}

spin_status spin_get_launch_count(const spin_system *s, uint64_t *launches) {
    if (!s || !launches) return fail(SPIN_ERR_INVALID_ARG, "NULL argument");
    *launches = s->launches;
    return SPIN_OK;
}

spin_status spin_set_launch_shape(spin_system *s, int32_t block, int32_t grid_num, int32_t grid_den) {
    if (!s) return fail(SPIN_ERR_INVALID_ARG, "handle is NULL");
    if (block == 0) block = (s->path == PATH_ISING_INT8 || s->path == PATH_ISING_BITPACK) ? 128 : 256;
    if (block != 64 && block != 128 && block != 256) return fail(SPIN_ERR_INVALID_ARG, "block must be 64, 128 or 256");
    if (grid_num < 1 || grid_den < 1) return fail(SPIN_ERR_INVALID_ARG, "grid_num / grid_den must be >= 1");
    s->block = block; s->grid_num = grid_num; s->grid_den = grid_den;
    return SPIN_OK;
}

spin_status spin_set_strip_rows(spin_system *s, int32_t rows) {
    if (!s) return fail(SPIN_ERR_INVALID_ARG, "handle is NULL");
    const int chosen = rows != 0;
    if (rows == 0) rows = 4;
    if (rows != 1 && rows != 2 && rows != 4 && rows != 8 && rows != 16)
        return fail(SPIN_ERR_INVALID_ARG, "strip rows must be 1, 2, 4, 8 or 16");
    s->strip_rows = rows;
    s->strip_rows_set = chosen;
    return SPIN_OK;
}

spin_status spin_set_option(spin_system *s, int32_t option, int64_t value) {
    if (!s) return fail(SPIN_ERR_INVALID_ARG, "handle is NULL");
    if (option == SPIN_OPT_PLAIN_KERNELS) {
        if (value != 0 && value != 1) return fail(SPIN_ERR_INVALID_ARG, "SPIN_OPT_PLAIN_KERNELS takes 0 or 1");
        s->vector_generic = (int)value;
        return SPIN_OK;
    }
    if (option == SPIN_OPT_TMA_KERNELS) {
        if (value != 0 && value != 1 && value != -1) return fail(SPIN_ERR_INVALID_ARG, "SPIN_OPT_TMA_KERNELS takes 0, 1 or -1");
        s->use_tma = (int)value;
        return SPIN_OK;
    }
    if (option == SPIN_OPT_TEMPORAL_BLOCKING) {
        if (value < -1 || value > 1) return fail(SPIN_ERR_INVALID_ARG, "SPIN_OPT_TEMPORAL_BLOCKING takes -1, 0 or 1");
        s->tblock = (int)value;
        return SPIN_OK;
    }
    if (option == SPIN_OPT_TBLOCK_ROWS) {
        if (value < 0 || value > (1 << 24)) return fail(SPIN_ERR_INVALID_ARG, "SPIN_OPT_TBLOCK_ROWS takes 0 (automatic) or a number of rows");
        s->tblock_rows = (int)value;
        return SPIN_OK;
    }
    if (option == SPIN_OPT_L2_KEEP) {
        if (value < -2 || value > 65535) return fail(SPIN_ERR_INVALID_ARG, "SPIN_OPT_L2_KEEP takes -2 (no hints), -1 (automatic) or a number of replicas");
        s->l2_keep = (int)value;
        graph_drop(s);
        return SPIN_OK;
    }
    if (option == SPIN_OPT_DEFER_CAP) {
        if (value < 0 || value > DEFER_CAP) return fail(SPIN_ERR_INVALID_ARG, "SPIN_OPT_DEFER_CAP takes 0 .. %d", DEFER_CAP);
        s->defer_cap = (int)value;
        graph_drop(s);
        return SPIN_OK;
    }
    if (option == SPIN_OPT_KERNEL_VARIANT) {
        if (value < 0 || value > 15) return fail(SPIN_ERR_INVALID_ARG, "SPIN_OPT_KERNEL_VARIANT takes 0 .. 15");
        s->variant = (int)value;
        graph_drop(s);
        return SPIN_OK;
    }
    if (option == SPIN_OPT_L2_PREFETCH) {
        if (value < -1 || value > (1 << 20)) return fail(SPIN_ERR_INVALID_ARG, "SPIN_OPT_L2_PREFETCH takes -1, 0 or a distance up to 2^20");
        s->l2_prefetch = (int)value;
        graph_drop(s);   // captured argument blocks hold the old distance
        return SPIN_OK;
    }
    return fail(SPIN_ERR_INVALID_ARG, "unknown option %d", (int)option);
}

}  // extern "C"
