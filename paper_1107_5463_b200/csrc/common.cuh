// common.cuh -- device-side building blocks shared by every libspin kernel (sm_100a).
// Product code: shares nothing with oracle/.  The algorithm both follow is DESIGN.md "The contract".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace spin {

// ---------------------------------------------------------------------------------------------
// Philox-4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  The ten round keys depend only on the seed,
// so the host expands them once and they reach the kernels as __grid_constant__ parameters: the
// XORs take them straight from the constant bank and a call is 20 IMAD.WIDE + 20 LOP3.
struct PhiloxKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const PhiloxKeys &K, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Counter layout of DESIGN.md: ctr = (unit, rho, t, tag), tag = colour + 16 domain + 256 call.
enum : uint32_t { DOM_ISING_UPDATE = 0, DOM_INIT = 1, DOM_BONDS = 2, DOM_VECTOR_UPDATE = 3 };
__host__ __device__ __forceinline__ uint32_t make_tag(uint32_t colour, uint32_t domain, uint32_t call) {
    return colour + 16u * domain + 256u * call;
}

// ---------------------------------------------------------------------------------------------
// Bulk L2 prefetch (sm_90+: cp.async.bulk.prefetch.L2): one thread asks the memory system to bring `bytes` contiguous
// bytes (a multiple of 16, 16-byte aligned) from HBM into L2.  No register or shared-memory cost; the half-sweep kernels
// use it to turn the DRAM latency of data that a later CTA / the next replica iteration will load into an L2 hit.
__device__ __forceinline__ void l2_prefetch_bulk(const void *p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// L2 eviction-priority hints (createpolicy + ld.global.L2::cache_hint): data that the next half-sweep reads again is loaded
// "evict_last", data that is streamed once per half-sweep "evict_first", so that a working set a little larger than L2 keeps its
// reusable part resident instead of thrashing the whole cache.
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint4 ldg_hint(const uint4 *ptr, uint64_t policy) {
    uint4 v;
    asm volatile("ld.global.nc.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(ptr), "l"(policy));
    return v;
}

__device__ __forceinline__ uint4 ld_hint(const uint4 *ptr, uint64_t policy) {   // coherent load (array written by the kernel)
    uint4 v;
    asm volatile("ld.global.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(ptr), "l"(policy) : "memory");
    return v;
}
__device__ __forceinline__ void st_hint(uint4 *ptr, const uint4 &v, uint64_t policy) {
    asm volatile("st.global.L2::cache_hint.v4.u32 [%0], {%1, %2, %3, %4}, %5;"
                 ::"l"(ptr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(policy) : "memory");
}

// ---------------------------------------------------------------------------------------------
// Division by a run-time constant fixed at handle creation: q = (n * mul) >> (32 + shift) for
// n < 2^31 (round-up method).  Two instructions instead of ~20.
struct FastDiv {
    uint32_t mul;
    uint32_t shift;
    uint32_t div;
};
__device__ __forceinline__ uint32_t fdiv(uint32_t n, const FastDiv &d) {
    return d.div == 1u ? n : (__umulhi(n, d.mul) >> d.shift);
}

// ---------------------------------------------------------------------------------------------
// Boltzmann thresholds for n = 1 ("pre-tabulation of the Boltzmann factors"):
// T(dE) = floor(exp(-beta dE) 2^32), compared bit-serially, most significant digit first, against
// the site's 32-bit uniform whose digit k is bit `lane` of Philox word k of the site's unit
// (bit-plane contract).  digit[th][k] is the k-th digit of T(4 (th + 1)) spread to a full mask
// (0 or ~0); always[th] = ~0 iff T = 2^32 (factor 1: every lane accepts).
struct IsingTable {
    uint32_t digit[3][32];
    uint32_t always[3];
    uint32_t T[13];       // low 32 bits of T(dE), dE = 0..12 (generic kernel)
    uint32_t Talways;     // bit dE set iff T(dE) = 2^32
};

// Heat-bath rule for n = 1: P(s = +1 | h) = 1 / (1 + exp(-2 beta h)), h = sum_j J s_j in {-q .. q},
// tabulated as T_hb = floor(P 2^32).  The bit-sliced kernels index by the number k of neighbour terms J s_j that
// equal -1 (h = q - 2 k, q = 2 d): digit[k][dg], always[k] as in IsingTable; T / Talways are indexed by h + 6.
struct HeatBathTable {
    uint32_t digit[7][32];
    uint32_t always[7];
    uint32_t T[13];
    uint32_t Talways;
};

// Lattice geometry in the colour-compressed layout.  A colour-c site (x, y, z) has compressed
// index j = (x >> 1) + RL (y + Ly z), RL = Lx / 2; all its neighbours are in the other colour's array:
// same row at x >> 1 and at (x >> 1) -+ 1 (minus if x is even), rows y -+ 1 and planes z -+ 1 at x >> 1.
struct Geometry {
    int32_t Lx, Ly, Lz, d;
    uint32_t RL;      // sites per row and colour = Lx / 2
    uint32_t rows;    // Ly * Lz
    uint32_t Nh;      // sites per colour = N / 2
    uint32_t WX;      // 32-site words per row and colour = RL / 32 (fast kernels only)
    uint32_t NW;      // words per colour = Nh / 32 (fast kernels only)
    FastDiv divRL, divWX, divLy;
    FastDiv divQW;    // by WX / 4 (quads of four words per row and colour; +-J quad kernel)
    FastDiv divQX;    // by RL / 4 (quads of 4 sites per row and colour; strip kernel of the n >= 2 models)
    // Slab decomposition: this handle holds planes [slab_offset, slab_offset + L_own) of a larger
    // lattice along its slowest axis (z for d = 3, y for d = 2), stored with two ghost planes on either side, so the
    // local arrays look like a periodic lattice of L_own + 4 planes.  The kernels sweep all of it (the ghost planes are
    // overwritten by the halo exchange before they are read) and only need the offsets that turn a local index into
    // the global one that feeds Philox, and the owned range for the measurements and the canonical get / set.
    // Not sharded: offsets 0, owned range = everything.
    uint32_t j_off;     // + local compressed index  -> global compressed index (mod 2^32)
    uint32_t unit_off;  // + local 32-site unit      -> global unit             (mod 2^32; fast layouts)
    uint32_t i_off;     // + local lexicographic idx -> global lexicographic index (mod 2^32)
    uint32_t own_j0, own_j1;   // owned compressed indices [own_j0, own_j1) of either colour
    uint32_t own_i0, own_in;   // owned lexicographic indices [own_i0, own_i0 + own_in)
    // What a half-sweep launch updates: planes [sw_p0, sw_p0 + sw_pn) along the slowest axis (z for d = 3, rows y for
    // d = 2) = compressed indices [sw_j0, sw_j0 + sw_jn).  Whole lattice: everything.  Slab handle: its owned planes (the
    // ghost planes are only read), or a sub-range of them when the caller updates the boundary planes first and the
    // interior while the halo exchange is in flight (spin_halfsweep_range).
    uint32_t sw_p0, sw_pn, sw_j0, sw_jn;
};

}  // namespace spin
