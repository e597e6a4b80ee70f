/*
 * spin.h -- C ABI of libspin: checkerboard single-spin-flip Metropolis sweeps for O(n)
 * lattice spin models on one B200 (sm_100a), plus the energy / magnetisation sums.
 *
 * What the calls compute (PAPER.md = the text of arXiv:1107.5463):
 *   PAPER.md:31-35  Eq. (1)  H = -sum_<ij> J_ij s_i . s_j ; n = 1 Ising, 2 XY, 3 Heisenberg;
 *                            square (d = 2) / simple-cubic (d = 3) lattice, nearest neighbours
 *   PAPER.md:37-38  Eq. (2)  p_acc(s -> s') = min[1, exp(-beta dE)]                 (spin_sweep)
 *   PAPER.md:42              checkerboard decomposition: all spins of one sub-lattice are
 *                            updated concurrently, then the other; tabulated Boltzmann
 *                            factors; a random number is drawn for every site      (spin_sweep)
 *   PAPER.md:44              fp32 spins, fp64 aggregates (total energy)            (spin_measure)
 *   PAPER.md:46, 52          disorder realisations side by side; multi-spin coding (n_replicas, BITPACK)
 * Readings where the paper is silent (periodic boundaries, one sweep = colour 0 then colour 1,
 * k = 1, Philox-4x32-10 keyed by (seed, sweep, colour, site), ...) are listed in DESIGN.md.
 *
 * Conventions
 *   - Every call returns a spin_status; nothing throws or aborts across the ABI; outputs are
 *     written only on SPIN_OK.  spin_last_error() gives a thread-local message.
 *   - The CALLER owns device memory: spin_create() carves everything it needs out of the
 *     device workspace passed in (size from spin_workspace_bytes()).  The only memory the library
 *     allocates itself: one device staging buffer for canonical arrays, created by the first HOST-array
 *     get/set call, reused by later ones and freed by spin_destroy() (the *_device variants take the
 *     caller's device arrays instead and allocate nothing); a few pinned host doubles for
 *     spin_measure's result (first call; spin_measure_noalloc has none); and the fixed 1 MiB device
 *     array of spin_measure_noalloc, part of the library image.
 *   - "stream" arguments are cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - spin_sweep / spin_sweep_record / spin_sweep_betas / spin_halfsweep* / spin_halo_* / spin_measure_noalloc and the
 *     *_async / *_device conversions only enqueue work; spin_measure and the host-array get/set calls block.
 *   - A handle is not thread-safe; different handles are independent.
 *   - Sites: (x, y, z), lexicographic index i = x + Lx (y + Ly z); colour = (x + y + z) mod 2;
 *     colour 0 is updated first.  Periodic boundaries in every direction.
 */
#ifndef SPIN_H
#define SPIN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spin_system spin_system; /* opaque, host-side, owned by the library */

typedef enum {
    SPIN_OK = 0,
    SPIN_ERR_INVALID_ARG = 1,         /* NULL pointer, odd dimension, beta < 0 or NaN, bad enum, ... */
    SPIN_ERR_UNSUPPORTED = 2,         /* valid request the kernels do not cover (see spin_config)     */
    SPIN_ERR_WORKSPACE_TOO_SMALL = 3,
    SPIN_ERR_CUDA = 4,                /* a CUDA runtime call failed; message has cudaGetErrorString   */
    SPIN_ERR_STATE = 5                /* sweep counter would pass 2^32 - 1                            */
} spin_status;

enum { SPIN_STORE_INT8 = 0,   /* n = 1: one byte per spin                                             */
       SPIN_STORE_BITPACK = 1,/* n = 1: one bit per spin, 32 same-colour sites per word (multi-spin
                                 coding); needs Lx % 64 == 0 and |J| = 1                 */
       SPIN_STORE_FP32 = 2,   /* n = 2, 3: fp32 unit vectors, one plane per component and colour      */
       SPIN_STORE_MSC = 3 };  /* n = 1, SPIN_J_BOND_PM1, replica_streams = 0, n_replicas % 32 == 0,
                                 N / 2 % 32 == 0: one bit per spin, the 32 realisations 32 k .. 32 k + 31
                                 of ONE site per word ("asynchronous" multi-spin coding over disorder
                                 realisations; Table 1 "Metro. multi-spin"): every
                                 realisation of a site sees the same random number.  Takes L = 32.      */
enum { SPIN_J_UNIFORM = 0,        /* J[0] on every bond                                               */
       SPIN_J_PER_DIRECTION = 1,  /* J[mu] on bonds in direction mu = x, y, z                         */
       SPIN_J_BOND_PM1 = 2 };     /* one +-1 per bond and replica (Edwards-Anderson); n = 1 */
enum { SPIN_UPDATE_METROPOLIS = 0, /* Eq. (2): accept with min[1, exp(-beta dE)]          */
       SPIN_UPDATE_HEATBATH = 1 }; /* the new spin is drawn from its conditional Boltzmann law in
                                      the local field h = sum_j J_ij s_j, whatever the old value.  n = 1:
                                      s = +1 iff U < floor(2^32 / (1 + exp(-2 beta h))); n = 3: cosine about h by
                                      inversion, c = 1 + ln(1 - u (1 - e^{-2H})) / H, H = beta |h|, uniform azimuth
                                      (DESIGN.md section 2).  n = 2 -> SPIN_ERR_UNSUPPORTED                   */
enum { SPIN_INIT_HOT = 0,         /* iid uniform spins drawn from the seed                            */
       SPIN_INIT_COLD = 1 };      /* all +1 (n = 1), (1, 0) (n = 2), (0, 0, 1) (n = 3)                */

typedef struct {
    int32_t dims[3];         /* Lx, Ly, Lz.  Lz == 1 -> d = 2.  Lx, Ly (and Lz if > 1) even, >= 2.      */
    int32_t n;               /* 1 Ising, 2 XY, 3 Heisenberg                                             */
    int32_t storage;         /* SPIN_STORE_*; INT8/BITPACK need n = 1, FP32 needs n >= 2                */
    int32_t coupling_kind;   /* SPIN_J_*                                                                */
    double  J[3];            /* UNIFORM: J[0]; PER_DIRECTION: Jx, Jy, Jz.  n = 1: each in {-1, 0, +1}   */
    const int8_t *bonds;     /* BOND_PM1: HOST array [replica][mu][i] (mu < d) of +-1, the coupling of
                                the bond leaving site i in direction +mu; NULL -> drawn iid +-1, p = 1/2,
                                from the seed.  Read during spin_create only.                          */
    int32_t n_replicas;      /* 1 <= R <= 65535 independent systems stored side by side   */
    int32_t replica_streams; /* 0: all replicas see the same random numbers (needs distinct bonds or
                                starts to be useful); 1: the replica index enters the Philox counter    */
    int32_t init;            /* SPIN_INIT_*                                                             */
    uint64_t seed;           /* Philox key                                                              */
    int32_t update_rule;     /* SPIN_UPDATE_*                                                           */
    /* Slab decomposition over several handles / GPUs; both 0 = the handle holds the whole lattice.
     * dims[] are then the LOCAL extents: the handle owns planes [slab_offset, slab_offset + dims[axis]) of a lattice
     * whose extent along the slowest axis (z for d = 3, y for d = 2) is slab_global.  Both even.  Random numbers are
     * keyed by GLOBAL site indices, so the slabs together reproduce the unsharded lattice bit for bit.  Uniform or
     * per-direction couplings only.  Drive with spin_halfsweep + spin_halo_get / spin_halo_put. */
    int32_t slab_global;
    int32_t slab_offset;
} spin_config;

/* Bytes of device workspace spin_create() needs for this configuration. */
spin_status spin_workspace_bytes(const spin_config *cfg, size_t *bytes);

/* Build a system inside d_workspace (DEVICE pointer, 256-byte aligned, `bytes` long, owned by the
 * caller and kept alive until spin_destroy): draws or uploads the bonds, initialises the spins,
 * sweep counter = 0.  Work is enqueued on `stream` and synchronised before returning. */
spin_status spin_create(const spin_config *cfg, void *d_workspace, size_t bytes, void *stream, spin_system **out);

/* n_sweeps full sweeps (half-sweep of colour 0, then of colour 1) at inverse temperature
 * beta >= 0, enqueued on `stream`; returns without synchronising.  sweep(b, a); sweep(b, c) is
 * identical to sweep(b, a + c).  The sweep counter (the Philox sweep index) advances by n_sweeps. */
spin_status spin_sweep(spin_system *s, double beta, int64_t n_sweeps, void *stream);

/* E[r] = -sum over bonds J s.s (each bond once), M[r*n + a] = sum_i s_i^a (Eq. (1); double
 * aggregates).  E, M are HOST pointers to R and R*n doubles.  n = 1: both are exact integers.
 * Runs on `stream` and blocks until the result is on the host. */
spin_status spin_measure(spin_system *s, double *E, double *M, void *stream);

/* The same measurement for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): E and M go to DEVICE doubles d_E[R], d_M[R*n] of the caller's, the call only enqueues work on
 * `stream` (no synchronisation) and calls no cudaMalloc, cudaFree or other allocating routine.  The kernels' scratch
 * (per-CTA partial sums, accumulator slots) lives in ONE array built into the library, SPIN_NOALLOC_SCRATCH_BYTES per
 * GPU (held by every GPU that loads the library until the process exits).  A system that needs more --
 * n = 1: 16 * min(64, 8192 / R rounded down to a power of two) * R bytes; n >= 2: up to 592 * 8 * (1 + n) * R bytes,
 * i.e. beyond about 55 Heisenberg replicas -- is refused with SPIN_ERR_UNSUPPORTED (use spin_measure).
 * Every call, of every handle, shares that array: calls that overlap on the GPU (different streams without ordering)
 * race; calls on one stream are safe, and the array is cleared where a kernel needs zeros.  Values are identical to
 * spin_measure's. */
#define SPIN_NOALLOC_SCRATCH_BYTES (1 << 20)
spin_status spin_measure_noalloc(spin_system *s, double *d_E, double *d_M, void *stream);

/* One half-sweep (colour 0, then colour 1, alternating; the sweep counter advances after colour 1), enqueued on
 * `stream`.  For slab handles the caller exchanges halos in between: before the half-sweep of colour c every handle
 * needs its neighbours' boundary planes of colour 1 - c (spin_halo_get on the owner, spin_halo_put here). */
spin_status spin_halfsweep(spin_system *s, double beta, int32_t colour, void *stream);

/* Slab handles: bytes of one face (one boundary plane of one colour, all replicas / components). */
spin_status spin_halo_bytes(const spin_system *s, size_t *bytes);
/* Copy the OWNED boundary plane of colour `colour` on side 0 (lowest owned plane) or 1 (highest) into the contiguous
 * DEVICE buffer d_buf / copy d_buf into the GHOST plane below (side 0) or above (side 1) the owned planes.  Async. */
spin_status spin_halo_get(spin_system *s, int32_t colour, int32_t side, void *d_buf, void *stream);
spin_status spin_halo_put(spin_system *s, int32_t colour, int32_t side, const void *d_buf, void *stream);

/* The half-sweep of `colour` restricted to planes [plane0, plane0 + n_planes) of the planes this handle updates (slab
 * handle: its owned planes, 0-based; whole lattice: planes along its slowest axis).  Sites of one colour do not
 * interact, so a half-sweep may be issued in pieces, in any order: a slab updates its two boundary planes first, sends
 * them, and updates the interior while the messages are in flight ("overlap by updating boundary planes
 * first").  last != 0 on the piece that completes the colour (the handle then expects the other colour; after colour 1
 * the sweep counter advances); the caller covers every plane exactly once.  n_planes = 0 with last != 0 only closes the
 * colour.  Asynchronous. */
spin_status spin_halfsweep_range(spin_system *s, double beta, int32_t colour, int32_t plane0, int32_t n_planes,
                                 int32_t last, void *stream);

/* Both faces of one colour with ONE kernel each way.  d_buf: device memory, 2 * spin_halo_bytes, 16-byte aligned.
 * pack:   d_buf = [lowest owned plane][highest owned plane] (the messages for the slab below and the slab above).
 * unpack: d_buf = [plane received from the slab below][plane received from the slab above] -> the two ghost planes.
 * Asynchronous on `stream`. */
spin_status spin_halo_pack(spin_system *s, int32_t colour, void *d_buf, void *stream);
spin_status spin_halo_unpack(spin_system *s, int32_t colour, const void *d_buf, void *stream);
/* A slab that is its own neighbour (one rank holds the whole extent, periodic): ghost below <- highest owned plane,
 * ghost above <- lowest owned plane, one kernel.  Asynchronous. */
spin_status spin_halo_wrap(spin_system *s, int32_t colour, void *stream);
/* Peer stores instead of messages ("direct peer stores over NVLink 5 / NVSwitch"): spin_colour_array gives
 * the device address (and size) of a handle's colour array, which the owner of a neighbouring slab may map on its own GPU
 * (same process: cudaDeviceEnablePeerAccess; another process: CUDA IPC); spin_halo_push then writes this handle's two
 * owned boundary planes of `colour` straight into the ghost planes of the slab below (d_peer_below = THAT handle's colour
 * array) and of the slab above, with one kernel and no message buffer.  Both neighbours must have this handle's slab
 * thickness and layout.  The push is ordered on `stream` only: the caller makes sure (event, barrier) that a neighbour
 * does not start the half-sweep that reads the ghosts before the push has completed.  Asynchronous. */
spin_status spin_colour_array(spin_system *s, int32_t colour, void **d_ptr, size_t *bytes);
spin_status spin_halo_push(spin_system *s, int32_t colour, void *d_peer_below, void *d_peer_above, void *stream);

/* Temperature axis ("trivial parallelization"): n_sweeps sweeps with replica r at
 * betas[r] (host array of n_replicas doubles, read before the call returns) -- many temperatures of one model side by
 * side, the layout parallel tempering needs.  Needs replica_streams = 1 (or one replica); replica r then follows exactly
 * the chain it would follow in a handle swept at betas[r].  Runs one launch per replica and half-sweep with the
 * ordinary kernels.  SPIN_ERR_UNSUPPORTED for bit-packed per-bond couplings and MSC storage.  Asynchronous. */
spin_status spin_sweep_betas(spin_system *s, const double *betas, int64_t n_sweeps, void *stream);

/* As spin_sweep, recording E and M after every sweep into DEVICE arrays d_E[n_sweeps][R] and
 * d_M[n_sweeps][R][n] (doubles).  Enqueues only. */
spin_status spin_sweep_record(spin_system *s, double beta, int64_t n_sweeps, double *d_E, double *d_M, void *stream);

/* Canonical HOST layouts.  n = 1: int8 [replica][i] of +-1; n >= 2: float [replica][i][n].  Blocking. */
spin_status spin_get_spins(spin_system *s, void *host, size_t bytes);
spin_status spin_set_spins(spin_system *s, const void *host, size_t bytes);

/* The same two conversions without a device-wide synchronisation and without library-owned memory.
 * spin_get_spins_device / spin_set_spins_device: the canonical array lives in DEVICE memory of the caller's (the same
 *   layout and size as above); the conversion kernel is enqueued on `stream`.  For n = 1 the +-1 check needs d_flag, one
 *   device int of the caller's: it is set nonzero if a value is not +-1, and the arrays are then left as they were.
 * spin_set_spins_async: host array (pinned for a truly asynchronous upload) -> arrays on `stream`: chunked upload into the
 *   handle's staging buffer, the +-1 check of each chunk under the remaining copies, one conversion kernel that the check
 *   guards on the device.  Returns after enqueueing; spin_set_spins_status(stream) synchronises `stream` and reports the
 *   check (SPIN_ERR_INVALID_ARG if it failed; the arrays are then unchanged).  The host array must stay valid until then. */
spin_status spin_get_spins_device(spin_system *s, void *d_canon, size_t bytes, void *stream);
spin_status spin_set_spins_device(spin_system *s, const void *d_canon, size_t bytes, int32_t *d_flag, void *stream);
spin_status spin_set_spins_async(spin_system *s, const void *host, size_t bytes, void *stream);
spin_status spin_set_spins_status(spin_system *s, void *stream);

/* Ising configurations as canonical BIT arrays (n = 1, INT8 or BITPACK storage, whole-lattice handles, Lx % 8 == 0):
 * bit (i & 7) of byte (r N + i) >> 3 is 1 iff spin i of replica r is -1; n_replicas * N / 8 bytes -- an eighth of the int8
 * array across PCIe, and every bit pattern is a valid configuration, so there is nothing to check.
 * spin_set_spins_bits_async: host array (pinned for an asynchronous upload; it must stay valid until `stream` has consumed
 * it) -> arrays, enqueued on `stream`.  spin_get_spins_bits: arrays -> host array; synchronises `stream`. */
spin_status spin_set_spins_bits_async(spin_system *s, const void *host_bits, size_t bytes, void *stream);
spin_status spin_get_spins_bits(spin_system *s, void *host_bits, size_t bytes, void *stream);
/* BOND_PM1 only: int8 [replica][mu][i] of +-1.  Blocking. */
spin_status spin_get_bonds(spin_system *s, int8_t *host, size_t bytes);

spin_status spin_get_sweep_count(const spin_system *s, uint64_t *t);
spin_status spin_set_sweep_count(spin_system *s, uint64_t t);

/* Number of kernel launches this handle has enqueued so far (bench.py's gpu_launches). */
spin_status spin_get_launch_count(const spin_system *s, uint64_t *launches);

/* Tuning knob for tests: multiply the default grid size by num/den and use `block` threads per CTA
 * (0 = default).  Results never depend on it (the RNG is counter-based). */
spin_status spin_set_launch_shape(spin_system *s, int32_t block, int32_t grid_num, int32_t grid_den);

/* Tuning knob of the int8 Ising kernel: rows of one unit column a thread sweeps before moving on
 * (1, 2, 4, 8 or 16; 0 = default).  Results never depend on it. */
spin_status spin_set_strip_rows(spin_system *s, int32_t rows);

/* Test knob: value 1 selects the plain kernels (one launch per half-sweep, one thread per site for n >= 2,
 * no resident small-lattice kernel), 0 (default) the tuned ones.  Results never depend on it bit for bit. */
enum { SPIN_OPT_PLAIN_KERNELS = 0,
       /* The TMA-staged kernel of the n >= 2 models (d = 3, Lx <= 512: tiles and halos staged in shared memory by
        * cp.async.bulk.tensor, PAPER.md:42 tile + boundary layer): 1 = every half-sweep, 0 = never (strip kernel),
        * -1 (default) = only for the colour-1 half-sweep of spin_sweep_record, where its fused E / M saves the
        * measurement pass; elsewhere the strip kernel is the faster one on B200 (profiles/).  Spins are bit-identical
        * whichever kernel runs. */
       SPIN_OPT_TMA_KERNELS = 1,
       /* Bulk L2 prefetch (cp.async.bulk.prefetch.L2) issued by the +-J quad kernel (value = replicas ahead) and the
        * n >= 2 strip kernel (value = CTAs ahead): -1 (default) = each kernel's own distance, 0 = off.  A pure
        * performance hint: results never depend on it. */
       SPIN_OPT_L2_PREFETCH = 2,
       /* A/B knob: 0 (default) = the tuned kernel of each family; 1 = the alternative kept beside it
        * (+-J shared stream: one thread per quad and all replicas, instead of the cooperative kernel with one CTA of replica-chunk warps per 32 quads;
        * many +-J realisations of a lattice of at most 512 words per colour, shared stream: one launch per half-sweep instead of the
        * kernel that keeps groups of realisations in shared memory for all sweeps of a spin_sweep call).  Results never
        * depend on it. */
       SPIN_OPT_KERNEL_VARIANT = 3,
       /* Exact temporal blocking ("k updates per tile load", made results-neutral): spin_sweep
        * runs pairs of sweeps in one pass over the lattice (each row read once and written once per two sweeps), bit-identical
        * to plain sweeps.  Offered for 2D Ising, INT8 storage, uniform J = +-1, both update rules, 2048 <= Lx <= 32768,
        * Lx % 2048 == 0, own random stream per replica; such handles ask for twice the spin storage (spin_workspace_bytes).
        * -1 (default) = on for the Metropolis rule on INT8 lattices too large for the CUDA-graph regime, 0 = off,
        * 1 = on wherever offered. */
       SPIN_OPT_TEMPORAL_BLOCKING = 4,
       /* rows per stripe of the temporal-blocking kernel; 0 (default) = one wave of resident CTAs */
       SPIN_OPT_TBLOCK_ROWS = 5,
       /* L2 eviction priorities of the +-J quad kernel (createpolicy / ld.global.L2::cache_hint): the spins and the coupling
        * words of `value` replicas are kept in L2 from half-sweep to half-sweep ("evict_last"), the other coupling words are
        * streamed ("evict_first").  -1 (default) = as many replicas as fit in two thirds of L2 when the working set exceeds
        * L2, -2 = no hints.  A pure performance hint. */
       SPIN_OPT_L2_KEEP = 6,
       /* Capacity (0 .. 32, default 32) of the per-warp queue of the deferred digit comparison (bit-packed / int8 strip
        * kernels, own-stream +-J kernel): a thread that finds the queue full finishes its word itself.  Results do not
        * depend on it (the same digits decide either way); 0 finishes every word inline.  Exists so that the overflow
        * path, which a full queue takes about once in 10^6 warps, can be exercised by tests. */
       SPIN_OPT_DEFER_CAP = 7 };
spin_status spin_set_option(spin_system *s, int32_t option, int64_t value);

/* Frees the handle only; never the workspace. */
spin_status spin_destroy(spin_system *s);

/* Thread-local message of the last failing call on this thread ("" if none). */
const char *spin_last_error(void);

/* Library version string, e.g. "libspin 0.1 sm_100a". */
const char *spin_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPIN_H */
