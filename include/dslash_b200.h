/*
 * dslash_b200.h -- C ABI of the B200-native Wilson Dslash library (libdslash_b200.so, sm_100a).
 *
 * The operator (section 1.1, Eq. 1; backward link argument corrected to x-mu^ as in
 * BASELINE.json's north_star -- DESIGN.md Reading R1):
 *
 *   out(x) = sum_{mu=0..3} [ (1 - gamma_mu) U_mu(x) in(x+mu^)  +  (1 + gamma_mu) U_mu(x-mu^)^dagger in(x-mu^) ]
 *
 * on a periodic 4-D lattice dims = {L_X, L_Y, L_Z, L_T}; U_mu(x) in SU(3) acts on the colour index
 * (COLORS = 3), gamma_mu (DeGrand-Rossi basis, DESIGN.md Reading R4) on the spin index (SPINS = 4)
 * (PAPER.md:52).  mu = 0,1,2,3 <-> x,y,z,t.  No mass term, no factor 1/2.
 *
 * Conventions common to every call
 *   - Every function returns an int status: DSLASH_OK (0) or a negative DSLASH_ERR_* code.  Nothing
 *     throws, aborts or prints.  dslash_error_string() names a code.
 *   - "device pointer" = CUDA global memory on the device that was current at dslash_create();
 *     "host pointer" = ordinary or pinned host memory.  The library never takes ownership of a
 *     caller's buffer, never frees it and never keeps it beyond the call (asynchronous work on
 *     `stream` excepted: buffers must stay alive until that work has finished).
 *   - stream: a cudaStream_t passed as an opaque pointer (NULL = the legacy default stream).  All
 *     device work of a call is enqueued on it; no call except dslash_apply_host() and
 *     dslash_destroy() synchronises.
 *   - A ctx may be used from one host thread at a time; distinct ctxs are independent.
 *   - There is no CPU fallback: without a CUDA device dslash_create() returns DSLASH_ERR_CUDA.
 *
 * Canonical layout ("array of structures", the flat arrays of PAPER.md:52 with the loop order of
 * PAPER.md:54; x fastest):   site s = x + L_X*(y + L_Y*(z + L_Z*t)),  V = L_X*L_Y*L_Z*L_T
 *     spinor  real[ ((s*4 + spin)*3 + colour)*2 + ri ]                      24 reals per site
 *     gauge   real[ (((s*4 + mu)*3 + row)*3 + col)*2 + ri ]                 72 reals per site
 *   ri = 0 real part, 1 imaginary part; (U v)[row] = sum_col U[row][col] v[col].
 *   real = double for DSLASH_FP64 contexts, float for DSLASH_FP32 contexts.
 *
 * Native layouts (what dslash_apply() reads and writes; sizes from dslash_*_bytes()):
 *   DSLASH_AOS                  the canonical layout itself (18 reals per link).
 *   DSLASH_AOS|DSLASH_RECON12   spinor canonical; gauge keeps rows 0,1 only:
 *                                 real[ (((s*4 + mu)*2 + row)*3 + col)*2 + ri ]
 *   DSLASH_SOA  (blocked "structure of arrays": sites are grouped in vectors of 32 consecutive site indices,
 *                v = s / 32, l = s % 32; inside a vector every component is a contiguous run of 32 elements.
 *                V is padded up to a multiple of 32 -- use dslash_*_bytes(); the padding is never read)
 *       FP64 spinor  double2[ (v*12 + k)*32 + l ]          k = spin*3 + colour = 0..11      (re, im)
 *       FP32 spinor  float4 [ (v*6  + q)*32 + l ]          q = 0..5: components k = 2q, 2q+1 (re,im,re,im)
 *       FP64 gauge   double2[ ((v*4 + mu)*R + e)*32 + l ]  e = row*3 + col; R = 9, or 6 with DSLASH_RECON12
 *       FP32 gauge   float2 [ ((v*4 + mu)*R + e)*32 + l ]
 *     A warp that handles 32 consecutive sites reads one contiguous 512-byte run per component, and all
 *     components of a site share one base address (the component stride is a compile-time constant).
 *   With DSLASH_RECON12 row 2 of every link is rebuilt in registers as conj(row0 x row1), which is
 *   exact for SU(3) input (DESIGN.md Reading R14).
 */
#ifndef DSLASH_B200_H
#define DSLASH_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dslash_ctx dslash_ctx;
typedef void *dslash_stream_t; /* a cudaStream_t */

#if defined(__GNUC__)
#define DSLASH_API __attribute__((visibility("default")))
#else
#define DSLASH_API
#endif

/* precision */
#define DSLASH_FP64 0
#define DSLASH_FP32 1
/* layout: base value, optionally OR-ed with DSLASH_RECON12 */
#define DSLASH_AOS 0
#define DSLASH_SOA 1
#define DSLASH_RECON12 16

/* status codes */
#define DSLASH_OK 0
#define DSLASH_ERR_NULL (-1)        /* a required pointer argument is NULL */
#define DSLASH_ERR_DIMS (-2)        /* an extent < 1, or the lattice exceeds the 32-bit indexing limit */
#define DSLASH_ERR_PRECISION (-3)   /* precision is not DSLASH_FP64 / DSLASH_FP32 */
#define DSLASH_ERR_LAYOUT (-4)      /* layout is not (AOS|SOA) [| RECON12] */
#define DSLASH_ERR_ALIGN (-5)       /* a field pointer is not 16-byte aligned */
#define DSLASH_ERR_ALIAS (-6)       /* out overlaps in */
#define DSLASH_ERR_UNSUPPORTED (-7) /* variant / tuning parameters outside the supported set */
#define DSLASH_ERR_CUDA (-8)        /* a CUDA runtime call failed; see dslash_last_cuda_error() */
#define DSLASH_ERR_NOMEM (-9)       /* host or device allocation failed */
#define DSLASH_ERR_TOO_LARGE (-10)  /* the field does not fit the library's built-in scratch array (dslash_eo_apply_schur_static) */

/* variant selection: collapse_depth DSLASH_VARIANT_TUNED selects the library's tuned kernel */
#define DSLASH_VARIANT_TUNED 0

/* operators of dslash_apply_op() */
#define DSLASH_OP_D 0        /* Eq. 1 */
#define DSLASH_OP_D_DAGGER 1 /* its adjoint: Eq. 1 with gamma_mu -> -gamma_mu (= gamma_5 D gamma_5) */
#define DSLASH_OP_M 2        /* Wilson matrix M = (4 + mass) - D/2 */
#define DSLASH_OP_M_DAGGER 3 /* M^dagger = (4 + mass) - D^dagger/2 */

/* schedules of the paper's offload variants, dslash_set_omp_variant() */
#define DSLASH_SCHED_STATIC 0
#define DSLASH_SCHED_DYNAMIC 1
#define DSLASH_SCHED_GUIDED 2

/* kernel selection of the tuned path, dslash_set_kernel() */
#define DSLASH_KERNEL_AUTO 0   /* the library picks: _DIRECT until dslash_tune() has measured and chosen */
#define DSLASH_KERNEL_DIRECT 1 /* one thread per site, all neighbours gathered from global memory through L1/L2 */
/* 2, 3, 4: kernels of round 1 (tile staged by bulk copies; spinor ring) that lost to the ones below and were removed */
#define DSLASH_KERNEL_WARP_PIPE 5 /* persistent warps, one 32-site x row per warp; every hop stage (neighbour spinors + links of
                                  the row: two contiguous runs in the blocked SoA layout) is brought into per-warp shared-memory
                                  slots by two bulk async copies, DSLASH_OPT_PIPE_SLOTS stages ahead, no block barriers
                                  (blocked SoA, L_X == 32); bit-identical to DSLASH_KERNEL_DIRECT */

#define DSLASH_KERNEL_MARCH 6 /* block-cooperative t-marching: a block owns up to 7 x rows that are neighbours in the (y,z) plane
                                  and marches through the time slices; every link and every spinor row of the patch crosses
                                  L2 -> SM once (links used for the own forward hop AND the neighbour's backward contribution,
                                  spinor rows kept in a shared-memory ring), all operands by bulk async copies
                                  (blocked SoA, L_X == 32); bit-identical to DSLASH_KERNEL_DIRECT */
/* (7 was DSLASH_KERNEL_GMARCH, the marching design for any L_X: built in round 2, 2.4-2.9 x slower than _DIRECT on every lattice,
   removed in round 3 -- profiles/r02b_gmarch.md, profiles/r03_fp32_path.md; dslash_set_kernel(ctx, 7) returns UNSUPPORTED) */

/* options of the tuned kernels, dslash_set_option() */
#define DSLASH_OPT_OCCUPANCY 2        /* blocks of <= 128 threads: 0 = 168 registers/thread (12 warps/SM), 1 = 128 (16 warps),
                                         2 = 255 (8 warps, deeper load hoisting) */
#define DSLASH_OPT_L2_POLICY 3        /* direct kernel: bit mask of L2 hints, -1 or 0 (default) = none: 1 spinor loads evict_last,
                                         2 U_t loads evict_last, 4 U_x/U_y/U_z loads evict_first, 8 stores of `out` evict_first,
                                         16 t-direction loads bypass L1 allocation.  The marching kernel does not read it (its
                                         bits mean other things: DSLASH_OPT_MARCH_POLICY), so a value tuned for one kernel never
                                         leaks into another and dslash_tune() compares every candidate under its own setting */
#define DSLASH_OPT_L1_CARVEOUT 4      /* direct kernel: preferred shared-memory carve-out in percent, -1 = driver default */
#define DSLASH_OPT_X_SHUFFLE 5        /* direct kernel: 1 (default for FP64; FP32 defaults to 0) = when a whole x row sits inside one warp
                                         (tile x-extent == L_X, a power of two <= 32) the two x hops are exchanged between
                                         lanes by warp shuffles instead of loaded; 0 = always load them.  Same result, bit
                                         for bit */

#define DSLASH_OPT_PIPE_SLOTS 7       /* warp-pipelined kernel: hop stages in flight per warp, 2..4 (0 = library default) */
#define DSLASH_OPT_PIPE_WARPS 8       /* warp-pipelined kernel: warps per thread block, 1, 2 or 4 (0 = library default) */
#define DSLASH_OPT_PIPE_ZBLOCK 9      /* z planes per block of the traversal order, a divisor of L_Z.  Warp-pipelined kernel: rows are
                                         visited y fastest, z inside a z block, then t, then the z blocks (0 = L_Z).  Direct kernel:
                                         tiles are numbered x, y, z inside a z block, t, z block (the value must be a multiple
                                         of the tile's z extent; 0 = automatic: no blocking while a time slice of the three
                                         fields is <= 40 MB, else the largest block whose slice is <= 20 MB).  Both shorten
                                         the L2 reuse distance of the t hops (48^3x96 fp32: HBM reads 1.26 x -> see profiles/) */
#define DSLASH_OPT_TUNE_MODE 10       /* what dslash_tune() optimises: DSLASH_TUNE_BURST (default; the first ~35 ms after idle, board at its
                                         boost clock) or DSLASH_TUNE_SUSTAINED (continuous load, board at its power-capped clock) */
#define DSLASH_OPT_MARCH_LEAD 11      /* marching kernel: steps a block may run ahead of the slowest block of its chunk, 0..16
                                         (0 = unbounded, the default: measured slower than unbounded on 32^3x64).  Blocks that
                                         stay close share their halo rows through L2.  Only single-wave plans honour it */
#define DSLASH_OPT_MARCH_POLICY 13    /* marching kernel (DSLASH_KERNEL_MARCH): bit mask           , -1 (default) = 4|8|16: 1 data other
                                         blocks read too evict_last (measured harmful), 4 links read once per application
                                         evict_first, 8 stores evict_first, 16 a ring row is fetched late, about one step before
                                         its first use instead of two.  0..31 */
#define DSLASH_TUNE_BURST 0
#define DSLASH_TUNE_SUSTAINED 1

/* host<->device mapping modes of dslash_apply_host() (section 4.1.2) */
#define DSLASH_MAP_MINIMAL 0 /* to: gauge, in;  from: out            (after the Advisor's data analysis) */
#define DSLASH_MAP_TOFROM 1  /* tofrom: gauge, in, out                (no data analysis)                  */

/*
 * Create a context for one lattice, precision and native layout on the current CUDA device.
 *   ctx        out: receives the new context (library-owned; release with dslash_destroy).
 *   dims       host pointer to {L_X, L_Y, L_Z, L_T}; every extent >= 1 (even or odd; L = 1 and 2 wrap
 *              onto the site itself / the same neighbour, as the modulo in Eq. 1's deltas says);
 *              36*V must be < 2^31 (32-bit vector indices; V <= 59 652 323 sites).
 *   precision  DSLASH_FP64 or DSLASH_FP32: storage and arithmetic type of all three fields.
 *   layout     DSLASH_AOS or DSLASH_SOA, optionally | DSLASH_RECON12.
 * The context starts with the tuned kernel selected (DSLASH_VARIANT_TUNED).
 * Errors: NULL, DIMS, PRECISION, LAYOUT, CUDA (no device), NOMEM.
 */
DSLASH_API int dslash_create(dslash_ctx **ctx, const int dims[4], int precision, int layout);

/* Free a context and any staging buffers it owns (synchronises the device if it owns any).
 * NULL is a no-op returning DSLASH_OK. */
DSLASH_API int dslash_destroy(dslash_ctx *ctx);

/*
 * out = D[gauge] in -- one application of Eq. 1, asynchronous on `stream`.
 *   out, in   device pointers, native spinor layout of the ctx, dslash_spinor_bytes() each,
 *             16-byte aligned, must not overlap.
 *   gauge     device pointer, native gauge layout, dslash_gauge_bytes(), 16-byte aligned.
 * Exactly one kernel launch (DSLASH_KERNEL_WARP_PIPE: preceded by an 8-byte cudaMemsetAsync of its row counters on
 * `stream`); no allocation, copy or synchronisation.
 * Errors: NULL, ALIGN, ALIAS, UNSUPPORTED (the current CUDA device is not the one the ctx was created on; an explicitly
 * selected kernel cannot run this lattice), CUDA (launch failure, also stored in the ctx).
 */
DSLASH_API int dslash_apply(dslash_ctx *ctx, void *out, const void *in, const void *gauge, dslash_stream_t stream);

/* Bytes of one spinor / of the gauge field in the ctx's native layout (0 if ctx is NULL). */
DSLASH_API size_t dslash_spinor_bytes(const dslash_ctx *ctx);
DSLASH_API size_t dslash_gauge_bytes(const dslash_ctx *ctx);
/* Bytes of the same fields in the canonical layout at the ctx's precision. */
DSLASH_API size_t dslash_canonical_spinor_bytes(const dslash_ctx *ctx);
DSLASH_API size_t dslash_canonical_gauge_bytes(const dslash_ctx *ctx);

/*
 * Layout module (north_star subsystem (1)): canonical <-> native, device to device, asynchronous
 * on `stream`, one kernel launch each.  src and dst must not overlap.  pack_gauge drops row 2 when
 * the ctx has DSLASH_RECON12.  For DSLASH_AOS without RECON12 these are plain copies.
 * Errors: NULL, ALIGN, CUDA.
 */
DSLASH_API int dslash_pack_spinor(dslash_ctx *ctx, void *dst_native, const void *src_canonical, dslash_stream_t stream);
DSLASH_API int dslash_unpack_spinor(dslash_ctx *ctx, void *dst_canonical, const void *src_native, dslash_stream_t stream);
DSLASH_API int dslash_pack_gauge(dslash_ctx *ctx, void *dst_native, const void *src_canonical, dslash_stream_t stream);

/*
 * Advisor-style variant selection (section 4.1.3; BASELINE.json configs[4]).
 *   collapse_depth     DSLASH_VARIANT_TUNED (0): the tuned kernel; the other two arguments are ignored.
 *                      1..4: the first `collapse_depth` of the loops (t, z, y, x) of Code 1
 *                       are collapsed into one parallel iteration space; each parallel
 *                      iteration runs the remaining inner loops serially in one thread.
 *   threads_per_block  64, 128, 256, 512 or 1024.
 *   sites_per_thread   1, 2 or 4 parallel iterations per thread, block-cyclic:
 *                      iteration = (blockIdx*S + k)*threads_per_block + threadIdx, k = 0..S-1.
 * The layout axis of the sweep is the ctx's own layout (create one ctx per layout).
 * Errors: NULL, UNSUPPORTED.
 */
DSLASH_API int dslash_set_variant(dslash_ctx *ctx, int collapse_depth, int threads_per_block, int sites_per_thread);
DSLASH_API int dslash_get_variant(const dslash_ctx *ctx, int *collapse_depth, int *threads_per_block, int *sites_per_thread);

/* Enumeration of the sweep space of BASELINE.json configs[4]: 4 x 5 x 3 x 2 = 120 variants.
 * dslash_variant_at(i, ...) writes variant i (0 <= i < dslash_variant_count()); layout is
 * DSLASH_AOS or DSLASH_SOA.  Order: layout slowest, then collapse depth, threads/block, sites/thread.
 * Errors: NULL, UNSUPPORTED (index out of range). */
DSLASH_API int dslash_variant_count(void);
DSLASH_API int dslash_variant_at(int index, int *collapse_depth, int *threads_per_block, int *sites_per_thread, int *layout);

/*
 * The paper's own variant space (section 4.1.3, Table 1).  For num_loops nested loops (1..4) a
 * variant is (parallel_position x, distribute_collapse a, parallel_collapse b, schedule, map_mode):
 *   x in 0..num_loops-1;  a = 0 if x == 0 (combined `teams distribute parallel for`), else 1 <= a <= x;
 *   1 <= b <= num_loops - x;  schedule in DSLASH_SCHED_*;  map_mode in DSLASH_MAP_* (the two host<->device
 *   data-transfer modes; it only matters to dslash_apply_host).
 * dslash_omp_variant_count(num_loops) = 6, 18, 42, 84 for 1..4 loops (Table 1; 0 for any other num_loops);
 * dslash_omp_variant_at enumerates them (order: x, then a, then b, then schedule, then map_mode fastest).
 * dslash_set_omp_variant selects the CUDA analogue of one loop structure for dslash_apply on the four Dslash loops
 * (t,z,y,x): a team is a thread block of team_size threads (32..256, multiple of 32), the league has num_teams blocks
 * (clamped to the distribute space; 0 = 4 per SM).  dslash_set_variant(ctx, DSLASH_VARIANT_TUNED, 0, 0) leaves it.
 * Errors: NULL, UNSUPPORTED (outside the space above).
 */
DSLASH_API int dslash_omp_variant_count(int num_loops);
DSLASH_API int dslash_omp_variant_at(int num_loops, int index, int *parallel_position, int *distribute_collapse,
                                     int *parallel_collapse, int *schedule, int *map_mode);
DSLASH_API int dslash_set_omp_variant(dslash_ctx *ctx, int parallel_position, int distribute_collapse, int parallel_collapse,
                                      int schedule, int num_teams, int team_size);

/*
 * Tuning of the tuned kernel: the thread block covers a tile of tile[0] x tile[1] x tile[2] x tile[3]
 * sites (x, y, z, t); each extent a power of two, product in {32, 64, ..., 1024}.  Lattice extents
 * need not be multiples of the tile (edge threads idle).  Errors: NULL, UNSUPPORTED.
 */
DSLASH_API int dslash_set_tile(dslash_ctx *ctx, const int tile[4]);
DSLASH_API int dslash_get_tile(const dslash_ctx *ctx, int tile[4]);

/*
 * Restrict dslash_apply / dslash_apply_op to the time slices t_begin <= t < t_end (default: the whole lattice); sites
 * outside the range are neither computed nor written (what dslash_apply_host and the dslash_slab_* calls use internally).
 * Every tuned kernel honours the range (the marching kernel's block plan is rebuilt by this call: synchronous); the sweep
 * variants and dslash_cg_solve need the full range (DSLASH_ERR_UNSUPPORTED otherwise).
 * Errors: NULL, UNSUPPORTED (not 0 <= t_begin < t_end <= L_T), CUDA.
 */
DSLASH_API int dslash_set_time_range(dslash_ctx *ctx, int t_begin, int t_end);
DSLASH_API int dslash_get_time_range(const dslash_ctx *ctx, int *t_begin, int *t_end);

/*
 * Choose the implementation behind DSLASH_VARIANT_TUNED: DSLASH_KERNEL_AUTO (default: _DIRECT until dslash_tune() has
 * picked one), _DIRECT, _WARP_PIPE or _MARCH (eligibility: see their definitions above).  The call also creates the
 * device-side resources the kernel needs besides the caller's fields (row counters of _WARP_PIPE, block plan of _MARCH:
 * one small cudaMalloc + cudaMemcpy, synchronous), so that dslash_apply itself never allocates, copies or synchronises.
 * If a kernel is selected explicitly and the lattice/layout do not allow it, dslash_apply returns DSLASH_ERR_UNSUPPORTED.
 * dslash_get_kernel reports the kernel the next dslash_apply would launch.  All kernels give bit-identical results.
 * Errors: NULL, UNSUPPORTED (unknown value; the ctx's device is not the current one), NOMEM, CUDA.
 */
DSLASH_API int dslash_set_kernel(dslash_ctx *ctx, int kernel);
DSLASH_API int dslash_get_kernel(const dslash_ctx *ctx, int *kernel);

/*
 * Host-side view of the work decomposition of DSLASH_KERNEL_MARCH (no device needed; what dslash_set_kernel uploads).
 * The rows of the (y,z) plane are ordered along a snake (strips of two z planes, boustrophedon in y) and cut into S
 * segments of at most 7 rows; the time slices t_begin <= t < t_end into G chunks; block c*S + s marches segment s through
 * chunk c.  S and G are chosen so that S*G fills whole waves of `wave` co-resident blocks (the SM count).
 *   dims      {32, L_Y, L_Z, L_T} (L_X must be 32);  ints: host array receiving, per block, 4 + 7*9 ints:
 *             {t0, nt, active warps, 0} then per warp {row, fwd[2], wr[2], rd[2], bwd[2]} (MarchWarpPlan in
 *             csrc/dslash_kernels.cuh); ints may be NULL to query *nblocks only; capacity_ints = its size in ints.
 * Errors: NULL, DIMS, UNSUPPORTED (L_X != 32, bad range, wave < 1, capacity too small).
 */
DSLASH_API int dslash_march_plan(const int dims[4], int t_begin, int t_end, int wave, int *ints, size_t capacity_ints, int *nblocks);

/*
 * Pick the kernel by measurement (the Advisor's own method, applied to the library's kernels): every kernel
 * that can run this context (DSLASH_KERNEL_DIRECT; where eligible DSLASH_KERNEL_MARCH and DSLASH_KERNEL_WARP_PIPE in
 * three slot/warp configurations) is timed on the caller's buffers
 * (2 warm-up + 8 timed applications each, CUDA events on `stream`; about 15 ms in all, so that every candidate is
 * timed inside the board's boost window -- call it on an idle device; with DSLASH_OPT_TUNE_MODE = DSLASH_TUNE_SUSTAINED:
 * every candidate runs 300 applications to reach its own power-capped steady state, then 100 timed ones, ~0.8 s in all) and the fastest
 * (DSLASH_KERNEL_MARCH if it is within 1 % of the fastest: it moves the fewest on-chip bytes and keeps its time under load) becomes the
 * context's kernel, as if set by dslash_set_kernel() (and DSLASH_OPT_PIPE_SLOTS / _WARPS).  out, in, gauge: device pointers as for dslash_apply(); out is left
 * holding D in.  *chosen (may be NULL) receives the kernel, *ms_per_apply (may be NULL) its time.  This call SYNCHRONISES
 * with `stream`.  Errors: those of dslash_apply(); DSLASH_ERR_UNSUPPORTED when a sweep variant is selected.
 */
DSLASH_API int dslash_tune(dslash_ctx *ctx, void *out, const void *in, const void *gauge, dslash_stream_t stream, int *chosen,
                           float *ms_per_apply);

/* Measurement aids that are not part of the operator (dslash_probe_launch, dslash_march_stats): include/dslash_b200_diag.h */

/*
 * The operators a caller of Dslash needs next (the paper: D is the "unpreconditioned Dirac operator", and
 * "is called several times throughout the LQCD application").
 * dslash_apply_op: out = OP in with OP one of DSLASH_OP_* (mass is used by _M and _M_DAGGER only); same buffers, layouts,
 *   alignment and aliasing rules as dslash_apply; one kernel launch on `stream`; uses the ctx's tile (<= 128 sites; a
 *   larger tile returns DSLASH_ERR_UNSUPPORTED), ignores the variant/kernel selection.
 * dslash_cg_solve: conjugate gradient on the normal equations M^dagger M x = b, started from x = 0, stopped when
 *   |r| / |b| <= tol or after max_iter iterations.  x, b: device spinors in the native layout (x is overwritten, b is
 *   not modified); the ctx owns four work spinors (allocated on first use).  Reductions are two-pass fp64 sums
 *   (deterministic).  The call synchronises `stream` (it reads the residual every iteration).  iterations / rel_residual
 *   (optional, may be NULL) receive the iteration count and the final |r|/|b| of the recurrence.
 *   Returns DSLASH_OK also when max_iter was reached without convergence (check rel_residual).
 * Errors: NULL, ALIGN, ALIAS, UNSUPPORTED (op, tile, tol <= 0, max_iter < 1), NOMEM, CUDA.
 */
DSLASH_API int dslash_apply_op(dslash_ctx *ctx, int op, double mass, void *out, const void *in, const void *gauge,
                               dslash_stream_t stream);
DSLASH_API int dslash_cg_solve(dslash_ctx *ctx, void *x, const void *b, const void *gauge, double mass, double tol, int max_iter,
                               int *iterations, double *rel_residual, dslash_stream_t stream);

/*
 * Even-odd (checkerboarded) form of Eq. 1 (PAPER.md:52 calls Eq. 1 the
 * "unpreconditioned" operator -- this is the preconditioned one).  Requires every extent to be even: then Eq. 1 couples
 * a site only to sites of the other parity, parity(x) = (x+y+z+t) mod 2, 0 = even, and
 *     D_{p,1-p} = P_p D P_{1-p}                           (P_p = projector on the sites of parity p)
 *     Mhat = (4+mass) - D_eo D_oe / (4 (4+mass))          (Schur complement of M = (4+mass) - D/2 on the even sites)
 * Solving M x = b then reduces to  Mhat x_e = b_e + D_eo b_o / (2 (4+mass)),  x_o = (b_o + D_oe x_e / 2) / (4+mass).
 *
 * Checkerboard layout: the site s of parity p has the half-index h = s >> 1 (L_X is even), s = 2h + ((p+y+z+t) & 1).
 *   half-lattice spinor   a native spinor field (the ctx's AoS or blocked-SoA formulas) over the V/2 "sites" h of one parity;
 *                         dslash_eo_spinor_bytes() bytes.
 *   checkerboarded gauge  two native gauge fields over h, the links U_mu(s) of the even sites first, then (at byte offset
 *                         dslash_eo_gauge_bytes()/2) those of the odd sites; rows 0,1 only with DSLASH_RECON12.
 * dslash_eo_pack_spinor / _unpack_spinor / _pack_gauge convert from / to the canonical full-lattice arrays (device
 * pointers; unpack writes only the sites of `parity` and leaves the others untouched).
 *
 * dslash_eo_apply        out = D_{p,1-p} in (dagger = 1: D^dagger), p = out_parity; `in` lives on parity 1-p.
 * dslash_eo_apply_xpay   out = a * c + b * D_{p,1-p} in;  c = half-lattice field of parity p, only read; it must not
 *                        overlap out.
 * dslash_eo_apply_schur  out_even = Mhat in_even (dagger = 1: Mhat^dagger); tmp_odd = caller's half-lattice scratch field.
 *                        Two launches, the axpy fused into the second.
 * dslash_eo_cg_solve     conjugate gradients on Mhat^dagger Mhat x_even = b_even (same conventions, determinism and error
 *                        behaviour as dslash_cg_solve; the ctx owns five half-lattice work fields).
 * dslash_eo_solve        solves the full Wilson system M x = b through the preconditioned one: forms the right-hand side
 *                        above, runs dslash_eo_cg_solve on Mhat^dagger Mhat x_e = Mhat^dagger (.), reconstructs x_o.  x and b are
 *                        given as their even and odd halves (four distinct half-lattice fields); rel_residual is that of the
 *                        normal equations.  7 launches around the CG.
 * All asynchronous on `stream` except dslash_eo_cg_solve / dslash_eo_solve, which synchronise it.
 * Errors: NULL, DIMS (an extent is odd), UNSUPPORTED (parity/dagger not 0/1, 4+mass == 0, tol, max_iter), ALIGN,
 * ALIAS (out overlaps in; x overlaps b), NOMEM, CUDA.  dslash_eo_*_bytes return 0 when an extent is odd.
 */
DSLASH_API size_t dslash_eo_spinor_bytes(const dslash_ctx *ctx);
DSLASH_API size_t dslash_eo_gauge_bytes(const dslash_ctx *ctx);
DSLASH_API int dslash_eo_pack_spinor(dslash_ctx *ctx, void *dst_half, const void *src_canonical, int parity, dslash_stream_t stream);
DSLASH_API int dslash_eo_unpack_spinor(dslash_ctx *ctx, void *dst_canonical, const void *src_half, int parity, dslash_stream_t stream);
DSLASH_API int dslash_eo_pack_gauge(dslash_ctx *ctx, void *dst_eo, const void *src_canonical, dslash_stream_t stream);
DSLASH_API int dslash_eo_apply(dslash_ctx *ctx, int out_parity, int dagger, void *out, const void *in, const void *gauge_eo,
                               dslash_stream_t stream);
DSLASH_API int dslash_eo_apply_xpay(dslash_ctx *ctx, int out_parity, int dagger, void *out, const void *in, const void *gauge_eo,
                                    const void *c, double a, double b, dslash_stream_t stream);
DSLASH_API int dslash_eo_apply_schur(dslash_ctx *ctx, int dagger, double mass, void *out_even, const void *in_even, void *tmp_odd,
                                     const void *gauge_eo, dslash_stream_t stream);
DSLASH_API int dslash_eo_cg_solve(dslash_ctx *ctx, void *x_even, const void *b_even, const void *gauge_eo, double mass, double tol,
                                  int max_iter, int *iterations, double *rel_residual, dslash_stream_t stream);
DSLASH_API int dslash_eo_solve(dslash_ctx *ctx, void *x_even, void *x_odd, const void *b_even, const void *b_odd, const void *gauge_eo,
                               double mass, double tol, int max_iter, int *iterations, double *rel_residual, dslash_stream_t stream);

/*
 * The Schur operator for callers that must not allocate device memory.
 *
 * dslash_eo_apply_schur() needs a half-lattice scratch field from its caller, and the solvers above cudaMalloc their work
 * fields on first use.  Some users of this library can do neither once they are running:
 *   - a program that handed all of the GPU's memory to its own pool at start-up (a framework's caching allocator, a job
 *     whose lattice fields were sized to fill HBM): a cudaMalloc made on its behalf fails, or takes memory the pool counts on;
 *   - a solver loop with a latency budget: cudaMalloc and cudaFree take driver-wide locks and can wait for all work on
 *     the device, which stalls the streams the loop is trying to keep busy;
 *   - a component that is only given pointers (a plug-in under a host application's memory policy) and has no way to
 *     obtain or to own a device buffer of its own.
 * For them dslash_eo_apply_schur_static() computes the same thing,
 *     out_even = Mhat in_even,   Mhat = (4+mass) - D_eo D_oe / (4 (4+mass))      (dagger = 1: Mhat^dagger),
 * with the odd-parity intermediate D_oe in_even held in an array that is part of the library image itself
 * (`static __device__`, csrc/dslash_eo.cu).  The caller passes only the input, the output and the gauge field.  The call
 * makes no cudaMalloc / cudaFree and uses no allocating library routine; results are bit-identical to
 * dslash_eo_apply_schur() (the same two kernels run on the same data).
 *
 * Limit.  The array is DSLASH_STATIC_SCRATCH_BYTES = 8 MiB (dslash_static_scratch_bytes() returns the same number).  A
 * ctx whose half-lattice spinor, dslash_eo_spinor_bytes(), is larger is refused with DSLASH_ERR_TOO_LARGE before anything
 * is launched: in FP64 that admits 43 690 sites per parity (16^4 fits: 6.3 MB; 24^4 does not), in FP32 twice as many.  Every GPU
 * on which the library's code is loaded holds these 8 MiB from then until the process exits, used or not.
 *
 * Set-up.  The first call on each device looks the array's device address up (cudaGetSymbolAddress, with that device
 * current) and remembers it; later calls on that device only launch.  Make that first call during initialisation, before
 * any stream capture is begun.  The ctx must belong to the current device (DSLASH_ERR_UNSUPPORTED otherwise).
 *
 * Sharing.  There is ONE array per device, shared by every ctx, stream and host thread in the process, and it keeps
 * whatever the last call left in it.  Nothing in it has to start at zero -- the first kernel writes every element the
 * second one reads -- so no clearing is done.  But two calls whose kernels can run at the same time on one GPU (different
 * streams without an ordering between them, two host threads) overwrite each other's intermediate and both results are
 * garbage: order such calls yourself (one stream, or events), or use dslash_eo_apply_schur() with separate scratch fields.
 *
 * Arguments as for dslash_eo_apply_schur() without tmp_odd: device pointers, 16-byte aligned, out_even must not overlap
 * in_even; asynchronous on `stream`; two launches.  Errors: NULL, DIMS (an extent is odd), UNSUPPORTED (dagger not 0/1,
 * 4+mass == 0, ctx of another device), TOO_LARGE, ALIGN, ALIAS, CUDA (including a failed address look-up).
 */
#define DSLASH_STATIC_SCRATCH_BYTES (8u << 20)
DSLASH_API size_t dslash_static_scratch_bytes(void);
DSLASH_API int dslash_eo_apply_schur_static(dslash_ctx *ctx, int dagger, double mass, void *out_even, const void *in_even,
                                            const void *gauge_eo, dslash_stream_t stream);

/*
 * Multi-GPU form of Eq. 1 by T-slab decomposition (the paper's future work).
 * A rank owns lt consecutive time slices of the global lattice; its ctx is created with dims {L_X, L_Y, L_Z, lt} and its fields
 * are ordinary native fields of that local lattice (no ghost slices; links never travel).  Of the eight hops only two leave
 * the slab, and both projectors (1 -+ gamma_t) have rank 2, so one application exchanges two FACES of half-spinors
 * (6 complex numbers per site of a time slice, dslash_slab_face_bytes() each: 3.1 MB at 32^3 FP64):
 *     face DOWN, to the rank that owns the slices below:  P^-_t in(x, 0)                         (receiver multiplies by ITS U_t)
 *     face UP,   to the rank that owns the slices above:  U_t(x, lt-1)^dagger P^+_t in(x, lt-1)  (complete contribution)
 * One application on every rank:
 *     dslash_slab_pack_faces(ctx, face_down, face_up, in, gauge, s)       one launch; then post the two sends / two receives
 *     dslash_slab_interior(ctx, out, in, gauge, s)                        slices 1 .. lt-2 while the faces travel (no launch if lt <= 2)
 *     dslash_slab_boundary(ctx, out, in, gauge, face_from_below, face_from_above, s)    slices 0 and lt-1, after the receives
 * face_from_below is the face UP of the rank below, face_from_above the face DOWN of the rank above (with one rank: the
 * rank's own faces -- the periodic wrap).  Together the three calls write every site of `out` once, with the arithmetic
 * and the order of the sum of dslash_apply: bit-identical to the single-GPU result on the global lattice.
 * All pointers: device memory, 16-byte aligned; faces are opaque (same ctx parameters on sender and receiver); out must not
 * overlap in or the received faces.  Asynchronous on `stream`; the caller orders the message passing against it.
 * Errors: NULL, ALIGN, ALIAS, UNSUPPORTED (a partial time range is set), CUDA.
 */
DSLASH_API size_t dslash_slab_face_bytes(const dslash_ctx *ctx);
DSLASH_API int dslash_slab_pack_faces(dslash_ctx *ctx, void *face_down, void *face_up, const void *in, const void *gauge,
                                      dslash_stream_t stream);
DSLASH_API int dslash_slab_interior(dslash_ctx *ctx, void *out, const void *in, const void *gauge, dslash_stream_t stream);
DSLASH_API int dslash_slab_boundary(dslash_ctx *ctx, void *out, const void *in, const void *gauge, const void *face_from_below,
                                    const void *face_from_above, dslash_stream_t stream);

/*
 * Performance options of the tuned kernels (DSLASH_OPT_*); they never change results beyond rounding order.
 * Errors: NULL, UNSUPPORTED (unknown option or value out of range).
 */
DSLASH_API int dslash_set_option(dslash_ctx *ctx, int option, int value);
DSLASH_API int dslash_get_option(const dslash_ctx *ctx, int option, int *value);

/*
 * End-to-end application from HOST buffers in the canonical layout at the ctx's precision
 * (the path of PAPER.md:138-148: map to the device, run the kernel, map back):
 *   H2D copy of gauge and in -> pack -> apply -> unpack -> D2H copy of out, then `stream` is synchronised.
 *   The lattice is cut into up to 32 slabs of whole time slices and the three phases run on three internal streams (ordered
 *   after the caller's earlier work on `stream`): slab k+1 travels to the device while slab k is packed, applied (direct
 *   kernel on the slab's time range) and unpacked and slab k-1 of `out` travels back, so both directions of the host link
 *   are busy.  Every byte crosses the link exactly once.  (A blocked-SoA lattice whose time slice is not a whole number of
 *   32-site vectors, or a ctx with a partial time range, runs as one slab.)
 *   The kernel is always the direct kernel with the ctx's tile and options: a kernel chosen by dslash_set_kernel() / dslash_tune()
 *   and a sweep variant chosen by dslash_set_variant() / dslash_set_omp_variant() are NOT used here (the call is bound by the host
 *   link, 50x slower than any of them).
 *   With DSLASH_MAP_TOFROM all three fields travel both ways (what an offload without
 *   data analysis does); with DSLASH_MAP_MINIMAL only gauge,in go to the device and only out comes back.
 *   out_host, in_host, gauge_host   host pointers (pinned memory makes the copies asynchronous and
 *   faster; pageable memory works).  DSLASH_MAP_TOFROM reads out_host and rewrites in_host/gauge_host
 *   with the identical values.
 * The ctx owns the device staging buffers, streams and events (created on first use, freed by dslash_destroy).
 * h2d_bytes / d2h_bytes (optional, may be NULL) receive the bytes copied in each direction.
 * Errors: NULL, UNSUPPORTED (map_mode; the current device is not the ctx's), NOMEM, CUDA.  After a CUDA error in mid-pipeline the
 * call waits for the copies it has already queued before it returns, so the host buffers are the caller's again on return.
 */
DSLASH_API int dslash_apply_host(dslash_ctx *ctx, void *out_host, const void *in_host, const void *gauge_host, int map_mode,
                      dslash_stream_t stream, size_t *h2d_bytes, size_t *d2h_bytes);

/* Number of kernels this ctx has launched since creation (bench.py's gpu_launches claim). */
DSLASH_API long long dslash_launch_count(const dslash_ctx *ctx);

/* The cudaError_t of the last failed CUDA call made through this ctx (0 = none). */
DSLASH_API int dslash_last_cuda_error(const dslash_ctx *ctx);

/* Static, NUL-terminated name of a status code ("DSLASH_OK", "DSLASH_ERR_ALIGN: ...", ...). */
DSLASH_API const char *dslash_error_string(int status);

/* Library version, "major.minor" as a static string. */
DSLASH_API const char *dslash_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DSLASH_B200_H */
