/*
 * liets.h -- C ABI of libliets.so: the B200-native (sm_100a CUDA) hot path of the list-indexed
 * explicit time-stepping (LIETS) QSGS generator of arxiv/paper_2602_11734.
 *
 * The calls follow the paper's statement of the problem (PAPER.md:38-39 seeding and growth,
 * :110-116 / Algorithm 3 :133-169 the list-indexed step, :122 seed spacing, Eq. (1) :126 the
 * volume-fraction dependent growth probability, :140 the stopping rule).  Readings of points
 * where the paper is silent are listed in DESIGN.md ("Readings", R1..R20).
 *
 * Conventions
 *   - Every call returns >= 0 (a status) or < 0 (an error); nothing throws or aborts across the
 *     ABI.  After an error, liets_last_error(ctx) holds a message (owned by ctx).
 *   - The library owns the ctx and, unless the caller passes one, the device workspace.  The
 *     caller owns every dst / *_out pointer.  Pointers are HOST pointers unless marked DEVICE.
 *   - All device work is enqueued on the CUDA stream given at create (a cudaStream_t passed as
 *     void*, NULL = the legacy default stream).  Calls that return a value to the host
 *     (*_out arguments, liets_grid with a host dst) synchronise that stream; the others do not.
 *   - Voxel (x, y, z) has linear index idx = x + nx*(y + ny*z); N = nx*ny*nz < 2^32.
 *   - There is no CPU fallback: without a CUDA device every call fails with LIETS_E_CUDA.
 */
#ifndef LIETS_H
#define LIETS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct liets_ctx liets_ctx;            /* opaque; owned by the library */

enum {
    LIETS_OK = 0,            /* success; for liets_generate: target solid fraction reached       */
    LIETS_FRONT_EMPTY = 1,   /* generate stopped: no solid voxel has a void neighbour (:140)      */
    LIETS_MAX_STEPS = 2,     /* generate stopped: max_steps steps done (R14)                      */
    LIETS_E_ARG = -1,        /* bad argument (dims < 1, N >= 2^32, probability outside [0,1], ..) */
    LIETS_E_STATE = -2,      /* call order: step/generate before seed; Eq.(1) law without target  */
    LIETS_E_CAPACITY = -3,   /* caller's workspace / dst buffer too small                         */
    LIETS_E_CUDA = -4        /* CUDA runtime error or no device                                   */
};

enum { LIETS_BOUNDARY_WALL = 0,          /* neighbours outside the domain are dropped                  */
       LIETS_BOUNDARY_PERIODIC = 1,      /* every coordinate wraps ("roll"), also on axes of length 1 or 2 (R5) */
       LIETS_BOUNDARY_PERIODIC_XY = 2 }; /* x and y wrap, walls in z: a slab -- and with nz = 1 the TWO-DIMENSIONAL periodic
                                            grid of Algorithm 2: the 8 in-plane directions only, because the
                                            18 directions with dz != 0 have no target.  (nz = 1 with LIETS_BOUNDARY_WALL is the
                                            2D grid of Algorithms 1 and 3, :53, :145.)                                     */
enum { LIETS_STORAGE_U8 = 0,      /* uint8 grid + explicit list of front VOXELS (uint32 indices)  */
       LIETS_STORAGE_TILE = 1,    /* bit-packed x-rows; the active set is an explicit list of front VOXELS while it
                                     is small and an explicit list of active 128x8x8 TILES afterwards, whose front
                                     voxels are re-listed in shared memory each step                               */
       LIETS_STORAGE_FULL = 2 };  /* bit-packed x-rows and NO active set: every step sweeps the full field
                                     (Algorithm 2, the paper's "vectorized QSGS"; same keyed draws, so
                                     the same grid).  Kept as the same-box comparison of :181; cost ~ N per step.      */
enum { LIETS_LAW_CONSTANT = 0, LIETS_LAW_EQ1 = 1 };
enum { LIETS_FORMAT_U8 = 0,       /* one byte per voxel in {0,1}, x fastest, N bytes              */
       LIETS_FORMAT_BITS = 1 };   /* bit idx%8 (LSB first) of byte idx/8, ceil(N/8) bytes         */

/* Bytes of DEVICE workspace liets_create needs for this grid and storage (0 if arguments bad). */
size_t liets_workspace_bytes(int nx, int ny, int nz, int storage);

/* Create a generator for an nx*ny*nz grid ("solid-void map").
 *   boundary   LIETS_BOUNDARY_*: neighbours outside the domain are dropped (:53, :145) or wrapped
 *              per coordinate (:76 "roll").
 *   storage    LIETS_STORAGE_*: internal layout of grid and front in HBM; results are identical.
 *   workspace  DEVICE pointer to >= liets_workspace_bytes() bytes, 256-byte aligned, owned by the
 *              caller and kept alive until liets_destroy; or NULL: the library allocates.
 *   cuda_stream cudaStream_t (as void*) all work is enqueued on.
 * Errors: E_ARG, E_CAPACITY (workspace_bytes too small), E_CUDA. */
int liets_create(liets_ctx** out, int nx, int ny, int nz, int boundary, int storage,
                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Reference directional growth probabilities G_ref of the 6 face, 12 edge and 8 corner
 * directions ("directional growth probability"; R1) and the law that turns them into
 * the per-step probability: LIETS_LAW_CONSTANT (G = G_ref) or LIETS_LAW_EQ1 (Eq. (1), :126:
 * G = G_ref (phi_s - 0.95 phi_a) / (0.05 phi_s), evaluated once per step from the solid count at
 * the start of the step, as exact integer thresholds; R6, R8).  Default: all 0, Eq. (1). */
int liets_set_growth(liets_ctx* ctx, double g_face, double g_edge, double g_corner, int law);

/* Seeding: voxel v is a candidate core iff its keyed draw < core_prob; then seed
 * spacing (:122, :131 diamond dilation): candidates are scanned in ascending index and accepted
 * iff no accepted seed lies at L1 distance < spacing_s (torus metric if periodic; spacing_s <= 1
 * accepts all; R11, R12) -- reproduced exactly by parallel rounds.  Resets the grid, the front
 * (A_0 = seeds) and the step counter t = 0.  *n_seeds_out (may be NULL) = number of seeds. */
int liets_seed(liets_ctx* ctx, double core_prob, int spacing_s, uint64_t rng_seed,
               uint64_t* n_seeds_out);

/* Same reset, but the seeds are the n given voxel indices (HOST array, duplicates allowed).  The indices are
 * staged in the library's seeding scratch: n <= max(8, N/2), else E_CAPACITY; an index >= N is E_ARG. */
int liets_seed_explicit(liets_ctx* ctx, const uint64_t* idx, uint64_t n, uint64_t rng_seed);

/* Multi-phase growth, independent phases (PAPER.md:40 step 4: "The remaining phases are generated on the still unassigned
 * cells ... its cores are placed and grown in the same way as for the first phase, using its own core probability and
 * growth probabilities"): hand over the cells the phases grown before have taken.  mask: N bytes, non-zero = taken
 * (LIETS_FORMAT_U8) or ceil(N/8) bytes, bit idx%8 of byte idx/8 (LIETS_FORMAT_BITS) -- what liets_grid writes, so one
 * phase's output is the next phase's input; HOST or DEVICE memory (mask_is_device); the library keeps a copy.  Those cells
 * are NOT VOID (never cores, never claimed, and they close a front voxel's neighbourhood like solid cells) and NOT OF THIS
 * PHASE (never sources, not counted in n_solid, not in liets_grid's output; liets_s2 counts the cells no phase has taken).
 * The target fraction stays a fraction of all N cells.  mask = NULL clears.  Takes effect at the next liets_seed /
 * liets_seed_explicit (E_STATE from step / generate / grid until then).  A front that dies inside an enclosure of taken
 * cells may be found empty one (claim-less) step after the serial algorithm would: status and grid are the same.
 * Phase-interaction probabilities I_i^{n,m} (growth of a phase ON the surface of another): liets_set_interaction.
 * Errors: E_ARG (format), E_CAPACITY (mask_bytes), E_CUDA.  Synchronises. */
int liets_set_blocked(liets_ctx* ctx, const void* mask, size_t mask_bytes, int format, int mask_is_device);

/* Interacting phases (PAPER.md:40 step 4; R20): the phase being grown also grows at its interface with the
 * phases handed over by liets_set_blocked -- a still unassigned cell q = p + e_d next to a cell p of an earlier phase is
 * taken with the phase-interaction probability I of d's class (face, edge, corner; constant over the run, the same keyed
 * draw of (p, t, d) compared with I instead of G).  The cells of the earlier phases that have a void neighbour are sources
 * beside the phase's own front; they keep their cells.  0, 0, 0 (the default) switches it off: independent phases (R18).
 * Bit-row storages only (E_ARG for LIETS_STORAGE_U8); liets_generate_batch refuses such a grid (E_ARG).  Seed again afterwards (E_STATE until
 * then); a run with interaction keeps its active set as tiles from the first step. */
int liets_set_interaction(liets_ctx* ctx, double i_face, double i_edge, double i_corner);

/* Target solid volume fraction phi_s in (0,1]: n_t = ceil(phi_s*N) (R7). Used by Eq. (1) and by
 * the stopping rule. */
int liets_set_target(liets_ctx* ctx, double target_solid_fraction);

/* Exactly one growth step t -> t+1 (Algorithm 3 lines 4-15), regardless of the
 * target: every front voxel p tries each of its 26 neighbours q = p + e_d that is void at the
 * start of the step; q becomes solid iff draw(rng_seed, t, p, d) < T_class(d).  Outputs (may be
 * NULL): solid count after the step; *n_front_out = size of the front the library holds, normative
 * only as zero (no solid voxel has a void neighbour) / non-zero.  Errors: E_STATE. */
int liets_step(liets_ctx* ctx, uint64_t* n_solid_out, uint64_t* n_front_out);

/* set_target + "while phi_a < phi_s and A not empty" + at most max_steps steps,
 * the loop running on the device (one CUDA graph with a WHILE node: growth kernel + control step per
 * iteration) with no host involvement until it ends.  Bit-exactly equal to repeated liets_step.  The fraction is tested between whole steps only.  Returns LIETS_OK /
 * LIETS_FRONT_EMPTY / LIETS_MAX_STEPS; *steps_out = steps done by this call. */
int liets_generate(liets_ctx* ctx, double target_solid_fraction, uint32_t max_steps,
                   uint32_t* steps_out, uint64_t* n_solid_out);

/* Copy the phase array out: dst (HOST, or DEVICE if dst_is_device) in LIETS_FORMAT_*.
 * Errors: E_STATE before the first liets_seed / liets_seed_explicit, E_CAPACITY (dst_bytes), E_ARG. */
int liets_grid(liets_ctx* ctx, void* dst, size_t dst_bytes, int format, int dst_is_device);

/* ---- Batched realisations ----------------------------------------------------------------------
 * The paper's use of the generator is a sweep: "five independent realizations ... for each value of s",
 * fifteen porosities (:217).  A batch is n <= 16 equally shaped LIETS_STORAGE_TILE generators on one stream whose step
 * loops run as ONE device-side loop: each iteration is one launch of the tile kernel over the tile lists of ALL grids (a
 * CTA that finds one grid's list used up moves on to the next grid) and one control step per grid; the loop ends when
 * every grid has stopped.  Small grids, whose few tiles cannot fill the GPU and whose steps are bound by launch latency,
 * share both.  Every grid's result is exactly that of its own liets_generate (draws are keyed per grid by its rng_seed).
 *
 * liets_create_batch: workspace = DEVICE memory of n * liets_workspace_bytes(.., LIETS_STORAGE_TILE) bytes, 256-byte
 *   aligned, or NULL (the library allocates).  Errors: E_ARG (n outside 1..16, bad dims), E_CAPACITY, E_CUDA.
 * liets_batch_ctx(b, i): the i-th generator, owned by the batch -- use it with liets_set_growth, liets_seed,
 *   liets_seed_explicit, liets_grid, liets_s2, liets_step_log (NOT liets_destroy); NULL if i is out of range.
 * liets_generate_batch: target_solid_fraction = HOST array of n; status_out / steps_out / n_solid_out = HOST arrays of n
 *   (may be NULL): per grid what liets_generate returns and reports; device_ms_out (may be NULL) = device time of the
 *   whole call.  Returns LIETS_OK or an error (E_ARG, E_STATE if a grid is not seeded, E_CUDA); synchronises. */
typedef struct liets_batch liets_batch;
int liets_create_batch(liets_batch** out, int n, int nx, int ny, int nz, int boundary, void* workspace, size_t workspace_bytes,
                       void* cuda_stream);
liets_ctx* liets_batch_ctx(liets_batch* batch, int i);
int liets_generate_batch(liets_batch* batch, const double* target_solid_fraction, uint32_t max_steps, int* status_out,
                         uint32_t* steps_out, uint64_t* n_solid_out, float* device_ms_out);
void liets_destroy_batch(liets_batch* batch);
const char* liets_batch_last_error(const liets_batch* batch);

/* Two-point correlation of the VOID phase of the current grid along one axis (0 = x, 1 = y, 2 = z), as exact integer
 * pair counts (R16; BASELINE.json asks for it, the paper does not define it): for r = 0 .. rmax,
 *   pairs[r] = #{ x : void(x) and void(x + r e_axis) },   valid[r] = #{ x : the pair (x, x + r e_axis) is counted },
 * with pairs inside the domain only on a walled grid and wrapped per coordinate on a periodic one; S2(r) = pairs / valid,
 * S2(0) = porosity.  pairs and valid are HOST arrays of rmax + 1 entries, rmax <= 65534.  Computed on the device from
 * the bit rows; synchronises.  Errors: E_ARG, E_STATE before the first seed, E_CUDA. */
int liets_s2(liets_ctx* ctx, int axis, int rmax, uint64_t* pairs, uint64_t* valid);

/* liets_s2 for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it):
 * the same pair counts (R16), same arguments and outputs, but the per-lag counters that liets_s2 takes from
 * cudaMalloc on every call sit in one file-scope device array of LIETS_S2_STATIC_MAX_LAGS 64-bit counters (32 KiB; every
 * GPU that loads the library holds it until the process exits).  The call makes no cudaMalloc, cudaFree or allocating
 * library call.  Limits: rmax + 1 <= LIETS_S2_STATIC_MAX_LAGS, else LIETS_E_CAPACITY; bit-row storages only
 * (LIETS_STORAGE_TILE, LIETS_STORAGE_FULL; a STORAGE_U8 grid would need N/8 bytes of packing scratch: LIETS_E_ARG).
 * The ctx's device must be current.  All calls on a device share the array, which keeps the last call's counts: every
 * call zeroes the counters it uses first.  Calls that overlap on the GPU would race on it; this entry point holds a
 * host mutex and synchronises the ctx's stream before it returns, so its own calls never overlap within a process.
 * pairs and valid are HOST arrays of rmax + 1 entries.  Errors: E_ARG, E_CAPACITY, E_STATE before the first seed, E_CUDA. */
#define LIETS_S2_STATIC_MAX_LAGS 4096
int liets_s2_static(liets_ctx* ctx, int axis, int rmax, uint64_t* pairs, uint64_t* valid);

/* Per-step counters of the steps done since the last seed (HOST arrays of capacity cap, may be
 * NULL): front size at the start of step i (list entries: voxels for STORAGE_U8; for STORAGE_TILE voxels while the
 * front is a voxel list, tiles afterwards -- bit 63 set: the step ran on the tile list; bit 62 set as well: it was
 * the hand-over step and the count is still the voxel list's), solid count after it, the number of Philox4x32-10 blocks the step evaluated
 * (one per front voxel with a void target, plus one per further nibble level of its tied directions),
 * and the number of front voxels with a void target (the sources of Algorithm 3 that made attempts).
 * Returns the number of steps recorded (<= 4096 kept). */
int liets_step_log(liets_ctx* ctx, uint64_t* front_in, uint64_t* solid_after, uint64_t* philox_blocks,
                   uint64_t* front_voxels, uint32_t cap);

/* Device time in milliseconds of the last liets_seed and the last liets_generate (CUDA events on
 * the ctx stream). */
int liets_timings(liets_ctx* ctx, float* seed_ms, float* generate_ms);

/* Profiling aid for the roofline report: when on, liets_generate / liets_step bracket every
 * growth-kernel launch with a CUDA event pair (at most 4096 kept per call). */
int liets_set_profiling(liets_ctx* ctx, int on);
/* Device time in milliseconds of each growth-kernel launch of the last liets_generate / liets_step
 * made with profiling on (HOST array of capacity cap). Returns the number of launches recorded. */
int liets_step_times(liets_ctx* ctx, float* ms, uint32_t cap);
/* Number of kernels this ctx has launched since liets_create (memsets and copies not counted). */
uint64_t liets_launch_count(const liets_ctx* ctx);

/* Variants of the spacing filter of liets_seed, used from the next liets_seed on.
 * order  LIETS_ORDER_INDEX (default): candidates are tried in ascending linear index (R12).
 *        LIETS_ORDER_KEYED: in ascending (key, index), key(v) = word v % 4 of Philox4x32-10 at counter
 *        (v / 4, 0, 1, 2^32 - 1) under the rng_seed's key: a random order fixed by the seed (R19; the paper does not say
 *        in which order cores are tried).  Another maximal set of seeds at pairwise L1 >= s; the
 *        dependency chains are a handful of rounds long instead of a sweep through the grid.
 * method LIETS_SPACING_SPARSE (default): works on the list of candidates.
 *        LIETS_SPACING_DENSE: the paper's mechanism (Fig. 1(D), "a small kernel but multiple iterations"):
 *        every round dilates bit planes of the WHOLE grid by s-1 passes of the 6-neighbour kernel.  Same seeds as the
 *        default (index order); LIETS_BOUNDARY_WALL only; kept as the same-box comparison for the paper's "seed spacing
 *        halves the generation rate" (:189).  liets_seed then synchronises once per round and may return E_CAPACITY when
 *        the candidate list and 8 bit planes (ceil(nx/64) * 8 * ny * nz bytes each) exceed the 4 N bytes of seeding scratch.
 * Errors: E_ARG (unknown value, DENSE with KEYED, DENSE on a periodic grid). */
enum { LIETS_ORDER_INDEX = 0, LIETS_ORDER_KEYED = 1 };
enum { LIETS_SPACING_SPARSE = 0, LIETS_SPACING_DENSE = 1 };
int liets_set_spacing(liets_ctx* ctx, int order, int method);
/* After liets_seed: rounds the keyed-order or dense-dilation spacing took (0 for the default path).  Errors: E_STATE. */
int liets_spacing_rounds(liets_ctx* ctx, uint32_t* rounds);

/* After liets_seed: the number of keyed candidates before spacing, and whether the spacing was
 * resolved by the rescan slow path (1) or by the adjacency lists (0); both may be NULL.  Errors: E_STATE. */
int liets_seed_info(liets_ctx* ctx, uint32_t* n_candidates, uint32_t* slow_path);
/* Test aid: shrink the status ring (a power of two in [2048, 2^17]) and the head table (<= 2^16) of the
 * single-CTA spacing resolve so that small grids exercise the ring wrap; ring = 0 restores the defaults.
 * The accepted seeds never depend on these sizes. */
int liets_debug_spacing_ring(liets_ctx* ctx, uint32_t ring, uint32_t head);
/* Test aid: the device's evaluation of Eq. (1) in counts (R6/R8),
 *   T = min(2^32, floor(R max(0, 20 n_t - 19 n_solid) / n_t)),
 * for n triples given as HOST arrays (R <= 2^32, 1 <= n_t <= 2^32, n_solid <= 2^32); T_out is a HOST array of n.
 * It runs the same device function the control step uses (no 128-bit arithmetic on the device), on the default
 * stream, and synchronises.  Errors: E_ARG, E_CUDA. */
int liets_debug_thresholds(const uint64_t* R, const uint64_t* n_t, const uint64_t* n_solid, uint64_t* T_out, uint32_t n);
/* Test / tuning aid (STORAGE_TILE; a no-op for STORAGE_U8): the active set is kept as a list of front VOXELS while it
 * is small ("the very early stages of growth") and as a list of tiles afterwards; a step that starts
 * with more than max_front_voxels front voxels, or whose list did not fit `capacity` entries, runs on tiles, and so do
 * all later ones.  max_front_voxels: 0 = tiles from the first step; UINT64_MAX = the default (max(N/128, 2^17), at most
 * half the capacity); larger values are clamped to the capacity.  capacity: 0 = the allocated max(2^18, N/16) entries,
 * smaller values shrink the list (so that small grids exercise the overflow hand-over).  The grid never depends on
 * either value.  Takes effect from the next step; call it before liets_seed for a whole run. */
int liets_debug_vox_list(liets_ctx* ctx, uint64_t max_front_voxels, uint32_t capacity);

/* Measured roofs for the roofline report (SURVEY.md 8(d) "Which roofline": the working set of the growth steps
 * is L2 resident and Philox makes the integer pipes a co-limit).  Runs probe `kind` `reps`
 * times (after one warm-up launch) on cuda_stream, timed with CUDA events, and returns the best launch:
 *   LIETS_PROBE_PHILOX   Philox4x32-10 blocks per second, nothing but the blocks
 *   LIETS_PROBE_LOP3 / _IMAD / _MIX  thread-level integer instructions per second: three-input logic ops (ALU
 *                        pipe), 32-bit multiply-adds (FMA pipe), and the two interleaved one to one
 *   LIETS_PROBE_L2_READ  bytes per second of 16-byte ld.global.cg loads over an L2-resident 32 MiB window
 *   LIETS_PROBE_HBM_READ bytes per second of the same loads over the whole scratch (make it >> L2)
 * device_scratch: DEVICE buffer of scratch_bytes >= 1 MiB, caller-owned (contents are read, 4 KiB may be
 * overwritten).  *ms_best (may be NULL) = duration of the best launch.  Needs no ctx.  Errors: E_ARG, E_CUDA. */
enum { LIETS_PROBE_PHILOX = 0, LIETS_PROBE_LOP3 = 1, LIETS_PROBE_IMAD = 2, LIETS_PROBE_MIX = 3,
       LIETS_PROBE_L2_READ = 4, LIETS_PROBE_HBM_READ = 5 };
int liets_probe(int kind, void* device_scratch, size_t scratch_bytes, void* cuda_stream, int reps,
                double* units_per_second, double* ms_best);

void liets_destroy(liets_ctx* ctx);
const char* liets_last_error(const liets_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif
