/*
 * ent.h -- C ABI of the B200-native particle hot path of arXiv 2511.17710 ("Entity", curvilinear
 *          special-relativistic PIC module).  P:nnn = line nnn of the paper text.
 *
 * The library runs sub-steps 3-8 of the paper's time step for one particle species:
 *   gather E,B at the particle -> code basis to global Cartesian basis
 *   -> relativistic Boris push (Eq. 3) -> move + back-map to code coordinates with
 *   cell-crossing bookkeeping -> charge-conserving conformal-current deposit
 *   (Eq. 6, "modified zig-zag" P:575), plus the cell/tile counting sort that keeps those stages
 *   memory-coherent (not in the paper; BASELINE.json north_star (e)).
 *
 * Conventions common to every call
 *   - every function returns 0 (ENT_OK) or a negative ent_status; it never throws, never exits and never
 *     synchronises the stream (except the *_host calls, ent_reserve and the counters of ent_get_stat, which say so; a call that
 *     has to grow the scratch pool because ent_reserve was not used also does).  Work is enqueued on the CUDA stream
 *     given to ent_create.  ent_last_error(ctx) returns a NUL-terminated message owned by ctx.
 *   - "device pointer" = memory allocated by the caller on the ctx's device (e.g. a torch tensor); the
 *     library never allocates or frees caller-visible memory.  All particle/field device pointers must be
 *     16-byte aligned (ENT_EINVAL otherwise).
 *   - grids: D = 2 or 3 dimensions, N[d] active cells, N_GHOST = 2 ghost layers on each side.
 *     A grid array ("padded planar array") has extents N[d] + 4, x1 fastest; active cell (i,j,k) is element
 *     (i+2) + P0*((j+2) + P1*(k+2)), P_d = N[d] + 4.  In 2D the third extent is 1 (no ghosts).
 *   - field components are contravariant code-basis components on the Yee lattice (P:181,
 *     P:1044-1053): element (i,j,k) of E1 is E^1(i+1/2,j,k), E2 (i,j+1/2,k), E3 (i,j,k+1/2),
 *     B1 (i,j+1/2,k+1/2), B2 (i+1/2,j,k+1/2), B3 (i+1/2,j+1/2,k).  Ghosts are filled by the caller.
 *   - currents are conformal currents \mathcal{J}^d = sqrt(h) J^d staggered like E, units
 *     charge * cells / time, written un-wrapped into the ghost layers (see ent_fold_current).
 *   - particles: structure of arrays, one struct per species.  Position = cell index +
 *     in-cell offset in [0,1); momentum u = gamma*v in the GLOBAL Cartesian basis, c = 1.
 */
#ifndef ENT_H
#define ENT_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ENT_NGHOST 2

typedef enum { ENT_OK = 0, ENT_EINVAL = -1, ENT_EUNSUPPORTED = -2, ENT_ECUDA = -3, ENT_ENOMEM = -4 } ent_status;
enum { ENT_CART = 0, ENT_SPH = 1, ENT_QSPH = 2 };             /* metric kind */
enum { ENT_PERIODIC = 0, ENT_ABSORB = 1, ENT_AXIS = 2 };      /* boundary rule of a dimension (both sides) */

typedef struct ent_ctx ent_ctx;                                /* opaque; owns only scratch memory */

/* Grid + metric parameters, exactly those of P:211 (Eq. 7) and P:227-267.  Host struct, passed by pointer,
 * copied by the call.  CART: cell size (xmax-xmin)/N per dimension.  SPH: r = xmin[0] + x1*dr, theta = x2*pi/N[1].
 * QSPH: r = r0 + exp(log(xmin[0]-r0) + x1*dR), theta = T + 2 vartheta T (1-2T/pi)(1-T/pi), T = x2*pi/N[1].
 * SPH/QSPH require D == 2 (axisymmetric; the particle carries phi), bc = {ABSORB, AXIS}. */
typedef struct {
    int32_t D;
    int32_t N[3];
    int32_t bc[3];
    int32_t kind;
    double  xmin[3], xmax[3];
    double  r0, vartheta;
} ent_grid;

/* Six padded planar fp32 arrays, order ex1,ex2,ex3,bx1,bx2,bx3.  Device pointers (host pointers
 * for the *_host calls).  Read-only for the library. */
typedef struct { const float *comp[6]; } ent_fields;

/* Three padded planar fp32 arrays, conformal J^1,J^2,J^3.  Device pointers.  The library ACCUMULATES into them. */
typedef struct { float *comp[3]; } ent_current;

/* One species.  n may be any value >= 0 (ragged tails are handled).
 *   cell  : int32[n]  linear ACTIVE cell index  i1 + N1*(i2 + N2*i3)   (2D: i1 + N1*i2)
 *   d[a]  : fp32[n]   in-cell offset along dimension a, 0 <= d < 1; d[2] = NULL when D == 2
 *   phi   : fp32[n]   azimuth in [0, 2 pi) for SPH/QSPH, NULL for CART
 *   u[a]  : fp32[n]   gamma*v, global Cartesian basis
 *   w     : fp32[n]   macro-particle weight (read-only for the library)
 *   tag   : uint8[n]  1 = alive, 0 = dead; NULL = all alive and no absorbing side in the grid
 *   q, m  : charge and mass of the species (q/m enters the push, q*w the deposit)
 * A particle that leaves through an ABSORB side gets tag = 0, keeps the momentum it had when
 * it left, its cell is clamped into the grid, and it deposits nothing for that step. */
typedef struct {
    int64_t  n;
    int32_t *cell;
    float   *d[3];
    float   *phi;
    float   *u[3];
    float   *w;
    uint8_t *tag;
    float    q, m;
} ent_particles;

/* ---- context -------------------------------------------------------------------------------------------
 * ent_create: device = CUDA ordinal; cuda_stream = a cudaStream_t (NULL = default stream) on which every call
 * of this ctx enqueues its work.  Fails with ENT_ECUDA when no usable CUDA device exists: there is NO CPU
 * fallback.  ent_destroy frees the ctx's scratch (synchronises the stream first). */
int ent_create(ent_ctx **out, int device, void *cuda_stream);
int ent_destroy(ent_ctx *ctx);
const char *ent_last_error(const ent_ctx *ctx);               /* never NULL; "" when no error was recorded */

/* Validates and installs the grid (D, N, bc, metric).  ENT_EINVAL: D not in {2,3}, N[d] < 3 on a periodic
 * dimension (|delta i| <= 1 would be ambiguous), N1*N2*N3 >= 2^31, xmax <= xmin, QSPH with xmin[0] <= r0 or
 * vartheta outside [0,1).  ENT_EUNSUPPORTED: SPH/QSPH with D != 2 or bc != {ABSORB, AXIS}; AXIS on a CART grid. */
int ent_set_grid(ent_ctx *ctx, const ent_grid *grid);

/* ---- the three calls of the problem statement ----------------------------------------------------------
 * ent_gather_push: sub-steps 3-7 + crossing bookkeeping for every alive
 * particle of `in`, result in `out` (same n; out may alias in array-by-array; out->w is not written).
 * u^(n-1/2) -> u^(n+1/2) with fields at n; x^(n) -> x^(n+1) with u^(n+1/2)/gamma^(n+1/2) * dt.
 * PERIODIC dimension: cell index wraps.  ABSORB: tag = 0 on leaving (needs out->tag != NULL, else ENT_EINVAL
 * at call time if the grid has an ABSORB side).  AXIS: theta stays in [0, pi] by construction. */
int ent_gather_push(ent_ctx *ctx, const ent_fields *EB, const ent_particles *in, ent_particles *out, float dt);

/* ent_deposit: sub-step 8.  For every particle alive in both blocks, adds the conformal current of
 * the move old -> new (two straight segments through the relay point of P:575; 3D per-segment weights
 * (1-W_a)(1-W_b) + D_a D_b/12, which make Eq. 6 hold to round-off) times q*w/dt to J, un-wrapped: a particle
 * that crossed a periodic face deposits into the ghost layer beyond it.  In 2D the out-of-plane J^3 is
 * q w v^3 (code basis) at n+1/2 taken from new->u, half per segment.  Requires |delta i| <= 1 per dimension
 * (violations are counted, see ENT_STAT_BAD_MOVES, and deposit nothing).  Uses old->w, old->q. */
int ent_deposit(ent_ctx *ctx, const ent_particles *old_, const ent_particles *new_, ent_current *J, float dt);

/* ent_sort: out-of-place counting sort of a species by sort key (S10).  key(cell) orders cells tile-major:
 * with tile extents T_d (ENT_STAT_TILE_1..3) and nt_d = ceil(N_d / T_d) tiles per dimension,
 *     tile  = t1 + nt1*(t2 + nt2*t3),  t_d = i_d / T_d
 *     local = l1 + T1*(l2 + T2*l3),    l_d = i_d % T_d
 *     key   = tile * (T1*T2*T3) + local          (0 <= key < ENT_STAT_NKEYS)
 * Dead particles keep their key.  On return `out` holds a permutation of `in` with non-decreasing keys
 * (order inside one cell unspecified) and, if key_offsets != NULL (device, int32[NKEYS+1]),
 * key_offsets[k] = number of particles with key < k.  in and out must not overlap; out's arrays must exist
 * wherever in's do (if only out has tags they are set to 1).  The ctx remembers `out` as "sorted" so that ent_step may take its
 * tiled path on it and ent_step_sorted accepts it.
 * Incremental form (ENT_OPT_SORT_MODE = 0, the default): when `in` is itself a block a previous ent_sort of this ctx
 * produced (same pointers and n; its particles have drifted since) and key_offsets is NULL, only tile contiguity is
 * re-established: `out` is a permutation of `in` in which tile(key) is non-decreasing; the order inside a tile is
 * unspecified (the tiled ent_step does not depend on it).  ENT_STAT_LAST_SORT_REBIN tells which form ran. */
int ent_sort(ent_ctx *ctx, const ent_particles *in, ent_particles *out, int32_t *key_offsets);

/* Copies the tile offsets the ctx keeps for a sorted block (the `out` of an ent_sort of this ctx) to tile_offsets (device,
 * int32[ENT_STAT_NTILES + 1]): tile t owns particles [tile_offsets[t], tile_offsets[t+1]) of the block.  ENT_EINVAL if the
 * block is not a sorted block of this ctx.  Enqueued on the ctx's stream. */
int ent_tile_offsets(ent_ctx *ctx, const ent_particles *block, int32_t *tile_offsets);

/* ---- fused hot path: the timed entry point ------------------------------------------------------------------
 * ent_step = ent_gather_push (in place) + ent_deposit(old, new) in one pass over the particles: the old
 * position stays in registers instead of the i_prev/dx_prev arrays of P:559.  Accumulates into J un-wrapped.
 * If `p` is the block the last ent_sort produced (same pointers and n), the tiled kernel runs: one CTA per
 * tile, E/B halo staged in shared memory by TMA, J accumulated in shared memory and flushed once; particles
 * that drifted out of their tile's halo since the sort take the global-atomic path inside the same kernel.
 * Otherwise the untiled kernel (global gathers, global atomics) runs.  Results agree up to fp32 summation order. */
int ent_step(ent_ctx *ctx, const ent_fields *EB, ent_particles *p, ent_current *J, float dt);

/* ent_step_pair = ent_step(p1) + ent_step(p2) for two species on the same grid (the pair plasma of the paper's runs) in ONE
 * launch of the tiled kernel: a CTA stages the E,B box of its tile once, advances the tile's particles of both blocks and flushes
 * one J tile (half the per-tile work and half the field / current traffic of two launches).  Both blocks must be sorted blocks of
 * this ctx on a Cartesian grid the tiled kernel supports, of at least 444 tiles (3 CTAs on each of the 148 SMs; ENT_OPT_STEP_IMPL = 3
 * lifts this), and either both or neither carry tags; otherwise the call is exactly the two ent_step calls.  A tile is not split across CTAs here: meant for plasmas whose tile populations are of one order.
 * Results agree with two ent_step calls up to fp32 summation order of J. */
int ent_step_pair(ent_ctx *ctx, const ent_fields *EB, ent_particles *p1, ent_particles *p2, ent_current *J, float dt);

/* ent_step_sorted = ent_step + the tile sort in ONE pass, out of place: every particle of `in` is advanced exactly as by
 * ent_step (accumulating into J un-wrapped) and written to `out`, in the range of the tile its cell lay in BEFORE the step.
 * `in` must be a sorted block of this ctx (the `out` of ent_sort or of a previous ent_step_sorted); `out` becomes one, ordered
 * by positions that are one step stale -- every particle lies within one cell of the tile whose range holds it, which is the
 * halo the kernel stages.  Calling it back and forth between two blocks (ping-pong) therefore never needs ent_sort again.
 * `in` is not modified; in and out must not overlap; out->tag must exist if in->tag does or the grid has an ABSORB side.
 * out->w, out->q, out->m are written.  Order of the particles inside a tile's range: unspecified.
 * Contract: between the call that produced a sorted block and the call that consumes it, the caller must not change its
 * cell / tag arrays (or must call ent_forget / ent_sort): the output layout is computed from per-tile populations recorded when
 * the block was written.  Particles that contradict it are counted in ENT_STAT_SLOT_ERRORS and dropped; particles found more
 * than one cell outside their tile take a slow global path (ENT_STAT_STRAYS) and are still placed correctly.
 * ENT_EUNSUPPORTED: SPH / QSPH grids, N1 % 4 != 0, non-default tile shapes (use ent_step + ent_sort there). */
int ent_step_sorted(ent_ctx *ctx, const ent_fields *EB, const ent_particles *in, ent_particles *out, ent_current *J, float dt);

/* ---- scratch memory ------------------------------------------------------------------------------------------
 * The ctx owns one device allocation ("pool") for sort keys, histograms, work lists and the layouts of up to 8 sorted blocks.
 * ent_workspace_bytes: size of that pool for blocks of up to npart particles on the current grid (host-side arithmetic only).
 * ent_reserve: allocates it now (may synchronise the stream).  Afterwards ent_sort / ent_step / ent_step_sorted on blocks of
 * at most npart particles never allocate and never synchronise.  Without it the pool is (re)allocated by the first call that
 * needs more, which synchronises and forgets every sorted block.  ent_set_grid releases the pool. */
int ent_workspace_bytes(ent_ctx *ctx, int64_t npart, size_t *bytes);
int ent_reserve(ent_ctx *ctx, int64_t npart);
/* The ctx recognises a sorted block by (cell pointer, n).  ent_forget drops that record: call it before re-using the memory of
 * a sorted block for something else, or after editing its cell / tag arrays (ent_gather_push does it for its `out`). */
int ent_forget(ent_ctx *ctx, const ent_particles *block);

/* J := 0 (all three padded arrays) */
int ent_zero_current(ent_ctx *ctx, ent_current *J);
/* "currents synchronization" for one periodic box: ghost layers of every PERIODIC dimension are added
 * onto the opposite active layers, then refilled with the periodic image. */
int ent_fold_current(ent_ctx *ctx, ent_current *J);

/* ---- tag sort ---------------------------------------------------------------------------------------------
 * ent_compact: out-of-place stable partition of a species by tag: the alive particles (tag != 0) come first, in their original
 * order, the dead ones after them, so that the first *n_alive records are the population and later calls may pass n = *n_alive.
 * Both blocks need tag arrays; in and out must not overlap; n_alive (may be NULL) is a DEVICE int64 written by the call.  A block
 * that was sorted stays tile-contiguous in its alive part, but the ctx forgets `out` (call ent_sort on the shortened block).
 * Scratch (12 bytes per particle) is allocated in the ctx on first use (may synchronise). */
int ent_compact(ent_ctx *ctx, const ent_particles *in, ent_particles *out, int64_t *n_alive);

/* ent_compact_static: the same operation and arguments as ent_compact for callers that cannot allocate device memory
 * (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the call makes NO cudaMalloc / cudaFree and calls
 * no allocating routine, and does not synchronise.  Its scratch (flags, positions and chunk sums of the scan, 12 bytes per particle)
 * is a static __device__ array inside the library, 12.6 MB, which every GPU that loads the library holds until the process exits;
 * its device address is looked up once per device (cudaGetSymbolAddress) when a ctx is created on that device.
 * Limit: n <= ENT_COMPACT_STATIC_MAX_N particles; a larger block is refused with ENT_EINVAL (message in ent_last_error), nothing is
 * launched.  in, out and n_alive are the caller's device memory as for ent_compact; the result is identical (bit for bit) to
 * ent_compact's.  The array is shared by EVERY call in the process on that GPU, whatever the ctx or stream, and keeps the last
 * call's contents (nothing in it has to start at zero: each call writes what it reads): two calls that overlap on the GPU race;
 * order them on one stream or with events. */
#define ENT_COMPACT_STATIC_MAX_N (1 << 20)
int ent_compact_static(ent_ctx *ctx, const ent_particles *in, ent_particles *out, int64_t *n_alive);

/* ---- step 9 of the loop: current post-processing ------------------------------------------------------------
 * ent_filter_current: `npasses` digital filter passes on the conformal currents (Eqs. 9-11: the (1/4, 1/2, 1/4)
 * kernel along every grid dimension, each component on its own staggered lattice) and then, if divide_by_sqrt_h != 0, the
 * current density J^i = conformal J^i / sqrt(h) at each component's own position.  Values beyond a component's lattice:
 * periodic image (PERIODIC); J^1 even, J^2 odd about the polar axis and J^3 = 0 on it (AXIS); zero (ABSORB).  On the
 * axis itself (sqrt(h) = 0) the conformal value is kept (Eqs. 12-13 use it).  In place; J must have been folded
 * (ent_fold_current).  Only the lattice points of each component are written (periodic dimension: 0 .. N-1; otherwise N points
 * for the component staggered along that dimension, N + 1 for the others); ghost layers keep what they held.  A second set of
 * current arrays is allocated in the ctx on first use (may synchronise). */
int ent_filter_current(ent_ctx *ctx, ent_current *J, int npasses, int divide_by_sqrt_h);

/* ---- field solver: sub-steps 2, 10, 11 of the loop --------------------------------------------------
 * Six padded planar fp32 arrays as in ent_fields, but WRITTEN by the library (device pointers, 16-byte aligned). */
typedef struct { float *comp[6]; } ent_fields_rw;

/* ent_faraday: Eq. A1: B^c -= dt / sqrt(h) * { E_b(+a) - E_b - (E_a(+b) - E_a) } at every lattice point of B^c, (c, a, b)
 * cyclic, E_i = h_ii E^i covariant, h_ii and sqrt(h) at the component's own Yee position, code coordinates in cells
 * (Delta x^i = 1).  The loop calls it twice per step with dt/2 (sub-steps 2 and 10).  Polar axis (Eq. 12): B^2 = 0 at
 * j = 0 and j = N_2, not advanced.  Only B is written, only on its lattice (periodic dimension: indices 0 .. N-1 with wrap-around
 * reads; otherwise N points for a component staggered along that dimension, N + 1 for the others); ghost layers are not touched. */
int ent_faraday(ent_ctx *ctx, ent_fields_rw *EB, float dt);

/* ent_ampere: Eq. A2: E^c += dt / sqrt(h) * { B_b - B_b(-a) - (B_a - B_a(-b)) - j_coeff * conformal J^c }.  j_coeff is the
 * 4 pi of Eq. A2 (a parameter: code units absorb it); J = the conformal currents of ent_deposit / ent_step after ent_fold_current
 * and ent_filter_current(.., divide_by_sqrt_h = 0), or NULL (vacuum).  On a non-periodic (ABSORB) face the E components tangential
 * to it are not advanced: they are the caller's boundary condition.  Polar axis: E^3 = 0 (Eq. 12); E^1 at j = 0 is advanced with the
 * integrated form, Eq. 13: E^1 += dt * { B_3(i+1/2, 1/2) - (j_coeff/2) J^1(i+1/2, 0) } / A(i+1/2), A the closed forms of
 * P:372-382, and its mirror image at j = N_2.  Only E is written, on its lattice. */
int ent_ampere(ent_ctx *ctx, ent_fields_rw *EB, const ent_current *J, float dt, float j_coeff);

/* Ghost layers of the six arrays as the gather of ent_step / ent_gather_push expects them: PERIODIC dimension: the periodic image;
 * AXIS: the mirror image about the axis, E^1 and B^1 even, the theta- and phi-components odd; ABSORB: left to the caller. */
int ent_fill_field_ghosts(ent_ctx *ctx, ent_fields_rw *EB);

/* ---- host-buffer variant (end-to-end measurement) --------------------------------------------------------------
 * Every pointer in EB, p and J is a HOST pointer (pinned memory recommended).  Copies E,B and the particle block to ctx-owned
 * device staging, zeroes the device J, sorts the block by tile (ent_sort, full form), runs `nsteps` x ent_step on the sorted
 * block (the tiled kernel where the grid supports it), copies the particle block and J back.  The block comes back PERMUTED
 * (tile-sorted order; every array alike, w included).  Synchronises the stream before returning.  *h2d_bytes / *d2h_bytes
 * (may be NULL) receive the bytes copied in each direction. */
int ent_step_host(ent_ctx *ctx, const ent_fields *EB, ent_particles *p, ent_current *J, float dt, int nsteps,
                  int64_t *h2d_bytes, int64_t *d2h_bytes);

/* The same for the two species of a pair plasma in one call, pipelined over three streams: each block is cut into eight sub-blocks
 * (consecutive quarters of its arrays) that are uploaded, sorted and advanced, and downloaded independently, so that the transfers
 * of neighbouring sub-blocks overlap the work and each other (the link is full duplex); E,B go up once, J (the sum of both species)
 * comes back once.  Every pointer is a HOST pointer (pinned memory: pageable memory serialises the copies).  Both blocks come back
 * permuted: every quarter of every array holds the same particles as before, tile-sorted.  Synchronises before returning. */
int ent_step_host_pair(ent_ctx *ctx, const ent_fields *EB, ent_particles *p1, ent_particles *p2, ent_current *J, float dt, int nsteps,
                       int64_t *h2d_bytes, int64_t *d2h_bytes);

/* ---- options and counters ----------------------------------------------------------------------------------- */
enum {
    ENT_OPT_STEP_IMPL = 1,     /* 0 = auto (tiled when the block is the sorted one), 1 = force untiled, 2 = two-kernel
                                  (gather_push to scratch copy + deposit; the paper's structure), 3 = as 0, and ent_step_pair
                                  takes its one-launch form on any grid (by default only on grids of at least 444 tiles: on a smaller
                                  one a CTA per tile cannot fill the GPU and two work-list launches are faster) */
    ENT_OPT_TILE_1 = 2, ENT_OPT_TILE_2 = 3, ENT_OPT_TILE_3 = 4,   /* tile extents in cells; takes effect at the next ent_set_grid */
    ENT_OPT_PUSHER = 7,        /* momentum update of sub-step 5: 0 = relativistic Boris (default), 1 = Vay (2008); 2 = "Boris,GCA", 3 = "Vay,GCA":
                                  the hybrid pusher of P:976-980 with the thresholds of ent_set_gca.  Takes effect at once. */
    ENT_OPT_CURV_FP64 = 6,     /* SPH / QSPH grids: 0 (default) = the move is evaluated in fp32 as a DISPLACEMENT in the local frame at the
                                  particle (increments of the code coordinates added to the in-cell offsets; same mathematics as
                                  P:147-153 + P:285-327); 1 = fp64 coordinate maps through the global Cartesian frame (the literal
                                  round trip; slower, kept for comparison).  Takes effect at once. */
    ENT_OPT_SORT_STAGING = 8,  /* 1 = the full form of ent_sort stages the records through a 32-byte-per-particle array-of-structures side buffer in
                                  the ctx (allocated on first use: may synchronise): every record is written as one full DRAM sector and unpacked
                                  by a second, coalesced pass.  For blocks that arrive in an unrelated (shuffled) order, where scattering eight
                                  4-byte arrays costs a sector read-modify-write per word; slower than the default (0) for blocks that are nearly
                                  ordered already.  Takes effect at once. */
    ENT_OPT_SORT_MODE = 5      /* 0 = auto (incremental re-bin when `in` is itself a block ent_sort produced and key_offsets is NULL),
                                  1 = always the full cell-level counting sort,
                                  2 = like 0, but the re-bin does not order the particles that stay in a tile by cell */
};
enum {
    ENT_STAT_TILE_1 = 1, ENT_STAT_TILE_2 = 2, ENT_STAT_TILE_3 = 3, ENT_STAT_NKEYS = 4, ENT_STAT_NTILES = 5,
    ENT_STAT_LAUNCHES = 6,     /* kernels launched by this ctx since creation */
    ENT_STAT_BAD_MOVES = 7,    /* particles with |delta i| > 1 seen by deposit/step (synchronises the stream) */
    ENT_STAT_STRAYS = 8,       /* particles that took the out-of-halo path in the last tiled ent_step (synchronises) */
    ENT_STAT_SCRATCH_BYTES = 9,
    ENT_STAT_LAST_STEP_TILED = 10,
    ENT_STAT_LAST_SORT_REBIN = 11,  /* 1 if the last ent_sort took the incremental re-bin path */
    ENT_STAT_SLOT_ERRORS = 12,      /* particles ent_step_sorted could not place (layout counts contradicted by the block: the caller
                                       edited the cell arrays of a sorted block without ent_forget / ent_sort); synchronises */
    ENT_STAT_CARRIES = 13,          /* since ent_create: signed wraps of a fixed-point J-tile accumulator carried into the global array
                                       (a node received > ~128 coherent contributions of the largest size); synchronises */
    ENT_STAT_GLOBAL_ADDS = 14       /* since ent_create: contributions of the axisymmetric tiled kernel too large for the tile's
                                       fixed-point range (J^3 next to the axis), added to the global array directly; synchronises */
};
int ent_set_option(ent_ctx *ctx, int key, int64_t value);
/* Thresholds of the hybrid pusher (ENT_OPT_PUSHER = 2, 3).  The paper's statement: the pusher "switches between the conventional
 * algorithm and the guiding center approximation depending on the ratio of |E|/|B| and the particle's nominal gyroradius at a given
 * timestep, rho_L ~ gamma beta m c^2 / q|B|"; "in the guiding center regime, the particle's momentum perpendicular to the local magnetic
 * field is set to zero".  Here (a reading, G26): with E, B the fields at the particle in the orthonormal basis and u the
 * momentum before the push, the regime holds when |B| > 0, |E| < e_over_b_max |B| and |u| m / (|q||B|) < rho_crit (c = 1; rho_crit in
 * the length unit of the grid's physical extent); the conventional push is then followed by u <- (u.b) b, b = B/|B|, and the move of
 * sub-step 6 is unchanged.  Defaults 0, 0 (never in the regime).  Takes effect at the next call. */
int ent_set_gca(ent_ctx *ctx, double rho_crit, double e_over_b_max);
int ent_get_stat(ent_ctx *ctx, int key, int64_t *value);

/* library version, "major.minor" */
const char *ent_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ENT_H */
