/* pic_b200.h — C ABI of the B200-native PIC particle step.
 *
 * One call = one piece of the per-supercell particle step of an electromagnetic
 * particle-in-cell code on a staggered Yee grid (§3.1 "PIConGPU";
 * the call list is BASELINE.json:north_star, the definitions SURVEY.md §8(c) steps 1-7):
 *
 *     gather E,B at x^n (CIC/TSC/PQS)  ->  relativistic Boris push  ->  move
 *     ->  charge-conserving Esirkepov deposit of J  ->  resort across supercells.
 *
 * Conventions (readings S1-S22): c = 1; u = gamma*v/c;
 * du/dt = (q/m)(E + v x B); all boundaries periodic; leapfrog time centring (the
 * loaded u is u^{n-1/2}); J is zeroed at the start of every step, so after
 * pic_step(n) it holds the current of the LAST step.
 *
 * Memory.  Every pointer is a DEVICE pointer unless the argument says "host".
 * The caller owns everything it passes.  The library owns no device memory of its
 * own: all of its state lives inside ONE caller-provided device workspace
 * (pic_workspace_bytes() -> size; allocate it e.g. as a torch uint8 tensor, 256-byte
 * aligned; hand it to pic_create; free it after pic_destroy).  All work is enqueued
 * on the cudaStream_t given to pic_create; calls that return host values
 * (pic_get_particles, pic_get_stats, pic_get_timing, pic_sync) synchronise that
 * stream, the others are asynchronous.
 *
 * Array layout.  Grid arrays (E, B, J components) are float32 of nx*ny*nz elements,
 * index i + nx*(j + ny*k), each component sampled at its Yee location
 * (SURVEY.md §8(c) step 2): Ex,Jx @ (i+1/2,j,k); Ey,Jy @ (i,j+1/2,k); Ez,Jz @ (i,j,k+1/2);
 * Bx @ (i,j+1/2,k+1/2); By @ (i+1/2,j,k+1/2); Bz @ (i+1/2,j+1/2,k).
 * Particle arrays are structure-of-arrays, one element per particle.
 *
 * Errors.  Every call returns 0 (PIC_OK) or a negative code; no exception crosses
 * the ABI.  pic_last_error(ctx) returns a static/owned human-readable string for
 * the last failing call on that context.  Faults detected on the device (frame pool
 * or exchange buffer exhausted, a particle moving >= 1 cell) set a sticky error word
 * that the next synchronising call (pic_get_*, pic_sync) reports as PIC_EDEVICE.
 */
#ifndef PIC_B200_H
#define PIC_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIC_OK        0
#define PIC_EINVAL   -1   /* bad argument (dims, order, c*dt >= cell, NULL, ...) */
#define PIC_ENOMEM   -2   /* workspace too small / capacity exceeded */
#define PIC_ECUDA    -3   /* a CUDA runtime or driver call failed */
#define PIC_ESTATE   -4   /* call out of order (step before fields / particles) */
#define PIC_EDEVICE  -5   /* sticky device-side fault, see pic_get_stats()[7] */

#define PIC_MAX_SPECIES 16

/* bits of the sticky device error word (pic_get_stats()[7]) */
#define PIC_DEV_FRAME_POOL_EXHAUSTED   1
#define PIC_DEV_EXCHANGE_OVERFLOW      2
#define PIC_DEV_TABLE_POOL_EXHAUSTED   4
#define PIC_DEV_MOVED_TOO_FAR          8
#define PIC_DEV_TMA_TIMEOUT           16
#define PIC_DEV_OVERFLOW_QUEUE_FULL   32   /* out-of-window particles exceeded the global overflow queue */
#define PIC_DEV_SORT_MISMATCH         64   /* internal: cell histogram and records disagree */
#define PIC_DEV_BAD_SPECIES          128   /* a loaded particle names a species id outside the table of pic_set_species */

typedef struct pic_ctx pic_ctx;   /* opaque, host-side */

/* Size in bytes of the device workspace pic_create needs for this geometry and
 * particle capacity.  grid[3] = cells per axis (each a multiple of supercell[a]);
 * supercell[3] = supercell extent in cells (must be {8,8,4}: the tile sizes are
 * compile-time); shape_order 1 CIC, 2 TSC, 3 PQS (S2);
 * max_particles = capacity over the life of the context.  host pointers. */
int32_t pic_workspace_bytes(const int32_t grid[3], const int32_t supercell[3],
                            int32_t shape_order, int64_t max_particles, uint64_t* bytes_out);

/* Create a context (BASELINE.json:north_star "pic_create(grid dims, cell size, dt,
 * supercell dims, shape order)").  cell[3] = cell size, dt = time step, both in units
 * with c = 1; requires dt < min(cell) so no particle moves a full cell per step
 * (SURVEY.md §8(c) step 5).  workspace = device memory of >= pic_workspace_bytes()
 * bytes, 256-byte aligned, zero-initialisation not required; stream = cudaStream_t
 * (0 = legacy default stream).  grid/cell/supercell are host pointers. */
int32_t pic_create(pic_ctx** out, const int32_t grid[3], const double cell[3], double dt,
                   const int32_t supercell[3], int32_t shape_order, int64_t max_particles,
                   void* workspace, uint64_t workspace_bytes, void* stream);

/* Species table (reading S15): charge q[s] and mass m[s], host pointers, n <=
 * PIC_MAX_SPECIES.  Until the first call every species id in [0, PIC_MAX_SPECIES) has q = -1, m = 1; after a call
 * with n > 0 the table has n entries: a particle loaded with a species id >= n raises the sticky device fault
 * PIC_DEV_BAD_SPECIES, and the fixed-point scale of the current follows max|q| over these n entries
 * (charges of any magnitude, e.g. 1.6e-19, keep the full resolution). */
int32_t pic_set_species(pic_ctx* ctx, int32_t n, const double* q, const double* m);

/* Append n particles ("pic_load_particles(SoA x/u/weight/species)").  x,y,z: float64
 * global positions in the units of cell[], anywhere (wrapped periodically into
 * [0, N*cell)); stored internally as (cell index, fp32 in-cell fraction) — exact
 * when x/cell is an integer plus an fp32 fraction.  ux,uy,uz: float32 gamma*beta at
 * t^{n-1/2} (S4).  w: float32 weight.  species: int32 in [0, PIC_MAX_SPECIES) or
 * NULL (= all 0).  Particle ids are the load order, starting at 0 and continuing
 * across calls.  Asynchronous on the stream; the arrays must stay valid until the
 * stream reaches this point. */
int32_t pic_load_particles(pic_ctx* ctx, int64_t n,
                           const double* x, const double* y, const double* z,
                           const float* ux, const float* uy, const float* uz,
                           const float* w, const int32_t* species);

/* Set the fields ("pic_set_fields(E,B)"): six float32 grid arrays [nz][ny][nx], copied into the workspace
 * by one kernel (asynchronous) — the workspace keeps them in one array padded with their periodic images, the form
 * the step kernel's TMA loads and the field update read and write.  They stay as set (static external fields, the contract's five configs) unless
 * pic_update_fields / option "field_update" advances them. */
int32_t pic_set_fields(pic_ctx* ctx, const float* Ex, const float* Ey, const float* Ez,
                       const float* Bx, const float* By, const float* Bz);

/* Advance n steps ("pic_step(n)"); asynchronous.  Each step, per supercell:
 * stage the E/B tile + guards in shared memory, gather, Boris push, move,
 * Esirkepov deposit into a shared-memory J tile flushed once to global J, and
 * resort of particles that changed supercell.  Leavers are
 * moved to their new supercell within the call; the cell-order sort of every supercell
 * is left pending and done by the next pic_step (in its kernel's prologue) or by the
 * next call that needs the sorted arrangement (pic_load_particles, pic_get_particles,
 * pic_get_counts) — invisible to the caller, results do not depend on it. */
int32_t pic_step(pic_ctx* ctx, int32_t n);

/* One Yee update of E and B with the last step's J, closing the PIC loop (PAPER.md:60
 * "fields generated by moving particles"; c = eps0 = mu0 = 1, periodic):
 *     B^{n+1/2} = B^n - (dt/2) curl E^n;   E^{n+1} = E^n + dt (curl B^{n+1/2} - J);
 *     B^{n+1} = B^{n+1/2} - (dt/2) curl E^{n+1},
 * curl E by forward differences onto the B locations, curl B by backward differences onto the E
 * locations.  E and B are both kept at the integer time level the particle step gathers at; J is
 * whatever pic_get_current would return (zero before the first step).  After pic_step(1) this
 * advances the fields consistently with the particles; with option "field_update" = 1 every step of
 * pic_step(n) ends with it.  Asynchronous; PIC_ESTATE before pic_set_fields. */
int32_t pic_update_fields(pic_ctx* ctx);

/* Copy the current E, B out: six float32 grid arrays [nz][ny][nx] (any may be NULL).  One kernel on the
 * stream (asynchronous); PIC_ESTATE before pic_set_fields. */
int32_t pic_get_fields(pic_ctx* ctx, float* Ex, float* Ey, float* Ez, float* Bx, float* By, float* Bz);

/* Copy the last step's J ("pic_get_current"), periodic-folded, three float32 grid
 * arrays (any may be NULL).  Asynchronous device-to-device copy on the stream. */
int32_t pic_get_current(pic_ctx* ctx, float* Jx, float* Jy, float* Jz);

/* Read particles back ("pic_get_particles"), supercell-major order (S21: match by
 * id).  capacity = elements available in each non-NULL array; *n_out (host) = number
 * of particles (written even if capacity is too small, in which case PIC_ENOMEM).
 * x,y,z float64 = (cell + fraction)*cell size; supercell = linear index
 * sx + nsx*(sy + nsy*sz) of the frame list holding the particle.  Synchronises. */
int32_t pic_get_particles(pic_ctx* ctx, int64_t capacity, int64_t* n_out,
                          double* x, double* y, double* z,
                          float* ux, float* uy, float* uz, float* w,
                          int32_t* species, uint32_t* id, int32_t* supercell);

/* Per-supercell particle counts, int32[nsx*nsy*nsz] on the DEVICE.  Asynchronous. */
int32_t pic_get_counts(pic_ctx* ctx, int32_t* per_supercell_count);

/* stats (host int64[8]): [0] particles, [1] supercell-leavers of the last step,
 * [2] frames in use, [3] frames in the pool, [4] max particles in one supercell,
 * [5] steps done, [6] cumulative leavers, [7] sticky device error word.
 * Synchronises; returns PIC_EDEVICE if [7] != 0. */
int32_t pic_get_stats(pic_ctx* ctx, int64_t stats[8]);

/* Wait for the stream and report a sticky device error, if any. */
int32_t pic_sync(pic_ctx* ctx);

/* Kernel variant / measurement switches (all variants compute the same step):
 * key "tma" (1 = stage E/B tiles with cp.async.bulk.tensor, 0 = plain loads; default 1),
 * key "deposit" (1 = shared J tile accumulated in split 32-bit fixed point with native integer
 * atomics — exact, order-independent sums; 0 = float atomics, a CAS loop on sm_100a; default 1),
 * key "segment" (2..16, default 3: work-item length of the one-phase step kernel in quarters of the mean
 * cell population),
 * key "two_phase" (1 = per-cell field stencils in registers, work items of at most 11 (PQS: 6) particles,
 * gathered values staged in shared memory, Esirkepov sums in a second phase; 0 = gather per particle
 * from the shared tile; default 1),
 * key "fuse_sort" (1 = a step leaves the supercells unsorted and the next step's kernel sorts each dense
 * supercell in its prologue; 0 = a separate sort kernel before every step; default 1),
 * key "field_update" (1 = every step of pic_step ends with pic_update_fields: the self-consistent loop; default 0;
 * PIC_EINVAL, as from pic_update_fields, unless dt*sqrt(1/dx^2 + 1/dy^2 + 1/dz^2) < 1, the CFL limit of the explicit
 * Yee scheme — the particle step alone only needs c*dt < cell),
 * key "cell_kernel" (which kernel steps the dense supercells: 0 = the round-1 kernels of pic_step.cu — work items of at
 * most 11 particles — default, the fastest measured; 1 = pic_cell_kernel, one thread per cell; 2 = pic_pcell_kernel,
 * persistent CTAs whose producer warps sort and stage the next supercell beside the consumer warps; same results
 * within fp32 rounding of the per-cell sums; fixed-point deposit only),
 * key "gather" (0 = momentum-conserving gather, every component at order o from its own staggered nodes — the contract's
 * path, default; 1 = energy-conserving (Galerkin) gather: order o-1 along the
 * axes a component is staggered on, so that a field -grad_h(phi) is gathered as the exact gradient of the order-o
 * interpolation of phi; implemented in the kernels that gather per particle, hence it switches "two_phase" and
 * "cell_kernel" to 0; only before the first pic_load_particles),
 * key "direct_below" (default 768: supercells with fewer particles take the one-thread-per-particle variant),
 * key "sparse_float" (1 = a step that only launches that variant accumulates J in float, default; 0 = always fixed point),
 * key "sparse_nosort" (1 = such a step also skips the re-sort of the previous step's result and walks the slots as they
 * are — holes of leavers, appended arrivals —, with one sort in 16 steps; default; N >= 2 = the same with one sort in N
 * steps; 0 = sort before every step),
 * keys "limit_frames", "limit_exchange", "limit_tables" (fault injection for tests: lower the number of particle
 * frames / exchange-buffer entries / frame-table entries below what the workspace was sized for; only before the
 * first pic_load_particles; the step then raises PIC_DEV_FRAME_POOL_EXHAUSTED / PIC_DEV_EXCHANGE_OVERFLOW /
 * PIC_DEV_TABLE_POOL_EXHAUSTED instead of writing out of bounds),
 * key "yee_tile" (8 or 16: y extent of the field-update kernel's tile; 0 = the measured best of the kernel in use,
 * default; same results),
 * key "yee_wide" (1 = on grids at least 64 cells wide along x the field update runs the kernel with four cells per
 * thread and 16-byte accesses — default; 0 = always the kernel with one cell per thread, which narrower grids get
 * anyway; same results to rounding order),
 * key "rest_skip" (1 = in the one-thread-per-particle variant a warp whose particles are all at rest, u = 0 exactly,
 * in a supercell whose staged E/B tile is all zero skips gather, push, deposit and write-back — the step would rewrite
 * their records bit for bit; default.  0 = every particle is stepped.  Bit-identical results: tests compare the two),
 * key "overlap" (1 = the two dense variants of a step, which take disjoint supercells, are launched side by side —
 * the crowded supercells' one on a second stream the context owns, forked from and joined to the context's stream by
 * events, so the stream order the caller sees is unchanged; default.  0 = one after the other.  Same results),
 * key "yee_index64" (1 = the field-update kernel indexes with 64 bits, as it does by itself once the padded six-component
 * array exceeds 2^32 elements; default 0; same results),
 * key "class_all" (-1 = decide from the population counters read at the last synchronisation which kernel
 * variants a step launches — default; 1 = the sparse variant takes every supercell, 2 = the dense variants
 * take every supercell, 0 = classify every supercell by its population and launch all variants),
 * "segment" and "two_phase" fix the work-item layout the sorts publish: PIC_ESTATE once particles are loaded,
 * key "timing" (1 = record CUDA events around every launch of the step kernel, read
 * with pic_get_timing; default 0).  key is a host string. */
int32_t pic_set_option(pic_ctx* ctx, const char* key, int64_t value);

/* With option "timing": total device time in ms of the step-kernel launches (including the
 * sort of the previous step's result, which runs inside or right before them) since the
 * last call, and how many there were (host pointers, either may be NULL).  Synchronises
 * and resets the accumulation. */
int32_t pic_get_timing(pic_ctx* ctx, double* step_kernel_ms, int64_t* step_kernel_launches);

/* Number of kernel launches enqueued by this context so far (host counter). */
int64_t pic_launch_count(const pic_ctx* ctx);

const char* pic_last_error(const pic_ctx* ctx);   /* ctx may be NULL: last create error */

int32_t pic_destroy(pic_ctx* ctx);                /* frees host state only */

/* Replace the current the next pic_update_fields uses (device pointers, layout of pic_get_current; device-to-device
 * copies on the stream).  For a domain decomposition above this library: a rank's own deposit lacks what
 * its neighbours deposited into its boundary cells; after the guard-plane exchange the completed J is put back here
 * before the field update.  The next pic_step overwrites it. */
int32_t pic_set_current(pic_ctx* ctx, const float* Jx, const float* Jy, const float* Jz);

/* ONE entry point that allocates nothing and needs no context or workspace, for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation): the Esirkepov deposit
 * (the same arithmetic as the step's per-particle deposit) of n particles given their positions
 * before (x0,y0,z0) and after (x1,y1,z1) one step dt — float64 device arrays, global positions in the units of cell[],
 * wrapped periodically; the move is taken as the minimum image and must be shorter than one cell per axis.  qw: float32
 * device array, charge times weight.  Jx,Jy,Jz: float32 device arrays of nx*ny*nz elements, index i + nx*(j + ny*k),
 * OVERWRITTEN with that step's current.  A particle that moved a cell or more (or a NaN position) is left out and
 * element 0 of Jx, Jy and Jz is set to NaN (the call is asynchronous: the error shows in its output).
 * Scratch (3 float64 sums per cell) lives in a file-scope device array of PIC_NOALLOC_MAX_CELLS cells = 6 MiB that every
 * GPU which loads the library holds until the process exits: grids with more cells are rejected with PIC_EINVAL.  The
 * array is shared by every call and cleared by each on its stream: calls that OVERLAP on the GPU (different streams, no
 * event between them) race; calls on one stream are safe.  The first call on a device looks up the array's address
 * (cudaGetSymbolAddress; make that call outside graph capture).  Calls no cudaMalloc/cudaFree.  grid, cell: host
 * pointers; stream: cudaStream_t; errbuf (host, may be NULL): receives a message when the return value is not PIC_OK. */
#define PIC_NOALLOC_MAX_CELLS 262144
int32_t pic_deposit_current_noalloc(const int32_t grid[3], const double cell[3], double dt, int32_t shape_order,
                                    int64_t n, const double* x0, const double* y0, const double* z0,
                                    const double* x1, const double* y1, const double* z1, const float* qw,
                                    float* Jx, float* Jy, float* Jz, void* stream, char* errbuf, int64_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* PIC_B200_H */
