/*
 * pic.h -- C ABI of libpic: the BIT1-style particle mover + arranger on one B200.
 *
 * What the calls compute (citations are PAPER.md lines of arxiv/paper_2603_24508; the
 * paper prints no equations for these routines, so the concrete scheme is the one fixed
 * in DESIGN.md section 3, "arithmetic contract"):
 *
 *   pic_push     the particle mover, phases (i)+(iv) of the PIC cycle (the
 *                grey box of Fig. 1; `move0`/`moveb`): linear
 *                (cloud-in-cell) gather of E_x from the 1D node grid, Boris velocity
 *                update in a uniform B, x advance, periodic wrap or absorbing-wall flag
 *                ("plasma is absorbed at the walls"), new cell index.
 *   pic_arrange  the arranger `arrj`, "a sorting function" that restores
 *                the per-cell grouping ("natural sorting"), together
 *                with the particle removal `rempar2`: a STABLE counting
 *                sort of the live particles by cell; absorbed particles are dropped.
 *   pic_wall_flux per-wall absorbed-particle counters.
 *
 * Memory model (allocate once, keep resident, release at the end;
 * kernels take raw device pointers).  The CALLER owns every large device
 * array (the two particle buffer sets and the workspace; normally torch tensors) and
 * keeps them alive and untouched until pic_destroy.  The library owns the handle and
 * small device objects (E copy, per-cell count/offset, counters).  HOST pointers are
 * copied during the call and never retained.  Every pointer below says HOST or DEVICE.
 *
 * All functions return PIC_OK (0) or a negative pic_status; nothing throws or aborts.
 * Work is enqueued on the stream given at pic_create; calls documented "syncs" wait for
 * it.  One host thread per pic_sim at a time; different sims may be driven from different threads
 * (what they share -- the memory pool of pic_trim_memory -- is locked).  There is no CPU fallback: without a CUDA device
 * every compute entry point fails with PIC_ECUDA.
 *
 * Tracing: every kernel class is launched inside an NVTX range of its name ("mover", "hist", "scan",
 * "scatter", "general", "fused", "deposit", "field"; the names pic_kernel_time takes), pic_push_all,
 * pic_cycle and pic_run_host inside a range of theirs -- for nsys, or `ncu --nvtx --nvtx-include "fused/"`.
 * No cost without a profiler attached.  PIC_TRACE=1 in the environment prints the launch geometry of the
 * fused step and the phases of pic_run_host to stderr.
 */
#ifndef PIC_H_
#define PIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    PIC_OK = 0,
    PIC_EINVAL = -1,    /* NULL / non-finite / out-of-range argument */
    PIC_ENOMEM = -2,    /* host or device allocation failed */
    PIC_ECUDA = -3,     /* CUDA runtime error (text via pic_last_error) */
    PIC_ECAPACITY = -4, /* n > capacity, or workspace too small */
    PIC_ESTATE = -5     /* call not valid in the current state (see each call) */
} pic_status;

typedef enum { PIC_PERIODIC = 0, PIC_ABSORBING = 1 } pic_boundary;

/* The 1D grid: nc cells of width dx, nodes j = 0..nc at x_j = j*dx, domain [0, L),
 * L = nc*dx.  E_nodes: nc+1 doubles, HOST, copied (for a periodic grid the caller sets
 * E_nodes[nc] = E_nodes[0]).  B: uniform field; omega_c = |q/m|*|B|; the caller does
 * the trigonometry.  stream: a cudaStream_t (e.g. torch.cuda.Stream.cuda_stream) or
 * NULL for the legacy default stream. */
typedef struct {
    int32_t nc;
    int32_t boundary; /* pic_boundary */
    double dx, dt;
    const double *E_nodes; /* HOST, nc+1 */
    double B[3];
    void *stream;
} pic_grid_desc;

/* One species.  x, vx, vy, vz (fp64) and cell (int32) are structure-of-arrays DEVICE
 * buffers of `capacity` elements each, 16-byte aligned, in two sets [0] and [1]
 * (ping-pong: the arranger writes the other set).  Set [0] holds the initial state in
 * slots [0, n): every particle live, 0 <= x < L, cell == min(floor(x*(1/dx)), nc-1).
 * If the initial state is grouped by cell (cell non-decreasing) the fast arranger is
 * used from the first step; otherwise the first arrange takes the general path.
 * arrange_every: 0 = arrange only on pic_arrange(); k > 0 = pic_push also arranges
 * right after every mover step whose cumulative step count is a multiple of k.
 * workspace: DEVICE scratch of workspace_bytes >= pic_workspace_bytes(nc, capacity),
 * 256-byte aligned; may be NULL only if workspace_bytes is 0, in which case an arrange
 * that needs the general path fails with PIC_ECAPACITY. */
typedef struct {
    double qm; /* q/m: -1 electrons, +1/3672 D+ */
    int64_t n, capacity;
    double *x[2], *vx[2], *vy[2], *vz[2]; /* DEVICE */
    int32_t *cell[2];                     /* DEVICE */
    int32_t arrange_every;
    int32_t reserved;
    void *workspace; /* DEVICE */
    size_t workspace_bytes;
} pic_species_desc;

/* Filled by pic_wall_flux.  left = wall at x = 0 (absorbed iff x' < 0), right = wall at
 * x = L (absorbed iff x' >= L).  *_recent cover the interval since the previous
 * pic_wall_flux call on this species; flux = count / (steps * dt), left to the caller. */
typedef struct {
    uint64_t left_total, right_total;
    uint64_t left_recent, right_recent;
    uint64_t steps_total, steps_recent;
} pic_wall_flux_t;

typedef struct pic_sim pic_sim;
typedef struct pic_species pic_species;

/* Create a simulation of `nspecies` species on the current CUDA device.  Copies E to the
 * device, computes the per-species Boris constants on the host, validates the initial
 * state on the device and builds per-cell count/offset.  Syncs.  Errors: PIC_EINVAL
 * (NULL, nc < 1, dx/dt/B/qm not finite or dx,dt <= 0, n < 0, misaligned pointers),
 * PIC_ECAPACITY (n > capacity or n >= 2^31-64), PIC_ESTATE (a particle violates the
 * initial-state conditions above), PIC_ECUDA, PIC_ENOMEM.  On error *out is NULL. */
int pic_create(const pic_grid_desc *grid, const pic_species_desc *species, int nspecies, pic_sim **out);

/* Species handle i (0-based), or NULL.  Owned by the pic_sim. */
pic_species *pic_species_at(pic_sim *sim, int i);

/* nsteps mover steps (with the arrange_every rule).  Asynchronous on the stream.
 * Absorbed particles are flagged cell = -1, keep their final x', v' and stay in their
 * slot until the next arrange.  Errors: PIC_EINVAL (NULL, nsteps < 0), PIC_ECUDA. */
int pic_push(pic_species *sp, int nsteps);

/* nsteps mover steps of EVERY species of the sim (step by step, species by species: the result is that of
 * pic_push(sp, nsteps) on each).  The species of a step are independent -- they share only the field, which they read
 * (the paper's mover runs over x[species][cell][particle]; SURVEY.md section 8(e) "two streams on one GPU") -- so
 * each species runs on an internal stream of its own for the duration of the call and their kernels overlap; fork and
 * join are events, on return all of it is ordered on the sim's stream.  Option "species_streams" = 0 runs them back to
 * back on the sim's stream instead.  Asynchronous.  Errors: as pic_push. */
int pic_push_all(pic_sim *sim, int nsteps);

/* One arrange now: per-cell histogram, device-wide exclusive scan, stable scatter into
 * the other buffer set, which becomes the active one; afterwards slots [0, n_live) hold
 * the live particles grouped by cell, in their previous relative order.  Asynchronous.
 * Does not touch the step counter.  Errors: PIC_EINVAL, PIC_ECUDA; a displacement bound
 * or workspace problem found on the device is reported by the next syncing call. */
int pic_arrange(pic_species *sp);

/* Read the wall counters.  Syncs.  Also reports any deferred device-side error
 * (PIC_ESTATE: a particle left the domain's gather range; PIC_ECAPACITY: the general
 * arranger was needed but the workspace is too small). */
int pic_wall_flux(pic_species *sp, pic_wall_flux_t *out);

/* Charge deposition on the arranged state: PIC phase (ii), "deposition to the grid, which maps
 * particle charges ... to the mesh", with the linear (cloud-in-cell) weights of the
 * gather.  rho_dev: DEVICE, nc+1 doubles, caller-owned:
 *   rho[j] (+)= weight * ( sum over particles in cell j of (1-w) + sum over particles in cell j-1 of w ),
 * w = x/dx - floor(x/dx); on a periodic grid nodes 0 and nc carry the same (summed) value; no
 * correction at absorbing walls.  weight: charge per macro-particle over dx, sign included.
 * accumulate: 0 overwrites rho, 1 adds to it (several species).  Asynchronous on the stream, except
 * that unchecked fused steps are checked first (which syncs).  PIC_ESTATE unless the state is
 * arranged (right after an arranging step or pic_arrange): the reduction runs per cell over the
 * arranged slots.  Deterministic (fixed summation tree); agrees with a sequential sum to rounding. */
int pic_deposit(pic_species *sp, double weight, double *rho_dev, int accumulate);

/* The same deposition (PIC phase (ii)) for a caller that must not cause a device allocation.
 *
 * Who that is.  pic_deposit takes its per-cell scratch (one pair of doubles per cell) from the library's memory
 * pool the first time a species deposits, and a handle only exists after pic_create, which allocates too.  A host
 * code built the way the paper builds BIT1 -- every device array mapped once at start-up and kept for the whole run
 * (PAPER.md:89), the rest of the GPU's memory budgeted to other owners -- may have nothing left to give, or may run
 * its time loop under a rule that nothing in it allocates: cudaMalloc and cudaFree serialise the whole device, so
 * an allocation hidden in a per-step call stalls every other stream (the other species, the copies running beside
 * them) exactly where the paper wants them to overlap.  Such a caller already owns x and an offset
 * table; this call needs nothing else.
 *
 * What it does.  No handle: the caller passes the arranged positions, the offset table and the grid, and gets rho.
 *   x_dev       DEVICE, n doubles: positions of the live particles grouped by cell (the active x buffer after an
 *               arrange), every x in [0, nc*dx) with min(floor(x*(1/dx)), nc-1) equal to its cell
 *   offset_dev  DEVICE, nc+1 int32: the particles of cell c are x_dev[offset[c] .. offset[c+1]), offset[0] = 0,
 *               offset[nc] = n (what pic_cell_counts returns, uploaded by the caller)
 *   n, nc, dx   particle count (0 <= n < 2^31), cells (1 <= nc <= PIC_DEPOSIT_STATIC_MAX_NC), cell width
 *   boundary    pic_boundary: on a periodic grid nodes 0 and nc are one point and carry the same summed value
 *   weight, accumulate, rho_dev   as pic_deposit (rho_dev: DEVICE, nc+1 doubles, caller-owned, the output)
 *   stream      a cudaStream_t of the current device, or NULL for the legacy default stream
 * Same kernels, same summation tree and therefore the same bits as pic_deposit on the same state (pic_deposit picks
 * its lanes per cell from an upper bound of n; where that bound is loose the two agree to rounding instead).
 * Asynchronous on `stream`.  Nothing is read or written on the host side except the arguments.
 *
 * The scratch is a fixed array inside the library image, 16 bytes per cell for PIC_DEPOSIT_STATIC_MAX_NC cells =
 * 16 MiB, which every GPU that loads libpic.so carries until the process exits, used or not.  The call never calls
 * cudaMalloc, cudaFree, a memory pool or any library routine that allocates; it launches two kernels.
 *   - The FIRST call on each device looks up the device address of that array (cudaGetSymbolAddress, once per
 *     device, with that device current) before it launches.  Make that first call during set-up, outside any
 *     stream capture; later calls on the device only launch.
 *   - There is ONE array per device and every call uses it.  Calls that may overlap on the GPU -- different
 *     streams without an event between them, or two host threads -- race on it and produce garbage in rho: keep all
 *     calls of a device on one stream or order them with events.  The array keeps what the last call left in it;
 *     nothing in it has to start at zero, because the first kernel writes the entry of every cell c < nc before
 *     the second reads it, so the call clears nothing.
 * Errors: PIC_EINVAL (NULL pointer, n or nc out of range, dx not finite or <= 0, weight not finite, boundary not a
 * pic_boundary), PIC_ECAPACITY (nc > PIC_DEPOSIT_STATIC_MAX_NC: nothing is launched; pic_last_error names both
 * numbers -- use pic_deposit, or split the grid), PIC_ECUDA.  Validation happens before any CUDA call. */
#define PIC_DEPOSIT_STATIC_MAX_NC (1 << 20)
int pic_deposit_static(const double *x_dev, const int32_t *offset_dev, int64_t n, int32_t nc, double dx,
                       int32_t boundary, double weight, int accumulate, double *rho_dev, void *stream);

/* Replace E from a HOST array (nc+1 doubles, copied).  Steps already enqueued run with the old field.  Syncs (the
 * caller's array may be pageable, and unchecked fused steps are checked first).  PIC_EINVAL for a non-finite value. */
int pic_set_field(pic_sim *sim, const double *E_nodes_host);

/* Replace E from a DEVICE array (nc+1 doubles, copied device-to-device on the sim's stream): the field stays
 * resident on the device between steps ("keep resident"; PAPER.md:148 raw device pointers).
 * Stream-ordered, no host round trip of the field; the caller's array must be ready on the sim's stream.  max |E|
 * (the host's bound on what one step can displace a particle) is reduced on the device and read at the next
 * synchronising call; until then the split arranger also enqueues its (guarded) general path.  Unchecked fused
 * steps are checked first, which syncs only if there are any. */
int pic_set_field_device(pic_sim *sim, const double *E_nodes_dev);

/* The field solve, PIC phase (iii): "the field solver, which computes the electric ... fields by solving ...
 * Poisson's equations" with BIT1's "native Poisson solver ... and smoothing operators".
 * The paper prints neither; readings S23-S28 of DESIGN.md section 12 (normalised, epsilon_0 = 1):
 *   1. smooth_passes passes of the 1-2-1 binomial filter rho'[j] = (rho[j-1] + 2 rho[j] + rho[j+1])/4 (periodic:
 *      wraps over the nc distinct nodes; absorbing walls: the quarter leaving the grid is reflected, charge kept);
 *   2. (phi[j-1] - 2 phi[j] + phi[j+1])/dx^2 = -rho'[j]; absorbing: phi[0] = phi[nc] = 0; periodic: rho' neutralised
 *      by a uniform background, phi of zero mean, phi[nc] = phi[0];
 *   3. E[j] = -(phi[j+1] - phi[j-1])/(2 dx), one-sided at absorbing walls, wrapped on a periodic grid; E replaces
 *      the sim's field on the device (as pic_set_field_device).
 * rho_dev: DEVICE, nc+1 doubles (what pic_deposit writes), read only, ready on the sim's stream.  phi_dev: DEVICE,
 * nc+1 doubles, receives phi, or NULL.  Asynchronous on the stream (unchecked fused steps are checked first).
 * Deterministic (fixed summation trees); agrees with a sequential elimination to rounding: within 1e-12 of
 * max |phi|.  PIC_EINVAL: NULL, smooth_passes outside [0, 1024], nc < 2. */
int pic_solve_field(pic_sim *sim, const double *rho_dev, int smooth_passes, double *phi_dev);

/* Copy the field in force (nc+1 doubles) to a HOST array.  Syncs. */
int pic_get_field(pic_sim *sim, double *E_nodes_host);

/* Number of slots in use: n_live after an arrange, else n at the last arrange (dead
 * particles included).  Syncs. */
int pic_n_slots(pic_species *sp, int64_t *n);

/* Number of live particles now: the slots in use minus the particles absorbed at the walls (flagged, still in
 * their slots) since the last arrange.  Equal to pic_n_slots right after an arrange.  Syncs. */
int pic_n_live(pic_species *sp, int64_t *n);

/* Which buffer set (0 or 1) holds the current state.  Syncs if fused steps are still unchecked (a
 * declined fused step is redone by the split kernels here, as in every synchronising call);
 * read the caller-owned buffers only after this or another synchronising call. */
int pic_active_buffer(pic_species *sp, int *which);

/* Per-cell counts (nc) and exclusive offsets (nc+1, offset[nc] = n_live) of the last
 * arrange, copied to HOST arrays (either may be NULL).  Syncs.  PIC_ESTATE if the
 * state has been pushed since the last arrange (the arrays would be stale). */
int pic_cell_counts(pic_species *sp, int32_t *count_host, int32_t *offset_host);

/* Cumulative mover steps of this species since pic_create.  Does not sync. */
int pic_step_count(pic_species *sp, int64_t *steps);

/* Largest displacement bound (in cells) accumulated since the last arrange, and whether
 * the last arrange used the general path (0/1).  Diagnostics for tests.  Syncs. */
int pic_arrange_info(pic_species *sp, int32_t *w_bound, int32_t *used_general);

/* State of the fused push+arrange step of this species.  *active: 1 if the next pic_push step
 * with an arrange would take it.  *decline_reasons: OR of the reasons any fused step has been
 * redone by the split kernels so far (1 = a particle moved more than one cell or broke the
 * grouping, 2 = a cell did not fit a tile, 4 / 8 = a boundary list overflowed);
 * 0 means every fused step so far completed.  After a decline the split kernels carry on; the
 * fused path is tried again once a synchronising call finds the state arranged and the last
 * step's displacements within one cell, 16 or more steps later.  *stage_slots, *ctas_per_sm: the launch geometry
 * the next fused step would use.  Any pointer may be NULL.  Syncs. */
int pic_fused_info(pic_species *sp, int32_t *active, int32_t *decline_reasons, int32_t *stage_slots,
                   int32_t *ctas_per_sm);

/* Bytes of caller-allocated workspace a species of this size needs. */
size_t pic_workspace_bytes(int32_t nc, int64_t capacity);

/* Variant switches and tuning knobs, for measurements (profiles/ compares them).  Flags (0/1):
 * "fused": 1 = single-pass push+arrange when arrange_every == 1 (default; particles and the E
 * nodes of each chunk staged in shared memory by TMA bulk copies), 0 = separate mover / scan /
 * scatter kernels (E through the read-only global path); "fused_tma": 1 = the fused step stages particles and E by TMA bulk copies (default),
 * 0 = it reads them with plain read-only global loads (the A/B variant of profiles/); "kernel_timing": 1 = record CUDA events
 * around every kernel launch (see pic_kernel_time).  Knobs of the fused step:
 * "fused_cells_per_cta" (cells per chunk, 1..256; 0 = automatic), "fused_rows" (rows
 * of 32 slots per tile: 8, 12 or 16; 0 = automatic from the largest per-cell count),
 * "fused_stage_slots" (largest tile in slots, even, <= 32*rows; 0 = 32*rows), "fused_stages"
 * (stages of the TMA ring: 1 or 2; 0 = automatic: 2 under 8-row tiles, else 1), "fused_pdl" (1 = the three kernels
 * of a step are programmatic dependent launches: the streaming kernel overlaps its prologue with the edge kernel, the
 * commit kernel and the next step's edge kernel are set up while their predecessor runs, default;
 * 0 = plain stream order), "fused_taper" (0..3: how many times the chunk size is halved towards the end of the grid, one
 * machine-load of CTAs per size, so that the CTAs that run last are short; -1 = automatic, default: 64-cell chunks
 * tapered three times on grids of four or more waves, no taper on smaller ones).  Other flags: "species_streams"
 * (pic_push_all: 1 = every species on an internal stream of its own, default), "cycle_async" (pic_cycle: 1 = no host
 * check between the calls of a cycle, default), "field_fused" (pic_solve_field: 1 = one cooperative kernel, default;
 * 0 = six or seven separate kernels, bit-identical), "field_blocks_per_sm" (0 = automatic, 1..8: resident blocks per SM
 * of that kernel).  Results never depend on any of them.
 * PIC_EINVAL for an unknown key or a value out of range. */
int pic_set_option(pic_sim *sim, const char *key, int value);

/* Device time of one kernel class since the previous query of that class, measured with CUDA
 * event pairs recorded on the sim's stream around each of its launches while option
 * "kernel_timing" is 1 (default 0: nothing is recorded).  kernel is one of "mover", "hist",
 * "scan", "scatter", "general", "fused", "deposit", "field".  *ms_total = summed milliseconds, *spans = number of
 * timed launches (either may be NULL).  Syncs.  PIC_EINVAL for an unknown name. */
int pic_kernel_time(pic_sim *sim, const char *kernel, double *ms_total, uint64_t *spans);

/* Number of kernel launches the library has enqueued for this sim since pic_create. */
int pic_launch_count(pic_sim *sim, uint64_t *launches);

/* One species described by HOST arrays, for pic_run_host.  x, vx, vy, vz (n doubles) and
 * cell (n int32) are HOST pointers, read as the initial state (same conditions as
 * pic_species_desc) and overwritten with the final state: slots [0, n_out) of the active
 * buffer (live particles grouped by cell if the last step arranged; otherwise absorbed ones
 * are still in place with cell = -1).  n_out, wall_left, wall_right are outputs. */
typedef struct {
    double qm;
    int64_t n;
    double *x, *vx, *vy, *vz; /* HOST, in/out */
    int32_t *cell;            /* HOST, in/out */
    int32_t arrange_every;
    int32_t reserved;
    int64_t n_out;
    uint64_t wall_left, wall_right;
} pic_host_species;

/* End-to-end convenience with HOST buffers: allocates device memory, copies the species up,
 * runs pic_create + pic_push_all(nsteps), copies the final state and the wall
 * counters back and releases everything (into the library's memory pool, see pic_trim_memory).
 * grid->stream is used as in pic_create.  Pinned
 * host arrays make the copies faster but are not required.  Syncs.  Errors as pic_create /
 * pic_push, PIC_ENOMEM when the device allocation fails. */
int pic_run_host(const pic_grid_desc *grid, pic_host_species *species, int nspecies, int nsteps);

/* ncycles closed PIC cycles (Fig. 1), the field never leaving the device:
 *     pic_push_all(sim, 1);  rho = sum over species i of pic_deposit(species i, weights[i]);
 *     pic_solve_field(sim, rho, smooth_passes, phi_dev)          -- E for the next step
 * with exactly the results of those calls, but enqueued WITHOUT the host-side check each of them makes of the fused
 * steps before it (one synchronisation per cycle): should a fused step decline, the device freezes the cycle (no
 * further fused step starts, E is not replaced) and the next synchronising call redoes every cycle from that one on
 * with the checked calls.  weights: HOST, one per species (charge per macro-particle over dx, sign included).
 * rho_dev: DEVICE, nc+1 doubles, caller-owned scratch and output (the last cycle's charge density); phi_dev: DEVICE,
 * nc+1 doubles or NULL; both must stay valid until the next synchronising call.  Asynchronous whenever every species
 * runs the fused step (arrange_every == 1, arranged, all live); otherwise each cycle is the three checked calls.
 * Option "cycle_async" = 0 forces the latter.  Errors: PIC_EINVAL (NULL, ncycles < 0, passes outside 0..1024, nc < 2,
 * weight not finite), PIC_ESTATE (a species is not arranged), PIC_ENOMEM, PIC_ECUDA. */
int pic_cycle(pic_sim *sim, int ncycles, const double *weights, int smooth_passes, double *rho_dev, double *phi_dev);

/* Device memory the library owns (the handles' small objects, the field-solve scratch, the arena of
 * pic_run_host) is taken from a stream-ordered memory pool of the current device that KEEPS freed
 * memory for the next call instead of returning it to the driver ("allocate once, keep
 * resident, release at the end"): after pic_destroy / pic_run_host the bytes are free for this library
 * but still held by the process.  pic_trim_memory returns everything not in use to the driver.  Syncs
 * the device.  Errors: PIC_ECUDA. */
int pic_trim_memory(void);

int pic_sync(pic_sim *sim);     /* wait for the stream; reports deferred device errors */
void pic_destroy(pic_sim *sim); /* frees library-owned memory (into the pool, see pic_trim_memory); caller buffers untouched */
const char *pic_strerror(int status);
const char *pic_last_error(void); /* text of the last CUDA error seen by this thread */

#ifdef __cplusplus
}
#endif
#endif /* PIC_H_ */
