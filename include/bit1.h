/*
 * bit1.h -- C ABI of libbit1: the data-parallel hot path of a BIT1-style 1D3V
 * electrostatic PIC-MC timestep on one NVIDIA B200 (sm_100a).
 *
 * The operation.  arxiv/paper_2606_28534 states the problem as the PIC cycle
 * "(i) particle mover ... (ii) deposition to the grid ... (iii) field solver ... (iv) particle force
 * evaluation ... density smoothing and MC collision handling" (Background), run by the
 * mover move0/moveb and the arranger arrj/narrj, between two walls that absorb
 * plasma and take its charge (Table 3), with checkpoint/restart of per-species particle
 * records plus counts per cell.  The paper prints no equations; the exact arithmetic is
 * fixed in DESIGN.md ("Readings", "Arithmetic policy") following SURVEY.md section 8(c).
 *
 * One step of bit1_step, for every particle in array order: gather E (linear), Boris push, move,
 * periodic wrap or wall absorption (+ re-injection / pair source), null-collision Monte Carlo against
 * a uniform neutral background (elastic, ionisation, charge exchange; births appended), then a STABLE
 * counting sort by cell that drops the dead and merges the born, charge deposition to the 1D grid in
 * int64 fixed point (unit 2^-40 C), and an exact integer-scan Poisson solve giving phi and E.
 *
 * Conventions
 *  - Plain C, no torch types.  Every pointer argument says HOST or DEVICE.
 *  - Ownership: the library allocates no device memory.  The caller supplies one DEVICE workspace of
 *    bit1_workspace_size() bytes, 256-byte aligned, alive until bit1_destroy.  All input arrays and
 *    tables are copied at the call; the caller keeps them.  Streams are borrowed cudaStream_t handles.
 *  - Errors: every call returns a bit1_status; nothing throws or aborts; out-parameters are untouched
 *    on error.  Device-side faults (capacity exceeded, particle escaped the domain) set a sticky flag
 *    word that bit1_sync reports as BIT1_ERR_DEVICE_FLAG (details in bit1_moments.flags).
 *  - Every input the oracle's algorithm accepts is accepted here: a step whose far movers and births do
 *    not fit the arranger's side list is redone by a general path (full radix sort of the store) at the
 *    next call that waits for the device; results are the same bits either way.
 *  - Threading: one context, one caller thread.
 *  - There is no CPU fallback: without a CUDA device bit1_create returns BIT1_ERR_CUDA.
 */
#ifndef BIT1_H
#define BIT1_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BIT1_MAX_SPECIES 8

typedef struct bit1_ctx bit1_ctx; /* opaque, host side, owned by the library */

typedef enum {
  BIT1_OK = 0,
  BIT1_ERR_INVALID_ARG = 1,
  BIT1_ERR_RANGE = 2,       /* fixed-point charge Q_s outside [1, 2^31) */
  BIT1_ERR_CAPACITY = 3,    /* more particles than capacity, or workspace too small */
  BIT1_ERR_STATE = 4,       /* call out of order (e.g. step before load) */
  BIT1_ERR_CUDA = 5,        /* a CUDA runtime call failed / no device */
  BIT1_ERR_CHECKPOINT = 6,  /* blob does not match this context */
  BIT1_ERR_DEVICE_FLAG = 7, /* sticky device flag set; see bit1_moments.flags */
  BIT1_ERR_STATIC_LIMIT = 8 /* bit1_field_solve_static only: more cells than BIT1_FIELD_STATIC_MAX_CELLS */
} bit1_status;

/* sticky device flag bits (bit1_moments.flags) */
#define BIT1_FLAG_CAPACITY 1u  /* births beyond capacity were dropped (SURVEY 8(c) "A") */
#define BIT1_FLAG_ESCAPE 2u    /* a particle crossed more than one domain length (reading A21) */
#define BIT1_FLAG_CHECK 16u    /* checked build (libbit1_checked.so): an index check in a kernel failed; see bit1_moments */
#define BIT1_FLAG_PID_WRAP 8u  /* the 32-bit particle-id counter wrapped: newborn particles share random streams with old ones */

/* species process flags */
#define BIT1_ELASTIC 1u             /* e-D elastic, isotropic (reading A14) */
#define BIT1_IONISE 2u              /* e-D ionisation (readings A15, A16) */
#define BIT1_CX 4u                  /* D+-D charge exchange */
#define BIT1_ION_PRODUCT 8u         /* species that receives ions born by ionisation */
#define BIT1_ELECTRON_PRODUCT 16u   /* species that receives electrons born by ionisation */
#define BIT1_TARGET_MAXWELLIAN 32u  /* collision partner sampled from the neutral Maxwellian (A13) */

#define BIT1_SRC_NONE 0 /* absorbed particles die */
#define BIT1_SRC_SELF 1 /* absorbed particles are re-injected in [src_lo, src_hi) (reading A9) */
#define BIT1_SRC_PAIR 2 /* as SELF, plus one particle of src_partner born at the same place */

/* Grid ("simulation domain"; 1D, x is the wall normal). */
typedef struct {
  int32_t nc;         /* cells, >= 2, < 2^28 */
  int32_t bc;         /* 0 periodic, 1 absorbing grounded walls (phi = 0 at both, reading A8) */
  double dx;          /* m */
  double area;        /* m^2 cross-section that turns the 1D density into coulombs (reading A4) */
  double Bx, By, Bz;  /* tesla, uniform (reading A7) */
} bit1_grid;

typedef struct {
  double q, m;          /* C, kg */
  double weight;        /* real particles per macro-particle; Q = llrint(e*weight*2^40) in [1, 2^31) */
  uint32_t flags;       /* BIT1_ELASTIC | ... */
  int32_t src_mode;     /* BIT1_SRC_* */
  int32_t src_partner;  /* species index for BIT1_SRC_PAIR, else ignored */
  int32_t _pad;
  double src_vth;       /* sqrt(e*T_src/m), m/s per component */
  double pnull, numax;  /* null-collision probability per step and nu_max (1/s), caller computed (A17) */
} bit1_species;

typedef struct {
  uint64_t seed;      /* Philox key */
  uint64_t capacity;  /* max particles incl. births, < 2^31 */
  double src_lo, src_hi;          /* re-injection interval, m */
  double n0, vth_n, E_ion, m_n;   /* neutral density m^-3, sqrt(e*T0/m_n) m/s, threshold eV, neutral mass kg */
  const double *sig_el, *sig_ion, *sig_cx; /* HOST, n_sig entries each, uniform grid in eV from 0; may be NULL if n_sig == 0 */
  int32_t n_sig;
  int32_t n_norm;          /* intervals of the inverse normal CDF table */
  double dE_eV;
  const double *inv_norm;  /* HOST, n_norm + 1 entries (reading A18) */
  void *workspace;         /* DEVICE, bit1_workspace_size() bytes, 256-byte aligned */
  size_t workspace_bytes;
  void *compute_stream;    /* cudaStream_t, borrowed; NULL = default stream */
  void *side_stream;       /* cudaStream_t for checkpoint device->host copies; NULL = compute stream */
  int32_t checkpoint_staging; /* 1: reserve a device snapshot area so that every later step overlaps bit1_checkpoint's copy */
  int32_t launch_mode;     /* 0 default: bit1_step(n >= 4) replays CUDA graphs of two timesteps; 1: direct launches */
  /* Arranger internals (readings R-win, R-side); 0 = default everywhere.  None of them changes a result. */
  int32_t window_radius_max;   /* upper bound, in cells, of the adaptive sort-window radius (default 16, at most 60);
                                  the workspace holds 2*radius_max + 4 row entries per 1024-particle tile */
  int32_t window_radius_fixed; /* k >= 1 pins the radius to k - 1 cells instead of adapting it every step */
  uint64_t side_list_capacity; /* far movers + births one step may route through the sorted side list (default
                                  max(65536, capacity/16)); a step with more takes the general path (slower, same bits) */
} bit1_options;

typedef struct {
  uint64_t step, n_live;
  uint64_t count[BIT1_MAX_SPECIES];
  double kinetic_J[BIT1_MAX_SPECIES]; /* 0.5 m w sum |v|^2 */
  double px[BIT1_MAX_SPECIES];        /* m w sum vx */
  double field_J;                     /* 0.5 eps0 area dx sum g_j E_j^2 */
  uint64_t wall_count[2][BIT1_MAX_SPECIES];
  int64_t wall_charge_fixed[2];       /* unit 2^-40 C */
  int64_t rho_total_fixed;
  uint32_t flags;                     /* sticky BIT1_FLAG_* */
  uint32_t next_pid;
  uint64_t nu_overflow, dir_fallback, escape, births, reinject;
  uint64_t candidates[BIT1_MAX_SPECIES];
  uint64_t events[BIT1_MAX_SPECIES][3]; /* elastic, ionise, cx */
  uint64_t far_movers, max_far_movers_per_step; /* entries that took the sorted side list */
  uint64_t recycled;                  /* wall-recycling events (NEXT-2) */
  uint64_t general_steps;             /* steps that took the general path (side list beyond its capacity) */
  uint32_t window_radius;             /* sort-window radius, in cells, that the next step will use */
  uint32_t check_failures;            /* checked builds only: index checks that failed (flag BIT1_FLAG_CHECK) ... */
  uint32_t check_line, _pad;          /* ... source line of the first one in its kernel file ... */
  int64_t check_index, check_limit;   /* ... and the index and bound it saw */
  double *density[BIT1_MAX_SPECIES];  /* HOST, optional (NULL to skip), ng entries each, m^-3 */
} bit1_moments;

/* Bytes of device workspace for this configuration.  Reads capacity, checkpoint_staging, window_radius_max,
 * window_radius_fixed and side_list_capacity of `opt` (the pointers in it are ignored); 0 for invalid arguments. */
size_t bit1_workspace_size(const bit1_grid *grid, int nspecies, const bit1_options *opt);

/* Create a context.  grid/species/opt are HOST structs, copied.  BIT1_ERR_RANGE if any Q_s is out of
 * range; BIT1_ERR_INVALID_ARG for nc < 2, non-positive dx/dt/m/weight, bad species indices, IONISE set
 * without both product species (of equal weight); BIT1_ERR_CAPACITY if the workspace is too small. */
bit1_status bit1_create(const bit1_grid *grid, const bit1_species *species, int nspecies, double dt,
                        const bit1_options *opt, bit1_ctx **out);

/* Load n particles (arrays of n entries; HOST pointers unless ptrs_on_device != 0; pid may be NULL =
 * 0..n-1).  Requires 0 <= x < nc*dx and species < nspecies.  Afterwards: particles stably sorted by
 * cell (given order kept inside a cell), rho/phi/E valid, step = 0.  v is v(t = -dt/2) (reading A25). */
bit1_status bit1_load_particles(bit1_ctx *ctx, uint64_t n, const double *x, const double *vx,
                                const double *vy, const double *vz, const uint8_t *species,
                                const uint32_t *pid_or_null, int ptrs_on_device);

/* Enqueue nsteps timesteps on the compute stream; returns without waiting.  For nsteps >= 4 (and profiling off) the steps
 * are replays of a CUDA graph that holds two timesteps, captured on first use and again after any call that changes the
 * captured launches (load, restart, the bit1_set_* calls); bit1_options.launch_mode = 1 launches directly. */
bit1_status bit1_step(bit1_ctx *ctx, uint64_t nsteps);
/* Wait for the compute stream; BIT1_ERR_DEVICE_FLAG if the sticky flag word is non-zero. */
bit1_status bit1_sync(bit1_ctx *ctx);

/* Getters synchronise the compute stream; outputs are caller-allocated HOST buffers. */
bit1_status bit1_get_count(bit1_ctx *ctx, uint64_t *n_live, uint64_t *step, uint64_t per_species[BIT1_MAX_SPECIES]);
bit1_status bit1_get_rho(bit1_ctx *ctx, int64_t *rho_fixed_or_null, double *rho_si_or_null); /* ng entries; SI = C/m^3 */
bit1_status bit1_get_phi(bit1_ctx *ctx, double *phi); /* nc+1 entries (periodic: ghost copy at nc) */
bit1_status bit1_get_E(bit1_ctx *ctx, double *E);     /* nc+1 entries */
bit1_status bit1_get_dens(bit1_ctx *ctx, int64_t *dens_fixed); /* nspecies*ng entries, species-major */
bit1_status bit1_get_moments(bit1_ctx *ctx, bit1_moments *out);
/* Any pointer may be NULL.  n_live entries each (bit1_get_count), cell_start nc+1 entries. */
bit1_status bit1_get_particles(bit1_ctx *ctx, double *x, double *vx, double *vy, double *vz,
                               int32_t *cell, uint32_t *pid, uint8_t *species, int64_t *cell_start_or_null);

/* Wall recycling ("Plasma is absorbed at the walls (depositing charge), recycling D+ ions into D neutrals";
 * SURVEY 8(f) NEXT-2; reading N2-a): every particle of `species` absorbed at a wall leaves one particle of
 * species `to_species` at that wall (x = 0 at the left, x = nc*dx - dx*2^-20 at the right), velocity half-Maxwellian into
 * the plasma with per-component thermal speed `vth` = sqrt(e*T_wall/m_to) (slot 14 of the parent's Philox stream).  The
 * absorbed particle's own fate (death / re-injection / pair source) is unchanged.  to_species = -1 switches it off.
 * Part of the configuration: call it after bit1_create and before bit1_load_particles / bit1_restart (it enters the
 * configuration hash a checkpoint is validated against).  BIT1_ERR_INVALID_ARG for bad indices or vth < 0. */
bit1_status bit1_set_recycling(bit1_ctx *ctx, int species, int to_species, double vth);

/* Neutral particles as the collision target ("density from dens_n instead of constant n0"; PAPER.md:37
 * natural sorting "accelerates collision operators"; reading N2-b): with `species` >= 0 every null-collision
 * candidate uses the density of that stored species in its own (new) cell -- the mean of the cell's two nodes of the
 * previous step's deposit -- in place of bit1_options.n0.  numax / pnull stay the caller's bound (computed for the
 * largest density expected; beyond it bit1_moments.nu_overflow counts).  The neutrals themselves are not depleted or
 * heated by the events.  -1 returns to the uniform background.  Part of the configuration hash: call before
 * bit1_load_particles / bit1_restart. */
bit1_status bit1_set_neutral_target(bit1_ctx *ctx, int species);

/* Density smoothing ("density smoothing", "smoothing operators"; SURVEY 8(f) NEXT-1;
 * DESIGN.md reading N1-a): `passes` (0..8, 0 = off) passes of the 1-2-1 binomial filter over rho before every
 * field solve, in exact integers (each pass yields 4 x the smoothed array; the 1/4 is folded into the field
 * constants).  Periodic: indices wrap; bounded: the quarter that would cross a wall stays on the wall node, so
 * total charge is conserved.  bit1_get_rho / bit1_get_dens keep returning the raw deposit; bit1_get_rho_smoothed
 * returns 4^passes x the smoothed array the last solve used (HOST, ng entries).  Takes effect at the next step. */
bit1_status bit1_set_smoothing(bit1_ctx *ctx, int passes);
bit1_status bit1_get_rho_smoothed(bit1_ctx *ctx, int64_t *rho_s_fixed);
/* Time-averaged diagnostics (Table 2: datfile, mvflag = window, mvStep = interval; DESIGN.md
 * reading N1-b): over the last `window` steps of every `interval` steps (step counter k, r = k mod interval read
 * as interval when 0, accumulate when r > interval - window) the per-species deposited charge (int64, exact) and
 * phi (fp64, summed in step order) are accumulated on the device; at r == interval the sums are latched and
 * cleared.  window = 0 switches it off; (re)arming clears all sums.  BIT1_ERR_INVALID_ARG unless
 * 0 <= window <= interval (interval ignored when window == 0).  bit1_get_average returns the latest latched
 * sums (HOST: nspecies*ng int64, nc+1 doubles), how many steps they hold and the step counter at the latch
 * (all zero before the first latch).  The sums are part of the checkpoint. */
bit1_status bit1_set_averaging(bit1_ctx *ctx, int window, int interval);
bit1_status bit1_get_average(bit1_ctx *ctx, int64_t *dens_sum, double *phi_sum, uint64_t *count, uint64_t *step);

/* Prescribed field: overwrite E (HOST, nc+1 entries) and optionally freeze the field solve (E stays as set while rho
 * keeps being deposited): test-particle runs in a given field; the closed-form push tests use it too.  While the field
 * is frozen bit1_checkpoint is refused (see there). */
bit1_status bit1_set_E(bit1_ctx *ctx, const double *E, int freeze_field);
/* Set the step counter (Philox counter words 1-2), e.g. to continue a run that was loaded from exported records. */
bit1_status bit1_set_step(bit1_ctx *ctx, uint64_t step);

/* Checkpoint: header + device state + the SoA records of the LIVE particles (x, v, id, species; the
 * cell index and the counts per cell are functions of x and are rebuilt at restart), copied to PINNED HOST memory on
 * the side stream behind an event.  bit1_checkpoint waits for the steps enqueued so far (the live count sizes the blob)
 * and returns with the copy in flight: with checkpoint_staging = 1 the state is first snapshotted on the device and
 * every later step overlaps the copy; without it the copy reads the store directly, the next step overlaps it and the
 * one after waits.  *written <= bit1_checkpoint_size() (the size at full capacity).  The blob is valid after
 * bit1_checkpoint_wait.  bit1_restart needs a context created with the identical configuration, validates the blob
 * (BIT1_ERR_CHECKPOINT) and reproduces the run bit-identically (BASELINE.json north_star).
 * The blob carries no E (restart solves it from rho), so a run under a prescribed frozen field (bit1_set_E with
 * freeze_field != 0) cannot be checkpointed: bit1_checkpoint returns BIT1_ERR_STATE until the field is released by
 * bit1_set_E(E, 0).  Such a run is continued by reloading its particles and calling bit1_set_E again. */
size_t bit1_checkpoint_size(bit1_ctx *ctx);
bit1_status bit1_checkpoint(bit1_ctx *ctx, void *pinned_host, size_t cap, size_t *written);
bit1_status bit1_checkpoint_wait(bit1_ctx *ctx);
bit1_status bit1_restart(bit1_ctx *ctx, const void *blob_host, size_t bytes);

/* Export of one species in the paper's checkpoint layout ("per-species particle records ... the vector of
 * particle counts per cell ... local extents and offsets ... load the position and velocity records"; SURVEY 8(f)
 * NEXT-4): counts_per_cell (HOST, nc entries) and the species' records in cell order, inside a cell in the store's
 * order (HOST, *n_out entries each; any of them may be NULL; pid is the library's own addition, needed to continue a
 * run with the same random streams).  With all record pointers NULL it only returns *n_out and the counts (size
 * query); BIT1_ERR_CAPACITY (with *n_out set) if capacity_out < *n_out.  Waits for a pending checkpoint and for the
 * compute stream; uses the idle half of the particle store as staging, the live state is untouched.
 * These records (and the slots of bit1_stream_*) are for analysis and for starting a NEW run from a saved plasma: loaded
 * back with bit1_load_particles + bit1_set_step they give the same charge, counts per cell and particle ids, but not a
 * bit-identical continuation -- concatenating species changes the order inside a cell, hence which newborn particle gets
 * which id, and next_pid, the wall / event counters and the averaging sums are not part of them.  For a continuation
 * that repeats the original run use bit1_checkpoint / bit1_restart. */
bit1_status bit1_export_species(bit1_ctx *ctx, int species, uint64_t capacity_out, uint64_t *n_out,
                                int64_t *counts_per_cell, double *x, double *vx, double *vy, double *vz,
                                uint32_t *pid_or_null);

/* Streaming checkpoints: the in-memory hand-off of the paper's openPMD/ADIOS2 "SST" engine ("SST for
 * in-memory streaming"; record order of PAPER.md:57; an in-situ consumer reads the
 * checkpoints "without interrupting execution"); SURVEY 8(f) NEXT-4.  No openPMD/ADIOS2 here: the transport is a ring
 * of 2..8 slots in caller-owned PINNED HOST memory (nslots * slot_bytes, 256-byte aligned; bit1_stream_slot_size() is
 * the worst case for this context) and a sequence number.
 *   Producer (the thread that drives the context): bit1_stream_publish waits for the steps enqueued so far, compacts
 * every species on the device into the paper's record layout -- counts per cell, then x, vx, vy, vz (and the particle
 * id) in cell order --, copies the slot out on the side stream and returns; bit1_step calls that follow overlap the
 * copy.  When the copy has landed a host function on the side stream writes the slot's sequence number.  It fills a
 * free slot, else overwrites the oldest unread one; BIT1_ERR_CAPACITY if the consumer holds every slot or a slot is
 * too small.  Needs checkpoint_staging = 1 and a side stream (BIT1_ERR_STATE otherwise).
 *   Consumer (any thread of the process): bit1_stream_acquire hands out the newest complete slot with a sequence
 * number > after_seq (BIT1_ERR_STATE if there is none yet; it never blocks) and keeps the producer off it until
 * bit1_stream_release(seq).  The slot starts with a bit1_stream_header; offsets are bytes from the slot's start.
 * A reader in another process that maps the same memory follows the seqlock: a slot is complete iff
 * seq == seq_begin != 0, before and after it has copied what it needs.
 *   bit1_stream_close (producer thread) waits for the copy in flight and detaches the ring.  Consumer threads must be
 * out of bit1_stream_acquire / bit1_stream_release, and hold no slot they still read, before it is called: the ring
 * pointer and slot count are plain fields, and the memory goes back to the caller. */
#define BIT1_STREAM_MAX_SLOTS 8
typedef struct {
  char magic[8];                       /* "BIT1STRM" */
  uint64_t seq_begin;                  /* sequence number of the snapshot being written / held by this slot */
  uint64_t seq;                        /* == seq_begin once the slot is complete */
  uint64_t step, n_total, bytes;       /* step counter of the snapshot, live particles, bytes used in the slot */
  int32_t nc, ns, bc, _pad;
  uint64_t count[BIT1_MAX_SPECIES];    /* particles of species s */
  uint64_t off_counts[BIT1_MAX_SPECIES]; /* int32[nc]: particles of species s per cell */
  uint64_t off_x[BIT1_MAX_SPECIES], off_vx[BIT1_MAX_SPECIES], off_vy[BIT1_MAX_SPECIES], off_vz[BIT1_MAX_SPECIES]; /* fp64[count] */
  uint64_t off_pid[BIT1_MAX_SPECIES];  /* uint32[count] */
} bit1_stream_header;
size_t bit1_stream_slot_size(bit1_ctx *ctx);
bit1_status bit1_stream_open(bit1_ctx *ctx, void *ring_pinned_host, size_t slot_bytes, int nslots);
bit1_status bit1_stream_publish(bit1_ctx *ctx, uint64_t *seq_or_null);
bit1_status bit1_stream_acquire(bit1_ctx *ctx, uint64_t after_seq, const void **slot, uint64_t *seq);
bit1_status bit1_stream_release(bit1_ctx *ctx, uint64_t seq);
bit1_status bit1_stream_close(bit1_ctx *ctx);

/* The field solve on its own, for callers that cannot allocate device memory.
 *
 * Every other call of this library works out of the workspace handed to bit1_create, which somebody had to cudaMalloc.
 * Not every caller can: a plug-in inside a host application whose GPU memory comes from the host's own pool, a callback
 * that runs while that pool is locked, a job whose device-memory budget was fixed when it started.  Such a caller owns
 * the arrays it was given and nothing more, and cudaMalloc is either forbidden to it or would stall the whole device
 * under somebody else's pipeline.  For them this one entry point runs the step's field solve -- `smoothing_passes`
 * (0..8) passes of the 1-2-1 filter of bit1_set_smoothing over rho, then the exact integer-scan Poisson solve
 * ("(iii) field solver", "density smoothing") -- with no context, no
 * workspace, and no cudaMalloc / cudaFree / allocating library routine anywhere inside: the temporaries the solve needs
 * (per-CTA partial sums, two int64 arrays for the filter) live in an array that is part of the library image itself.
 *
 *   rho_fixed  DEVICE, in: ng int64 entries (ng = nc + 1 with walls, nc periodic), unit 2^-40 C, what bit1_get_rho returns
 *   phi, E     DEVICE, out: nc + 1 doubles each (periodic: entry nc repeats entry 0); must not overlap rho_fixed
 *   nc, bc, dx, area   as in bit1_grid
 *   stream     cudaStream_t, borrowed; NULL = default stream.  The call enqueues one kernel and returns without waiting.
 * phi and E are bit-identical to what a context with the same grid and bit1_set_smoothing(passes) computes from the
 * same rho (bit1_get_phi / bit1_get_E).
 *
 * Limits and rules that follow from the built-in array:
 *  - nc <= BIT1_FIELD_STATIC_MAX_CELLS (1 048 576, the largest grid of BASELINE.json).  A larger grid is refused with
 *    BIT1_ERR_STATIC_LIMIT and nothing is launched; use a context (bit1_create) for it.
 *  - The array (about 16 MiB) occupies device memory on every GPU of the process that loads this library, from load
 *    until the process exits, whether or not this call is ever made.
 *  - The first call on each device looks up the array's device address (cudaGetSymbolAddress) and the SM count and
 *    remembers them; make that first call with the device current and outside any CUDA stream capture.  Later calls on
 *    that device do no set-up.  The device current at the call must be the one `stream` belongs to.
 *  - All calls on one device share the one array, which still holds whatever the previous call left there.  The kernel
 *    writes every entry before it reads it, so nothing needs clearing and a call never sees an earlier call's data; but two
 *    calls that run on the GPU at the same time (different streams, or different threads) overwrite each other's
 *    temporaries and both results are garbage.  Keep the calls of one device on one stream, or order them with events.
 * BIT1_ERR_INVALID_ARG: a NULL pointer, nc < 2, bc not 0/1, dx or area not positive, passes outside 0..8.
 * BIT1_ERR_CUDA: no device, the address look-up or the launch failed. */
#define BIT1_FIELD_STATIC_MAX_CELLS 1048576
bit1_status bit1_field_solve_static(const int64_t *rho_fixed, double *phi, double *E, int32_t nc, int32_t bc, double dx,
                                    double area, int32_t smoothing_passes, void *stream);

void bit1_destroy(bit1_ctx *ctx);
const char *bit1_error_string(bit1_status s);
/* Per-kernel device timing for the roofline report.  While enabled, bit1_step
 * records CUDA events on the compute stream around each of its four kernels (first 4096 steps kept).
 * bit1_get_profile waits for the stream and returns the summed milliseconds of
 * [mover pass A, side-list + cell scan, arranger pass B, field solve] and the number of steps they
 * cover, then clears the record. */
bit1_status bit1_profile(bit1_ctx *ctx, int enable);
bit1_status bit1_get_profile(bit1_ctx *ctx, double ms[4], uint64_t *steps);
/* Kernels launched by this context since create (bench.py's gpu_launches). */
uint64_t bit1_launch_count(bit1_ctx *ctx);
/* 1 for libbit1_checked.so (the same sources built with -DBIT1_CHECKED: every index the step kernels compute from
 * particle data is compared with its bound before use; profiles/r2_sanitizer.md), 0 for the shipped library. */
int bit1_build_is_checked(void);
/* Checked build: runs one deliberately out-of-range index through the check on the device and returns BIT1_OK iff it
 * was caught and recorded (the record is cleared again).  BIT1_ERR_STATE in the shipped library. */
bit1_status bit1_check_selftest(bit1_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* BIT1_H */
