// Shared device/host structures of libbit1 (CUDA side only; the CPU oracle shares nothing with this).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bit1 {

constexpr int kMaxSpecies = 8;
// Geometry of the two particle passes (compile-time).  Two CTAs of 256 threads share an SM,
// each streaming tiles of 1024 particles: while one CTA sits at a barrier or waits for its tile, the other issues.
#ifndef BIT1_THREADS
#define BIT1_THREADS 256
#endif
#ifndef BIT1_ITEMS
#define BIT1_ITEMS 4
#endif
#ifndef BIT1_MINBLOCKS
#define BIT1_MINBLOCKS 2
#endif
#ifndef BIT1_WCAP
#define BIT1_WCAP 128
#endif
constexpr int kThreads = BIT1_THREADS;    // threads per CTA of the particle passes
constexpr int kItems = BIT1_ITEMS;        // particles per thread and tile
constexpr int kMinBlocks = BIT1_MINBLOCKS;  // CTAs per SM the passes are compiled and launched for
constexpr int kTile = kThreads * kItems;  // particles per tile (one TMA stage)
constexpr int kWCap = BIT1_WCAP;          // max cells in a tile's window (smem histogram bins)
constexpr int kWarps = kThreads / 32;
static_assert(kWCap <= kThreads && (32 % kWarps == 0 || kWarps % 32 == 0), "pass geometry");
static_assert((kWarps & (kWarps - 1)) == 0, "pass B rotates the tile hand-over among the warps by it & (kWarps - 1)");

// side-list ("far mover" / birth) key: cell | cls(2) | ord(Params::ord_bits), packed so that the radix sort of a long
// list only visits the bits in use (Params::key_bits)
constexpr unsigned long long kInvalidKey = ~0ull;
// sort-window radius: adaptive per step (DevState::R_cur) up to Params::R_max <= kMaxR
constexpr int kMaxR = (BIT1_WCAP - 8) / 2;

constexpr unsigned kFlagCapacity = 1u, kFlagEscape = 2u, kFlagPidWrap = 8u, kFlagCheck = 16u;
constexpr unsigned kElastic = 1u, kIonise = 2u, kCx = 4u, kIonProduct = 8u, kElectronProduct = 16u,
                   kTargetMaxwellian = 32u;
constexpr int kSrcNone = 0, kSrcSelf = 1, kSrcPair = 2;

struct __align__(16) SpeciesP {
  double h, tx, ty, tz, sx, sy, sz;          // the per-particle fast path reads these seven and pthr
  unsigned long long pthr;                   // u52(w) < pnull  <=>  w < pthr  (52-bit w; exact, see api.cu)
  double pnull;
  double src_vth, numax, kin_eV, two_e_over_m, el_loss;
  long long Q;
  int sign;
  unsigned flags;
  int src_mode, src_partner;
  int recycle_to, pad_;      // NEXT-2: species born at the wall when this one is absorbed (-1 = none)
  double recycle_vth;
};

// SoA particle store: 41 B per particle.
struct Particles {
  double *x, *vx, *vy, *vz;
  int *cell;
  unsigned *pid;
  unsigned char *sp;
  int2 *desc;  // per tile of this buffer: (cell of its first particle, cell of its last particle), written by k_mid
};

struct OvfRec {  // one far mover or birth, full state (48 B)
  double x, vx, vy, vz;
  unsigned pid;
  unsigned sp;
};

// Mutable device-side counters; every kernel reads n/step from here so that bit1_step never syncs.
struct DevState {
  unsigned long long step;
  unsigned n;         // live particles at step start
  unsigned n_next;    // live particles after this step's sort
  unsigned next_pid;
  unsigned ovf_count; // far movers + births appended this step
  unsigned flags;     // sticky
  unsigned freeze_field;
  unsigned load_error;
  unsigned ovf_valid; // side-list entries that k_mid placed (ovf_count minus dropped births)
  // sort window (reading R-win): radius of this step, radius chosen for the next one
  unsigned R_cur, R_next;
  // 1: this step's side list did not fit (ovf_count > ovf_cap).  Nothing of the step is committed and every later
  // kernel returns at once until the host has taken the step through the general path (api.cu settle())
  unsigned stalled;
  unsigned pad0_;
  // excess[e]: particles whose new cell lies e cells outside their tile's old cell range (e >= 2; the last bin holds
  // everything beyond kMaxR); filled by pass A, read and cleared by k_mid when it chooses R_next
  unsigned long long excess[kMaxR + 2];
  unsigned long long general_steps;   // steps that took the general path
  // checked builds (-DBIT1_CHECKED, see BIT1_CHECK below): the first failed index check and how many failed
  unsigned check_count, check_line;
  long long check_idx, check_limit;
  unsigned long long wall_count[2][kMaxSpecies];
  long long wall_charge[2];
  unsigned long long nu_overflow, dir_fallback, escape, births, reinject, recycled;
  unsigned long long candidates[kMaxSpecies];
  unsigned long long events[kMaxSpecies][3];
  unsigned long long far_movers, max_far_movers;
  long long rho_total;
  // NEXT-1: settings ride along so that a checkpoint carries them; the running/latched window counters
  int smooth_passes, avg_window, avg_interval, pad_;
  unsigned long long acc_count, avg_count, avg_step;
};

struct Params {
  int nc, bc, ng, ns;
  int R_max;     // upper bound of the adaptive window radius (rows of the banded arrays are sized for it)
  int R_fixed;   // >= 0: the radius is pinned to this value (tests); -1: adaptive
  int ord_bits, cell_shift, key_bits;   // side-list key: cell << cell_shift | cls << ord_bits | ord
  int n_sig, n_norm;
  int sp_ep, sp_ip;
  int dep_u32;   // 1: every Q_s * kTile < 2^32, shared-memory deposit counters may be 32-bit
  unsigned seed_lo, seed_hi;
  unsigned capacity, ovf_cap;
  int max_tiles;
  double inv_dx, L, dt, dx, area;
  double src_lo, src_span;
  double n0, vth_n, E_ion, dE_eV;
  double Kphi, KE;
  double field_J_factor;
  const double *sig_el, *sig_ion, *sig_cx, *inv_norm;
  DevState *st;
  // grids
  long long *dens;  // ns * ng: this step's deposit (cleared in pass A, accumulated in pass B)
  long long *dens_old;  // ns * ng: the previous step's deposit (swapped with dens every step); read by collide()
  int target_species;   // NEXT-2 (reading N2-b): species whose density is the collision target, -1 = uniform n0
  double kn;            // (0.5 * weight_n) / ((Q_n * area) * dx): node pair sum -> density of the cell
  long long *rho;   // ng
  double *phi, *E;  // nc + 1
  // NEXT-1 (density smoothing, time-averaged diagnostics; readings N1-a, N1-b)
  int smooth;                    // passes of the 1-2-1 filter over rho before the field solve (0 = off)
  int avg_window, avg_interval;  // mvflag, mvStep (0 = off)
  long long *rho_s, *rho_t;      // ng each: 4^smooth x smoothed rho (what the solve used), ping-pong scratch
  long long *acc_dens, *avg_dens;  // ns * ng: running / latched sums of dens over the averaging window
  double *acc_phi, *avg_phi;       // nc + 1
  int *cell_count;  // nc
  int *cell_start;  // nc + 1: of the arrangement this step produces (k_mid)
  int *cell_start_old;  // nc + 1: of the arrangement this step reads (swapped with cell_start every step)
  int *scan_part;   // one partial sum per CTA of k_mid
  void *coop_scratch;  // k_field: per-CTA partial sums (16-byte aligned)
  int *cell_base;   // nc: cell_start + far movers placed before the windowed particles
  int *ovf_before;  // nc
  int *ovf_lb, *ovf_ub;  // nc: first / one-past-last sorted side-list position of a cell's group (long lists)
  unsigned *radix_hist;  // 256 * (CTAs of k_mid): digit counts of the grid-wide radix sort
  // tiles
  unsigned *tile_hist;  // banded histogram rows: row t (one count per window cell) at tile_row_offset(clo_t, t, R)
  int *tile_base;       // same layout: destination of the tile's first particle of each window cell
  unsigned *tile_pre;   // row t at kWarps * tile_row_offset: per (window cell, warp of pass A/B) the number of the
                        // tile's particles for that cell held by earlier warps of the tile
  unsigned *evt;        // one bit per particle slot: pass B must take the slow path (wall hit / MC candidate)
  // overflow list
  // side list (far movers and births of the step), ovf_cap entries each
  unsigned long long *ovf_key;  // unsorted, then sorted in place
  unsigned *ovf_idx;            // record index of sorted position
  OvfRec *ovf_rec;
  int *ovf_dst;                 // destination slot of sorted position
  unsigned long long *tmp_key, *tmp2_key;  // scratch: birth ordering, radix ping-pong
  unsigned *tmp_idx, *tmp2_idx;
  SpeciesP sp[kMaxSpecies];
};

// Checked build (build.py --checked -> libbit1_checked.so; profiles/r2_sanitizer.md): every index the step kernels
// compute from particle data -- shared-memory histogram, window, deposit and counter slots, scatter destinations,
// side-list slots, banded-row offsets, cell indices, radix destinations -- is compared with its bound before use.  A
// failure is recorded (first site and value, count), raises the sticky flag kFlagCheck and the access is redirected to
// index 0 instead of corrupting memory.  The shipped library compiles the checks away.
#ifdef BIT1_CHECKED
__device__ __noinline__ inline void check_fail(DevState* st, int line, long long idx, long long limit) {
  if (atomicAdd(&st->check_count, 1u) == 0u) {
    st->check_line = (unsigned)line;
    st->check_idx = idx;
    st->check_limit = limit;
  }
  atomicOr(&st->flags, kFlagCheck);
}
template <class T, class U>
__device__ __forceinline__ T checked_index(DevState* st, int line, T idx, U limit) {
  if ((unsigned long long)(long long)idx < (unsigned long long)(long long)limit) return idx;
  check_fail(st, line, (long long)idx, (long long)limit);
  return (T)0;
}
#define BIT1_CHECK(st, idx, limit) checked_index((st), __LINE__, (idx), (limit))
#else
#define BIT1_CHECK(st, idx, limit) (idx)
#endif

// Rows never overlap: clo is monotone in the tile index and a row holds chi - clo + 1 + 2R <= the distance to the
// next row's start.  Offsets are multiples of 4 words so that a row can be fetched by a 16-byte bulk copy.
__host__ __device__ inline size_t tile_row_offset(int clo, int tile, int R) {
  return ((size_t)clo + (size_t)tile * (size_t)(2 * R + 4) + 3) & ~(size_t)3;
}
__host__ __device__ inline size_t tile_row_words(int nc, int max_tiles, int R) {
  return (size_t)nc + (size_t)(max_tiles + 1) * (size_t)(2 * R + 4) + (size_t)kWCap + 16;
}

}  // namespace bit1
