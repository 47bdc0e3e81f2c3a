// The kernels of one timestep:
//   k_pass_a   mover: advance every particle, banded per-tile histogram of new cells, event bits, side list of
//              far movers and births                               (PAPER.md:111 move0/moveb)
//   k_mid      order the side list, counts -> cell_start, banded column scan: destination base of every
//              (tile, window cell)                                  (row a4, scan part)
//   k_pass_b   arranger: stable ranks inside the tile, scatter to the sorted position with the charge
//              deposition fused                                    (rows a4-a5; PAPER.md:111 arrj/narrj)
//   k_field    exact integer-scan Poisson solve -> phi, E          (row a6; PAPER.md:33 step (iii))
// Both particle passes are persistent (kMinBlocks CTAs per SM) and read their tiles through the two-stage
// bulk-async pipeline of pipeline.cuh.  The store's cell array is not touched by a step (cell == cell_of(x)); a step
// whose side list does not fit stalls (DevState::stalled) and is taken by general_kernels.cu instead.
#include <cooperative_groups.h>

#include <type_traits>

#include "advance.cuh"
#include "block_ops.cuh"
#include "step_kernels.h"

namespace cg = cooperative_groups;

namespace bit1 {

// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void load_species(const Params& P, SpeciesP* s_sp) {
  const int words = P.ns * (int)(sizeof(SpeciesP) / 8);
  const unsigned long long* src = reinterpret_cast<const unsigned long long*>(P.sp);
  unsigned long long* dst = reinterpret_cast<unsigned long long*>(s_sp);
  for (int i = threadIdx.x; i < words; i += blockDim.x) dst[i] = src[i];
}

constexpr int kAuxThreads = 256;

// dynamic shared memory of both passes: [2 x Stage][pass-specific arrays][species][2 barriers]
constexpr int kDensWords = (kWCap + 1) * kMaxSpecies;
struct PassSmem {
  static constexpr size_t stages = 2 * sizeof(Stage);
  static constexpr size_t a_hist = stages;                                  // unsigned[2][kWCap][kWarps]
  static constexpr size_t a_sp = a_hist + 2 * (size_t)kWCap * kWarps * 4;   // SpeciesP[kMaxSpecies]
  static constexpr size_t a_bar = (a_sp + kMaxSpecies * sizeof(SpeciesP) + 15) & ~(size_t)15;  // 2 x u64
  static constexpr size_t a_exc = a_bar + 16;                               // unsigned[kMaxR + 2]
  static constexpr size_t a_total = a_exc + (((size_t)(kMaxR + 2) * 4 + 15) & ~(size_t)15);
  static constexpr size_t b_wc = stages;                                    // unsigned[kWarps][2][kWCap]: destinations, row counts
  static constexpr size_t b_dens = b_wc + 2 * (size_t)kWCap * kWarps * 4;   // unsigned[2][kWCap + 1][kMaxSpecies]
  static constexpr size_t b_sp = b_dens + 2 * (size_t)kDensWords * 4;
  static constexpr size_t b_bar = (b_sp + kMaxSpecies * sizeof(SpeciesP) + 15) & ~(size_t)15;
  static constexpr size_t b_total = b_bar + 16;
};

// first 52 bits of the two-word uniform of slot C0 as an integer: u52(a, b) = (w + 0.5) * 2^-52
__device__ __forceinline__ unsigned long long w52(unsigned a, unsigned b) {
  return (((unsigned long long)a << 32) | (unsigned long long)b) >> 12;
}

// ---------------------------------------------------------------------------------------------
// Pass A writes nothing into the particle store: counts, one event bit per particle, the side list.
// Per tile: phase 1 is straight-line arithmetic over the thread's kItems particles (no warp-wide operation in
// it, so the compiler interleaves the independent dependency chains); phase 2 redoes the rare particles (wall
// hit, periodic wrap, null-collision candidate, move beyond the window) through the full advance(); phase 3
// builds the banded histogram.  One CTA barrier per tile: the histogram is double-buffered.
__global__ void __launch_bounds__(kThreads, kMinBlocks) k_pass_a(const __grid_constant__ Params P, Particles cur) {
  constexpr int kWarpSpan = 32 * kItems;
  static_assert(kItems <= 4, "the (cell, warp) histogram counter holds one byte per row of the warp");
  if (P.st->stalled) return;
  typedef PassSmem SM;
  extern __shared__ __align__(128) unsigned char smem[];
  Stage* stg = reinterpret_cast<Stage*>(smem);
  unsigned* s_hist2 = reinterpret_cast<unsigned*>(smem + SM::a_hist);
  SpeciesP* s_sp = reinterpret_cast<SpeciesP*>(smem + SM::a_sp);
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem + SM::a_bar);
  unsigned* s_exc = reinterpret_cast<unsigned*>(smem + SM::a_exc);

  const unsigned n = P.st->n;
  const unsigned long long step = P.st->step;
  const int R = (int)P.st->R_cur;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ntiles = (int)((n + kTile - 1) / kTile);
  const int G = gridDim.x;

  if (threadIdx.x == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    mbar_fence_init();
    fence_proxy_async();
    for (int k = 0; k < 2; ++k) {
      const int t = blockIdx.x + k * G;
      if (t < ntiles) issue_tile(P, cur, &stg[k], &bar[k], t, cur.desc[t], R, false, true, false);
    }
  }
  load_species(P, s_sp);
  for (int k = threadIdx.x; k < 2 * kWCap * kWarps; k += kThreads) s_hist2[k] = 0;
  if (threadIdx.x < kMaxR + 2) s_exc[threadIdx.x] = 0;
  // the deposition of this step accumulates into dens: clear it here (nobody reads it during pass A)
  {
    const size_t tot = (size_t)P.ns * (size_t)P.ng;
    for (size_t i = (size_t)blockIdx.x * kThreads + threadIdx.x; i < tot; i += (size_t)G * kThreads) P.dens[i] = 0;
  }
  __syncthreads();

  int it = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += G, ++it) {
    Stage* S = &stg[it & 1];
    unsigned* s_hist = s_hist2 + (it & 1) * (kWCap * kWarps);   // [window cell][warp]
    const unsigned base = (unsigned)tile * kTile;
    const unsigned cnt = min((unsigned)kTile, n - base);
    // cells of the tile after next (its load is issued at the end of this iteration)
    int2 dn = make_int2(0, 0);
    const int tnext = tile + 2 * G;
    if (threadIdx.x == 0 && tnext < ntiles) dn = cur.desc[tnext];
    mbar_wait(&bar[it & 1], (unsigned)(it >> 1) & 1u);

    const int clo = S->d.x, chi = S->d.y;
    const TileWin tw = make_window(clo, chi, R);
    int e0, ne;
    const double* Eptr = e_window(clo, chi, e0, ne) ? (S->E - e0) : P.E;

    // The tile body, compiled twice: for whole tiles (every tile but the store's last) without the per-particle
    // "is this slot live" predicates, and for the ragged last tile with them.
    auto tile_body = [&](auto full_c) {
    constexpr bool kFull = decltype(full_c)::value;
    // phase 1
    int cn[kItems];
    double x[kItems], vx[kItems], vy[kItems], vz[kItems];
    unsigned long long thr[kItems];
    unsigned evm = 0;
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
      const int off = warp * kWarpSpan + r * 32 + lane;
      const bool have = kFull || (unsigned)off < cnt;
      const int sp = have ? (int)S->sp[off] : 0;
      const SpeciesP& s = s_sp[sp];
      x[r] = S->x[off]; vx[r] = S->vx[off]; vy[r] = S->vy[off]; vz[r] = S->vz[off];
      const int c = have ? cell_of(P, x[r]) : clo;
      const bool inside = push_fast(P, s, Eptr, c, x[r], vx[r], vy[r], vz[r]);
      cn[r] = cell_of(P, x[r]);
      const int k = cn[r] - tw.wlo;
      thr[r] = have ? s.pthr : 0ull;
      if (have && !(inside && k >= 0 && k < tw.W)) evm |= 1u << r;
    }
    unsigned long long any = 0;
#pragma unroll
    for (int r = 0; r < kItems; ++r) any |= thr[r];
    if (any) {
#pragma unroll
      for (int r = 0; r < kItems; ++r) {
        const int off = warp * kWarpSpan + r * 32 + lane;
        const uint4 w = draw(P, S->pid[off], step, 0u);  // slot C0
        if (w52(w.x, w.y) < thr[r]) evm |= 1u << r;
      }
    }
    // phase 2
    if (evm) {
#pragma unroll
      for (int r = 0; r < kItems; ++r) {
        if ((evm >> r) & 1u) {
          const int off = warp * kWarpSpan + r * 32 + lane;
          const unsigned i = base + (unsigned)off;
          const int c = slow_advance<SinkList>(P, s_sp, step, Eptr, S, off, i);
          cn[r] = c;
          if (c >= 0) {
            const int k = c - tw.wlo;
            if (!(k >= 0 && k < tw.W)) {
              emit_record(P, make_key(P, c, c < tw.wlo ? 1u : 0u, (unsigned long long)i), S->x[off], S->vx[off],
                          S->vy[off], S->vz[off], S->pid[off], (int)S->sp[off]);
              cn[r] = -2;  // placed through the side list
              // see phase 3 (a tile too sparse for its window sends cells of its own old range here: no excess)
              const int ex = max(clo - c, c - chi);
              if (ex >= 2) atomicAdd(&s_exc[BIT1_CHECK(P.st, min(ex, kMaxR + 1), kMaxR + 2)], 1u);
            }
          }
        }
      }
    }
    // phase 3
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
      const int off = warp * kWarpSpan + r * 32 + lane;
      const bool have = kFull || (unsigned)off < cnt;
      unsigned key = 0x80000000u | (unsigned)lane;  // unique: matches nobody
      if (have && cn[r] >= 0) key = (unsigned)(cn[r] - tw.wlo);
      {
        const unsigned eb = __ballot_sync(0xffffffffu, (evm >> r) & 1u);
        if (lane == 0) P.evt[BIT1_CHECK(P.st, (base >> 5) + (unsigned)(warp * kItems + r), (unsigned)(P.max_tiles + 1) * (kTile / 32))] = eb;
      }
      // the (window cell, warp) counter is four bytes, one per row of the warp: the leader of every (row, cell) group
      // writes the group's size into its own byte -- no read-modify-write, no ordering between the rows
      const unsigned m = __match_any_sync(0xffffffffu, key);
      if (!(key & 0x80000000u) && lane == __ffs(m) - 1)
        reinterpret_cast<unsigned char*>(s_hist)[(BIT1_CHECK(P.st, key, (unsigned)tw.W) * kWarps + warp) * 4 + r] =
            (unsigned char)__popc(m);
    }
    // how far outside the tile's old cell range the windowed particles land: k_mid picks the next step's radius from
    // these counts and the far movers' (phase 2).  At radius 1 a windowed particle is at most one cell outside and
    // there is nothing to count; the loop is kept out of the phases above, whose instruction count bounds the pass.
    if (R > 1) {
#pragma unroll
      for (int r = 0; r < kItems; ++r) {
        const bool have = kFull || (unsigned)(warp * kWarpSpan + r * 32 + lane) < cnt;
        const int ex = max(clo - cn[r], cn[r] - chi);
        if (have && cn[r] >= 0 && ex >= 2) atomicAdd(&s_exc[BIT1_CHECK(P.st, min(ex, kMaxR + 1), kMaxR + 2)], 1u);
      }
    }
    if (evm) fence_proxy_async();   // only the slow path writes into the stage (generic proxy) before its reload
    };   // tile_body
    if (cnt == (unsigned)kTile) tile_body(std::true_type{});
    else tile_body(std::false_type{});
    __syncthreads();
    const int kfirst = threadIdx.x, kstep = kThreads;
    // per window cell: the warps' counts become exclusive prefixes (tile_pre, read back by pass B: this warp's
    // particles for that cell start that far into the tile's run), their sum is the tile's count
    const size_t rowo = tile_row_offset(clo, tile, R);
    for (int k = kfirst; k < tw.W; k += kstep) {
      unsigned run = 0;
      unsigned* pre = P.tile_pre + BIT1_CHECK(P.st, rowo + (size_t)k, tile_row_words(P.nc, P.max_tiles, P.R_max)) * kWarps;
#pragma unroll
      for (int w = 0; w < kWarps; ++w) {
        const unsigned t = __dp4a(s_hist[k * kWarps + w], 0x01010101u, 0u);   // sum of the four rows' bytes
        s_hist[k * kWarps + w] = 0;
        pre[w] = run;
        run += t;
      }
      P.tile_hist[rowo + k] = run;
      const int c = tw.wlo + k;
      if (run && c >= 0 && c < P.nc) atomicAdd(&P.cell_count[c], (int)run);
    }
    if (threadIdx.x == 0 && tnext < ntiles) issue_tile(P, cur, S, &bar[it & 1], tnext, dn, R, false, true, false);
  }
  __syncthreads();
  if (threadIdx.x < kMaxR + 2) {
    const unsigned v = s_exc[threadIdx.x];
    if (v) atomicAdd(&P.st->excess[threadIdx.x], (unsigned long long)v);
  }
}

// ---------------------------------------------------------------------------------------------
// k_mid helpers: sorts of the side list (CTA-wide bitonic in shared memory for short lists, radix over the whole
// cooperative grid for long ones), block scans.
constexpr int kMidThreads = 1024;
constexpr int kMidWarps = kMidThreads / 32;
constexpr int kSortSmem = 2048;
constexpr int kMidRaw = 256 * kMidWarps * 4;   // bytes: radix counters [digit][warp]; the bitonic sort's keys + values alias them
static_assert(kSortSmem * 12 <= kMidRaw, "k_mid shared memory");

__device__ void cta_bitonic(unsigned long long* key, unsigned* val, unsigned n) {
  for (unsigned k = 2; k <= n; k <<= 1) {
    for (unsigned j = k >> 1; j > 0; j >>= 1) {
      for (unsigned i = threadIdx.x; i < n; i += blockDim.x) {
        const unsigned ixj = i ^ j;
        if (ixj > i) {
          const unsigned long long a = key[i], b = key[ixj];
          const bool asc = (i & k) == 0;
          if ((a > b) == asc) {
            key[i] = b; key[ixj] = a;
            const unsigned t = val[i]; val[i] = val[ixj]; val[ixj] = t;
          }
        }
      }
      __syncthreads();
    }
  }
}

__device__ __forceinline__ unsigned next_pow2(unsigned v) {
  unsigned p = 1;
  while (p < v) p <<= 1;
  return p;
}

__device__ __forceinline__ unsigned lower_bound_u64(const unsigned long long* a, unsigned n, unsigned long long v) {
  unsigned lo = 0, hi = n;
  while (lo < hi) {
    const unsigned mid = (lo + hi) >> 1;
    if (a[mid] < v) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// sort n <= kSortSmem (key, val) pairs held in global memory by one CTA; the sorted pairs stay in s_key / s_val
// (padded with kInvalidKey up to the next power of two) for the caller's binary searches
__device__ void cta_sort(unsigned long long* gkey, unsigned* gval, unsigned n, unsigned long long* s_key,
                         unsigned* s_val) {
  const unsigned P2 = next_pow2(n > 1 ? n : 1);
  for (unsigned i = threadIdx.x; i < P2; i += blockDim.x) {
    s_key[i] = i < n ? gkey[i] : kInvalidKey;
    s_val[i] = i < n ? gval[i] : 0u;
  }
  __syncthreads();
  cta_bitonic(s_key, s_val, P2);
  for (unsigned i = threadIdx.x; i < n; i += blockDim.x) { gkey[i] = s_key[i]; gval[i] = s_val[i]; }
  __syncthreads();
}

// One-CTA cooperative grids (small workloads) need no grid-wide barrier: a CTA barrier orders the block's own global
// writes for its own threads, and saves the round trip through the barrier word in global memory.
__device__ __forceinline__ void grid_or_cta_sync(cg::grid_group& grid) {
  if (gridDim.x == 1) __syncthreads();
  else { __threadfence(); grid.sync(); }
}

// Stable LSD radix sort (8-bit digits over key bits [0, nbits)) of n (key, val) pairs over the whole cooperative
// grid; (k1, v1) is scratch of the same size; the result ends in (k0, v0).  Side lists of 1e5..1e7 entries (a hot
// tail, a sheath start-up, a pinned small radius) cost a few passes over 12 B per entry instead of the
// O(n log^2 n) exchanges and grid barriers of a bitonic network.  Every CTA owns a contiguous chunk of the array and
// every warp a contiguous segment of the chunk, so "stable" is "in warp-segment order": per pass (a) per-(digit,
// warp) counts, (b) after a grid barrier every CTA derives the start of each of its (digit, warp) runs from all
// CTAs' digit totals, (c) the warps walk their segments again and scatter.
__device__ void grid_radix_sort(cg::grid_group& grid, const Params& P, unsigned long long* k0, unsigned* v0,
                                unsigned long long* k1, unsigned* v1, unsigned n, int nbits, unsigned* s_cnt,
                                int* s_warp) {
  const int G = gridDim.x, b = blockIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  unsigned per = (n + (unsigned)G - 1u) / (unsigned)G;
  per = (per + (unsigned)kMidThreads - 1u) & ~((unsigned)kMidThreads - 1u);      // whole 32-element rows per warp
  const unsigned lo = min((unsigned)b * per, n), hi = min(lo + per, n);
  const unsigned seg = per / (unsigned)kMidWarps;
  const unsigned w_lo = min(lo + (unsigned)warp * seg, hi), w_hi = min(w_lo + seg, hi);
  unsigned* ghist = P.radix_hist;   // [256][G]
  int pass = 0;
  for (int shift = 0; shift < nbits; shift += 8, ++pass) {
    for (int k = threadIdx.x; k < 256 * kMidWarps; k += kMidThreads) s_cnt[k] = 0;
    __syncthreads();
    for (unsigned i0 = w_lo; i0 < w_hi; i0 += 32) {
      const unsigned i = i0 + (unsigned)lane;
      const unsigned d = i < w_hi ? (unsigned)((k0[i] >> shift) & 255ull) : (0x80000000u | (unsigned)lane);
      const unsigned m = __match_any_sync(0xffffffffu, d);
      if (i < w_hi && lane == __ffs(m) - 1) s_cnt[d * kMidWarps + warp] += (unsigned)__popc(m);
      __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x < 256) {
      unsigned t = 0;
      for (int w = 0; w < kMidWarps; ++w) t += s_cnt[threadIdx.x * kMidWarps + w];
      ghist[(size_t)threadIdx.x * G + b] = t;
    }
    grid_or_cta_sync(grid);
    int tot = 0, mine = 0;
    if (threadIdx.x < 256) {
      for (int bb = 0; bb < G; ++bb) {
        const int v = (int)ghist[(size_t)threadIdx.x * G + bb];
        tot += v;
        if (bb < b) mine += v;
      }
    }
    int dummy;
    const int ex = block_exclusive_scan<int>(tot, s_warp, &dummy);   // entries with a smaller digit, all CTAs
    if (threadIdx.x < 256) {
      unsigned run = (unsigned)(ex + mine);
      for (int w = 0; w < kMidWarps; ++w) {
        const unsigned t = s_cnt[threadIdx.x * kMidWarps + w];
        s_cnt[threadIdx.x * kMidWarps + w] = run;
        run += t;
      }
    }
    __syncthreads();
    for (unsigned i0 = w_lo; i0 < w_hi; i0 += 32) {
      const unsigned i = i0 + (unsigned)lane;
      const bool have = i < w_hi;
      const unsigned long long key = have ? k0[i] : 0ull;
      const unsigned val = have ? v0[i] : 0u;
      const unsigned d = have ? (unsigned)((key >> shift) & 255ull) : (0x80000000u | (unsigned)lane);
      const unsigned m = __match_any_sync(0xffffffffu, d);
      const int leader = __ffs(m) - 1;
      unsigned old = 0;
      if (have && lane == leader) {
        old = s_cnt[d * kMidWarps + warp];
        s_cnt[d * kMidWarps + warp] = old + (unsigned)__popc(m);
      }
      old = __shfl_sync(0xffffffffu, old, leader);
      if (have) {
        const unsigned dst = old + (unsigned)__popc(m & lt);
        k1[BIT1_CHECK(P.st, dst, n)] = key;
        v1[dst < n ? dst : 0u] = val;
      }
      __syncwarp();
    }
    grid_or_cta_sync(grid);
    { unsigned long long* t = k0; k0 = k1; k1 = t; }
    { unsigned* t = v0; v0 = v1; v1 = t; }
  }
  if (pass & 1) {   // the result sits in the scratch pair: bring it home (k0 / k1 have swapped names)
    for (unsigned i = lo + threadIdx.x; i < hi; i += kMidThreads) { k1[i] = k0[i]; v1[i] = v0[i]; }
    grid_or_cta_sync(grid);
  }
}

// The next step's window radius (reading R-win), from pass A's excess counts: the smallest radius that leaves no more
// than one far mover per four tiles among the particles landing within R_max cells of their tile's old range -- a
// wider window costs every tile two more row entries per cell of radius, a far mover costs a side-list record, a
// sort key and a scattered placement.  Farther ones are far movers under every radius and do not bear on the choice.
__device__ void choose_radius(const Params& P, DevState* st, unsigned n) {
  int Rn = 1;
  if (P.R_fixed >= 0) {
    Rn = P.R_fixed;
  } else {
    const unsigned long long thr = (unsigned long long)(n >> 12);
    unsigned long long beyond = 0;   // particles landing r+1 .. R_max cells outside
    Rn = P.R_max;
    for (int r = P.R_max - 1; r >= 1; --r) {
      beyond += st->excess[r + 1];
      if (beyond > thr) break;
      Rn = r;
    }
  }
  st->R_next = (unsigned)Rn;
  for (int e = 0; e < kMaxR + 2; ++e) st->excess[e] = 0;
}

// k_mid: cooperative launch, one CTA per SM at most.
//   phase 0          side list: births get their pids in (parent, kind) order, the list is ordered by (cell, class,
//                    order), every cell's group joins the cell's count.  Short lists: CTA 0, in shared memory; long
//                    lists: the whole grid (radix sort).  A list beyond its capacity stalls the step (see DevState).
//   phase 1          exclusive scan of the cell counts over all CTAs -> cell_start, cell_base; counts zeroed; the
//                    (first cell, last cell) descriptor of every tile of the new arrangement (desc_out)
//   phase 2          destinations of the side-list entries; banded column scan (do_colscan): one thread per cell
//                    walks, in tile order, the tiles whose window holds the cell and hands each its destination
//                    base = cell_base[c] + what the earlier tiles send to c.  Those tiles are the ones that hold
//                    old cells c-R .. c+R, found from the previous step's cell_start.  Last, the next step's window
//                    radius is chosen from pass A's excess counts.
__global__ void __launch_bounds__(kMidThreads) k_mid(const __grid_constant__ Params P, Particles cur, int2* desc_out,
                                                     int do_colscan) {
  __shared__ __align__(16) unsigned char s_raw[kMidRaw];
  __shared__ int s_warp[33];
  __shared__ unsigned s_cnt;
  unsigned long long* s_key = reinterpret_cast<unsigned long long*>(s_raw);
  unsigned* s_val = reinterpret_cast<unsigned*>(s_raw + kSortSmem * 8);
  unsigned* s_radix = reinterpret_cast<unsigned*>(s_raw);
  cg::grid_group grid = cg::this_grid();
  DevState* st = P.st;
  if (st->stalled) return;
  const unsigned n = st->n;
  const int G = gridDim.x, b = blockIdx.x;
  const unsigned M = st->ovf_count;
  if (M > P.ovf_cap) {
    // the side list did not fit: nothing of this step is committed (pass A has only counted); the host takes the
    // step through the general path.  Every CTA sees the same count, so the whole grid leaves here.
    if (b == 0 && threadIdx.x == 0) {
      st->stalled = 1u;
      choose_radius(P, st, n);   // pass A's counts are complete: the step after the general one gets a fitting window
    }
    return;
  }
  const unsigned long long ord_mask = (1ull << P.ord_bits) - 1ull;
  const int cshift = P.cell_shift, oshift = P.ord_bits;
  const size_t gt = (size_t)b * kMidThreads + threadIdx.x, gs = (size_t)G * kMidThreads;

  const bool big = M > (unsigned)kSortSmem;   // uniform over the grid
  if (big) {
    // (a) births, compacted into (tmp_key = order, tmp_idx = record), ordered, numbered
    if (gt == 0) P.scan_part[0] = 0;
    grid_or_cta_sync(grid);
    for (size_t i = gt; i < (size_t)M; i += gs) {
      const unsigned long long key = P.ovf_key[i];
      if (((key >> oshift) & 3ull) == 2ull) {
        const int j = atomicAdd(&P.scan_part[0], 1);
        P.tmp_key[j] = key & ord_mask;
        P.tmp_idx[j] = (unsigned)i;
      }
    }
    grid_or_cta_sync(grid);
    const unsigned B = (unsigned)P.scan_part[0];
    if (B > 0) {
      if (B <= (unsigned)kSortSmem) {
        if (b == 0) cta_sort(P.tmp_key, P.tmp_idx, B, s_key, s_val);
        grid_or_cta_sync(grid);
      } else {
        grid_radix_sort(grid, P, P.tmp_key, P.tmp_idx, P.tmp2_key, P.tmp2_idx, B, P.ord_bits, s_radix, s_warp);
      }
      const unsigned room = P.capacity > n ? P.capacity - n : 0u;
      const unsigned next_pid = st->next_pid;
      for (size_t r = gt; r < (size_t)B; r += gs) {
        const unsigned rec = P.tmp_idx[r];
        if (r < room) P.ovf_rec[rec].pid = next_pid + (unsigned)r;
        else P.ovf_key[rec] = kInvalidKey;
      }
      grid_or_cta_sync(grid);
      if (gt == 0) {
        const unsigned created = B < room ? B : room;
        if (next_pid + created < next_pid) st->flags |= kFlagPidWrap;
        st->next_pid = next_pid + created;
        st->births += created;
        if (B > room) st->flags |= kFlagCapacity;
      }
    }
    // (b) the whole list by (cell, class, order); dropped births (kInvalidKey) sort behind everything
    for (size_t i = gt; i < (size_t)M; i += gs) P.ovf_idx[i] = (unsigned)i;
    grid_or_cta_sync(grid);
    grid_radix_sort(grid, P, P.ovf_key, P.ovf_idx, P.tmp_key, P.tmp_idx, M, P.key_bits, s_radix, s_warp);
    const unsigned Mv = lower_bound_u64(P.ovf_key, M, kInvalidKey);
    // (c) groups per cell: the first and last entry of every group publish its bounds ...
    for (size_t p = gt; p < (size_t)Mv; p += gs) {
      const unsigned long long key = P.ovf_key[p];
      const unsigned long long c = key >> cshift;
      const unsigned cls = (unsigned)((key >> oshift) & 3ull);
      const bool first = p == 0 || (P.ovf_key[p - 1] >> cshift) != c;
      unsigned long long nk = 0;
      const bool last = p + 1 == (size_t)Mv || ((nk = P.ovf_key[p + 1]) >> cshift) != c;
      if (first) P.ovf_lb[BIT1_CHECK(st, c, (unsigned long long)P.nc)] = (int)p;
      if (last) P.ovf_ub[BIT1_CHECK(st, c, (unsigned long long)P.nc)] = (int)p + 1;
      if (cls == 0 && (last || ((nk >> oshift) & 3ull) != 0ull)) P.ovf_before[c] = (int)p + 1;   // made relative below
    }
    grid_or_cta_sync(grid);
    // ... then every entry takes its rank from them: class 0 counts from the cell's start, classes 1-2 from its end
    for (size_t p = gt; p < (size_t)Mv; p += gs) {
      const unsigned long long key = P.ovf_key[p];
      const int c = (int)(key >> cshift);
      const unsigned cls = (unsigned)((key >> oshift) & 3ull);
      const int lb = P.ovf_lb[c], ub = P.ovf_ub[c];
      if ((int)p == lb) {
        P.cell_count[c] += ub - lb;
        const int ub0 = P.ovf_before[c];
        P.ovf_before[c] = ub0 > lb ? ub0 - lb : 0;   // class-0 entries open the group, so ub0 > lb iff there are any
      }
      P.ovf_dst[p] = cls == 0 ? (int)p - lb : (int)p - ub;
    }
    if (gt == 0) {
      st->ovf_valid = Mv;
      st->far_movers += M;
      if (M > st->max_far_movers) st->max_far_movers = M;
    }
  } else if (b == 0) {
    unsigned Mv = 0;
    if (M > 0) {
      // (a) births: order by (parent index, kind), assign pid = next_pid + r, drop those beyond capacity
      if (threadIdx.x == 0) s_cnt = 0;
      __syncthreads();
      for (unsigned i = threadIdx.x; i < M; i += blockDim.x) {
        const unsigned long long key = P.ovf_key[i];
        if (((key >> oshift) & 3ull) == 2ull) {
          const unsigned j = atomicAdd(&s_cnt, 1u);
          P.tmp_key[j] = key & ord_mask;
          P.tmp_idx[j] = i;
        }
      }
      __syncthreads();
      const unsigned B = s_cnt;
      __syncthreads();
      if (B > 0) {
        cta_sort(P.tmp_key, P.tmp_idx, B, s_key, s_val);
        const unsigned room = P.capacity > n ? P.capacity - n : 0u;
        const unsigned next_pid = st->next_pid;
        for (unsigned r = threadIdx.x; r < B; r += blockDim.x) {
          const unsigned rec = s_val[r];
          if (r < room) P.ovf_rec[rec].pid = next_pid + r;
          else P.ovf_key[rec] = kInvalidKey;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
          const unsigned created = B < room ? B : room;
          if (next_pid + created < next_pid) st->flags |= kFlagPidWrap;
          st->next_pid = next_pid + created;
          st->births += created;
          if (B > room) st->flags |= kFlagCapacity;
        }
      }
      // (b) order the whole list by (cell, class, order)
      for (unsigned i = threadIdx.x; i < M; i += blockDim.x) P.ovf_idx[i] = i;
      __syncthreads();
      cta_sort(P.ovf_key, P.ovf_idx, M, s_key, s_val);
      // the sorted keys are still in shared memory: the binary searches below are chains of dependent loads, a few
      // dozen ns each there against most of a microsecond each in global memory
      const unsigned long long* K = s_key;
      Mv = lower_bound_u64(K, M, kInvalidKey);
      // (c) groups per cell: rank inside the group, group size joins the cell count
      for (unsigned p = threadIdx.x; p < Mv; p += blockDim.x) {
        const unsigned long long key = K[p];
        const unsigned long long c = key >> cshift;
        const unsigned lb = lower_bound_u64(K, Mv, c << cshift);
        const unsigned ub = lower_bound_u64(K, Mv, (c + 1ull) << cshift);
        const unsigned cls = (unsigned)((key >> oshift) & 3ull);
        if (p == lb) {
          const unsigned ub0 = lower_bound_u64(K, Mv, (c << cshift) | (1ull << oshift));
          P.cell_count[c] += (int)(ub - lb);
          P.ovf_before[c] = (int)(ub0 - lb);
        }
        // class 0 counts from the cell's start, classes 1-2 from the cell's end
        P.ovf_dst[p] = cls == 0 ? (int)(p - lb) : (int)(p - lb) - (int)(ub - lb);
      }
    }
    if (threadIdx.x == 0) {
      st->ovf_valid = Mv;
      st->far_movers += M;
      if (M > st->max_far_movers) st->max_far_movers = M;
    }
  }
  grid_or_cta_sync(grid);

  // phase 1: scan of the cell counts.  CTA b owns cells [c_lo, c_hi).
  const int nc = P.nc;
  int per = (nc + G - 1) / G;
  per = (per + 3) & ~3;
  const int c_lo = min(b * per, nc), c_hi = min(c_lo + per, nc);
  {
    int sum = 0;
    for (int c = c_lo + (int)threadIdx.x; c < c_hi; c += kMidThreads) sum += P.cell_count[c];
    sum = block_sum<int>(sum, s_warp);
    if (threadIdx.x == 0) P.scan_part[b] = sum;
  }
  grid_or_cta_sync(grid);
  int carry, total;
  {
    int mine = 0, all = 0;
    for (int i = threadIdx.x; i < G; i += kMidThreads) {
      const int v = P.scan_part[i];
      all += v;
      if (i < b) mine += v;
    }
    carry = block_sum<int>(mine, s_warp);
    total = block_sum<int>(all, s_warp);
  }
  for (int c0 = c_lo; c0 < c_hi; c0 += kMidThreads * 4) {
    const int c = c0 + (int)threadIdx.x * 4;
    int v[4], bf[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const bool in = c + k < c_hi;
      v[k] = in ? P.cell_count[c + k] : 0;
      bf[k] = in ? P.ovf_before[c + k] : 0;
    }
    const int tsum = (v[0] + v[1]) + (v[2] + v[3]);
    int chunk;
    int ex = carry + block_exclusive_scan<int>(tsum, s_warp, &chunk);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (c + k < c_hi) {
        P.cell_start[c + k] = ex;
        P.cell_base[c + k] = ex + bf[k];
        P.cell_count[c + k] = 0;
        P.ovf_before[c + k] = 0;
        // descriptors of the new arrangement's tiles (first, last cell): the tiles that slots [ex, ex + v) touch
        // take this cell as their first cell if their first slot lies in it, as their last if their last slot does
        if (v[k] > 0) {
          const int end = ex + v[k];
          for (int t = ex / kTile; t * kTile < end; ++t) {
            const int last = min(t * kTile + kTile, total) - 1;
            if (t * kTile >= ex) desc_out[t].x = c + k;
            if (last < end) desc_out[t].y = c + k;
          }
        }
      }
      ex += v[k];
    }
    carry += chunk;
  }
  if (b == 0 && threadIdx.x == 0) {
    P.cell_start[nc] = total;
    st->n_next = (unsigned)total;
  }
  grid_or_cta_sync(grid);

  // phase 2
  const unsigned Mv = st->ovf_valid;
  for (size_t p = gt; p < Mv; p += gs) {
    const unsigned long long key = P.ovf_key[p];
    const int c = (int)(key >> cshift);
    const unsigned cls = (unsigned)((key >> oshift) & 3ull);
    const int rel = P.ovf_dst[p];
    P.ovf_dst[p] = (cls == 0 ? P.cell_start[BIT1_CHECK(st, c, P.nc)] : P.cell_start[BIT1_CHECK(st, c, P.nc) + 1]) + rel;
  }
  if (do_colscan && n > 0) {
    const int R = (int)st->R_cur;
    const int* cso = P.cell_start_old;
    for (size_t cc = gt; cc < (size_t)nc; cc += gs) {
      const int c = (int)cc;
      const int lo = cso[max(c - R, 0)];              // first old particle with cell >= c - R
      const int hi = cso[min(c + R + 1, nc)] - 1;     // last old particle with cell <= c + R
      if (lo >= (int)n || hi < 0) continue;
      const int t0 = lo / kTile, t1 = hi / kTile;
      int run = P.cell_base[c];
      // four tiles at a time: the descriptor and count loads of a batch are independent of one another, only the running
      // sum is serial (a dense cell is covered by dozens of tiles, and every load is a trip to L2)
      for (int tb4 = t0; tb4 <= t1; tb4 += 4) {
        int2 d[4];
        size_t off[4];
        unsigned cnt[4];
        bool in[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) d[q] = cur.desc[min(tb4 + q, t1)];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const TileWin tw = make_window(d[q].x, d[q].y, R);
          const int k = c - tw.wlo;
          in[q] = tb4 + q <= t1 && k >= 0 && k < tw.W;
          off[q] = tile_row_offset(d[q].x, min(tb4 + q, t1), R) + (size_t)(in[q] ? k : 0);
          cnt[q] = in[q] ? P.tile_hist[BIT1_CHECK(st, off[q], tile_row_words(nc, P.max_tiles, P.R_max))] : 0u;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          if (in[q]) {
            P.tile_base[off[q]] = run;
            run += (int)cnt[q];
          }
        }
      }
    }
  }
  // (a scan on behalf of load, restart or the general path has no excess counts to go by: the radius stays)
  if (gt == 0 && do_colscan) choose_radius(P, st, n);
}

// ---------------------------------------------------------------------------------------------
// Pass B.  A tile arrives with its particles, its window of E, its row of tile_base (destination of the tile's
// first particle of every window cell, from k_mid) and its row of tile_pre (how many of those belong to
// earlier warps, from pass A).  So every warp knows where its own particles of each cell start and works alone:
// phase 1 recomputes the push as straight-line arithmetic, phase 1b redoes the particles pass A flagged
// through the full advance(), phase 2 ranks inside (warp, cell), deposits and scatters.  The hand-over of a tile
// (flush of its double-buffered deposit, reload of its stage) is a split barrier: seven warps announce that they are
// done (bar.arrive) and go on to the tile waiting in the other stage; the eighth, taking turns, waits for them
// (bar.sync), flushes and reloads.  A warp can run one tile ahead of the slowest, never two: the stage it would need
// is only reloaded after every warp has left it, which also keeps the mbarrier phases and the two barrier ids apart.
__global__ void __launch_bounds__(kThreads, kMinBlocks)
k_pass_b(const __grid_constant__ Params P, Particles cur, Particles nxt) {
  constexpr int kWarpSpan = 32 * kItems;
  if (P.st->stalled) return;
  typedef PassSmem SM;
  extern __shared__ __align__(128) unsigned char smem[];
  Stage* stg = reinterpret_cast<Stage*>(smem);
  unsigned* s_wc = reinterpret_cast<unsigned*>(smem + SM::b_wc);        // [kWarps][kWCap] next destination
  unsigned* s_dens2 = reinterpret_cast<unsigned*>(smem + SM::b_dens);   // [2][kWCap + 1][ns]
  SpeciesP* s_sp = reinterpret_cast<SpeciesP*>(smem + SM::b_sp);
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem + SM::b_bar);

  const unsigned n = P.st->n;
  const unsigned long long step = P.st->step;
  const int R = (int)P.st->R_cur;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;   // lanes below this one (cheaper to rematerialise than S2R SR_LTMASK)
  const int ntiles = (int)((n + kTile - 1) / kTile);
  const int G = gridDim.x;
  const int ns = P.ns;
  unsigned* wc = s_wc + warp * (2 * kWCap);   // destination of the warp's first particle of every window cell
  unsigned* cw = wc + kWCap;                  // per window cell, one byte per row of the warp: the row's particles for it
  static_assert(kItems <= 4, "one byte per row in a 32-bit word");

  if (threadIdx.x == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    mbar_fence_init();
    fence_proxy_async();
    for (int k = 0; k < 2; ++k) {
      const int t = blockIdx.x + k * G;
      if (t < ntiles) issue_tile(P, cur, &stg[k], &bar[k], t, cur.desc[t], R, true, true, true);
    }
  }
  load_species(P, s_sp);
  for (int k = threadIdx.x; k < 2 * kDensWords; k += kThreads) s_dens2[k] = 0;
  __syncthreads();

  int it = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += G, ++it) {
    Stage* S = &stg[it & 1];
    unsigned* s_dens = s_dens2 + (it & 1) * kDensWords;
    const unsigned base = (unsigned)tile * kTile;
    const unsigned cnt = min((unsigned)kTile, n - base);
    int2 dn = make_int2(0, 0);
    const int tnext = tile + 2 * G;
    const bool owner = warp == (it & (kWarps - 1));
    if (owner && lane == 0 && tnext < ntiles) dn = cur.desc[tnext];
    mbar_wait(&bar[it & 1], (unsigned)(it >> 1) & 1u);
    // the stage's descriptor is only valid once its barrier has completed
    const int2 d = S->d;
    const TileWin tw = make_window(d.x, d.y, R);

    // destination of this warp's first particle of every window cell
    for (int k = lane; k < tw.W; k += 32) {
      wc[k] = (unsigned)S->tb[k] + S->pre[k * kWarps + warp];
      cw[k] = 0;
    }
    __syncwarp();

    int e0, ne;
    const double* Eptr = e_window(d.x, d.y, e0, ne) ? (S->E - e0) : P.E;

    // The tile body, compiled twice: for whole tiles (every tile but the store's last) without the per-particle
    // "is this slot live" predicates, and for the ragged last tile with them.
    auto tile_body = [&](auto full_c) {
    constexpr bool kFull = decltype(full_c)::value;
    // phase 1: new state of every particle of the tile
    double x[kItems], vx[kItems], vy[kItems], vz[kItems];
    int key[kItems];        // window-relative new cell, or -1 when the particle is not placed by this tile
    unsigned evm = 0;
    unsigned spk = 0;       // the kItems species tags, one byte each
    // pass A's event bits of this warp's kItems rows (set for live slots only)
    unsigned evw[kItems];
    if constexpr (kItems == 4) {
      const uint4 e4 = *reinterpret_cast<const uint4*>(&S->evt[warp * kItems]);
      evw[0] = e4.x; evw[1] = e4.y; evw[2] = e4.z; evw[3] = e4.w;
    } else {
#pragma unroll
      for (int r = 0; r < kItems; ++r) evw[r] = S->evt[warp * kItems + r];
    }
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
      const int off = warp * kWarpSpan + r * 32 + lane;
      const bool have = kFull || (unsigned)off < cnt;
      x[r] = S->x[off]; vx[r] = S->vx[off]; vy[r] = S->vy[off]; vz[r] = S->vz[off];
      int c = have ? cell_of(P, x[r]) : d.x;
      const int sp = have ? (int)S->sp[off] : 0;
      spk |= (unsigned)sp << (8 * r);
      evm |= ((evw[r] >> lane) & 1u) << r;
      push_fast(P, s_sp[sp], Eptr, c, x[r], vx[r], vy[r], vz[r]);
      c = cell_of(P, x[r]);
      const int k = c - tw.wlo;
      key[r] = (have && k >= 0 && k < tw.W) ? k : -1;
    }
    // phase 1b: the particles pass A flagged take the full step again, side effects off
    if (evm) {
#pragma unroll
      for (int r = 0; r < kItems; ++r) {
        if ((evm >> r) & 1u) {
          const int off = warp * kWarpSpan + r * 32 + lane;
          const int c = slow_advance<SinkNone>(P, s_sp, step, Eptr, S, off, base + (unsigned)off);
          x[r] = S->x[off]; vx[r] = S->vx[off]; vy[r] = S->vy[off]; vz[r] = S->vz[off];
          const int k = c - tw.wlo;
          key[r] = (c >= 0 && k >= 0 && k < tw.W) ? k : -1;
        }
      }
    }
    // phase 2: stable rank inside (warp, cell) -> destination; deposit; scatter.  Written as batches of the
    // same operation over the kItems particles so that the shared-memory and warp-wide operations of different
    // particles overlap instead of forming one long dependent chain.
    int sp[kItems];
    unsigned m[kItems], a[kItems];
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
      const bool valid = key[r] >= 0;
      sp[r] = (int)((spk >> (8 * r)) & 0xffu);
      m[r] = __match_any_sync(0xffffffffu, valid ? (unsigned)key[r] : (0x80000000u | (unsigned)lane));
      a[r] = valid ? deposit_a(x[r], tw.wlo + key[r], P.inv_dx, (unsigned)s_sp[sp[r]].Q) : 0u;
    }
    // stable order inside (warp, cell) is row by row, lane by lane: the leader of every (row, cell) group writes the
    // group's size into the cell's byte for that row -- distinct bytes, no read-modify-write, no ordering between the
    // rows -- and after one warp barrier every lane adds up the earlier rows' bytes of its own cell
    {
      unsigned char* cb = reinterpret_cast<unsigned char*>(cw);
#pragma unroll
      for (int r = 0; r < kItems; ++r)
        if (key[r] >= 0 && lane == __ffs(m[r]) - 1)
          cb[BIT1_CHECK(P.st, key[r], tw.W) * 4 + r] = (unsigned char)__popc(m[r]);   // 32 is written as 32: fits a byte
    }
    __syncwarp();
    // deposit (SURVEY 8(c) "D"): one shared-memory atomic pair per (cell, species) run of the warp
    if (P.dep_u32) {
      // Q < 2^21: the sum of a over a warp stays below 2^26
#pragma unroll
      for (int r = 0; r < kItems; ++r) {
        const bool valid = key[r] >= 0;
        const unsigned mk2 = valid ? ((unsigned)key[r] << 3) | (unsigned)sp[r] : (0x80000000u | (unsigned)lane);
        const unsigned m2 = __match_any_sync(0xffffffffu, mk2);
        const unsigned sa = __reduce_add_sync(m2, a[r]);
        if (valid && lane == __ffs(m2) - 1) {
          atomicAdd(&s_dens[BIT1_CHECK(P.st, key[r] * ns + sp[r], kDensWords)],
                    (unsigned)__popc(m2) * (unsigned)s_sp[sp[r]].Q - sa);
          atomicAdd(&s_dens[BIT1_CHECK(P.st, (key[r] + 1) * ns + sp[r], kDensWords)], sa);
        }
      }
    } else {
#pragma unroll
      for (int r = 0; r < kItems; ++r) {
        if (key[r] >= 0) {
          const int c = tw.wlo + key[r];
          int j1 = c + 1;
          if (!P.bc && j1 == P.nc) j1 = 0;
          const unsigned Q = (unsigned)s_sp[sp[r]].Q;
          atomicAdd((unsigned long long*)&P.dens[(size_t)sp[r] * P.ng + c], (unsigned long long)(Q - a[r]));
          atomicAdd((unsigned long long*)&P.dens[(size_t)sp[r] * P.ng + j1], (unsigned long long)a[r]);
        }
      }
    }
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
      if (key[r] >= 0) {
        const int off = warp * kWarpSpan + r * 32 + lane;
        const unsigned rows = cw[key[r]];
        unsigned o = wc[key[r]];
#pragma unroll
        for (int q = 0; q < r; ++q) o += (rows >> (8 * q)) & 0xffu;
        const unsigned dst = BIT1_CHECK(P.st, o + (unsigned)__popc(m[r] & lt), P.st->n_next);
        nxt.x[dst] = x[r]; nxt.vx[dst] = vx[r]; nxt.vy[dst] = vy[r]; nxt.vz[dst] = vz[r];
        nxt.pid[dst] = S->pid[off]; nxt.sp[dst] = (unsigned char)sp[r];
      }
    }
    if (evm) fence_proxy_async();   // only the slow path writes into the stage (generic proxy) before its reload
    };   // tile_body
    if (cnt == (unsigned)kTile) tile_body(std::true_type{});
    else tile_body(std::false_type{});
    // one warp (taking turns) hands the tile over: it waits for the others, flushes the tile's deposit and only then
    // reloads the stage (the tile after next deposits into this buffer once its load has landed)
    if (!owner) { named_bar_arrive(1 + (it & 1), kThreads); continue; }
    named_bar_sync(1 + (it & 1), kThreads);
    const int kfirst = lane, kstep = 32;
    if (P.dep_u32) {
      for (int k = kfirst; k < ns * (tw.W + 1); k += kstep) {
        const unsigned v = s_dens[k];
        if (v) {
          s_dens[k] = 0;
          const int kk = k / ns, s = k - kk * ns;
          int j = tw.wlo + kk;
          if (!P.bc && j == P.nc) j = 0;
          atomicAdd((unsigned long long*)&P.dens[(size_t)s * P.ng + j], (unsigned long long)v);
        }
      }
    }
    __syncwarp();
    if (lane == 0 && tnext < ntiles) issue_tile(P, cur, S, &bar[it & 1], tnext, dn, R, true, true, true);
  }

  // side list: far movers and births go to the slots k_mid computed for them
  const unsigned Mv = P.st->ovf_valid;
  for (unsigned p = blockIdx.x * kThreads + threadIdx.x; p < Mv; p += G * kThreads) {
    const int dst = BIT1_CHECK(P.st, P.ovf_dst[p], P.st->n_next);
    const OvfRec rec = P.ovf_rec[BIT1_CHECK(P.st, P.ovf_idx[p], P.ovf_cap)];
    const int c = (int)(P.ovf_key[p] >> P.cell_shift);
    nxt.x[dst] = rec.x; nxt.vx[dst] = rec.vx; nxt.vy[dst] = rec.vy; nxt.vz[dst] = rec.vz;
    nxt.pid[dst] = rec.pid; nxt.sp[dst] = (unsigned char)rec.sp;
    const unsigned Q = (unsigned)s_sp[rec.sp].Q;
    const unsigned a = deposit_a(rec.x, c, P.inv_dx, Q);
    int j1 = c + 1;
    if (!P.bc && j1 == P.nc) j1 = 0;
    atomicAdd((unsigned long long*)&P.dens[(size_t)rec.sp * P.ng + c], (unsigned long long)(Q - a));
    atomicAdd((unsigned long long*)&P.dens[(size_t)rec.sp * P.ng + j1], (unsigned long long)a);
  }
}

// ---------------------------------------------------------------------------------------------
// Standalone deposit (load / restart / general path; also SURVEY 8(a) row a5 as its own kernel).  *n_ptr particles.
__global__ void __launch_bounds__(kAuxThreads) k_deposit(const __grid_constant__ Params P, Particles cur,
                                                         const unsigned* n_ptr) {
  const unsigned n = *n_ptr;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  // whole warps iterate together (the match below is warp-wide)
  for (size_t i0 = (size_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u); i0 < n; i0 += stride) {
    const size_t i = i0 + (threadIdx.x & 31u);
    const bool have = i < n;
    const double x = have ? cur.x[i] : 0.0;
    const int c = cell_of(P, x), s = have ? (int)cur.sp[i] : 0;
    const unsigned Q = (unsigned)P.sp[s].Q;
    const unsigned a = deposit_a(x, c, P.inv_dx, Q);
    // neighbours in the sorted array mostly share (cell, species): one atomic per run inside the warp
    const unsigned gk = have ? (unsigned)c * kMaxSpecies + (unsigned)s : (0x80000000u | (threadIdx.x & 31u));
    const unsigned m = __match_any_sync(0xffffffffu, gk);
    unsigned long long lo = Q - a, hi = a;
    // segmented sum over the match group (small groups: loop over members)
    unsigned long long slo = 0, shi = 0;
    for (unsigned mm = m; mm; mm &= mm - 1) {
      const int src = __ffs(mm) - 1;
      slo += __shfl_sync(m, lo, src);
      shi += __shfl_sync(m, hi, src);
    }
    if (have && (int)(threadIdx.x & 31) == __ffs(m) - 1) {
      int j1 = c + 1;
      if (!P.bc && j1 == P.nc) j1 = 0;
      atomicAdd((unsigned long long*)&P.dens[(size_t)s * P.ng + c], slo);
      atomicAdd((unsigned long long*)&P.dens[(size_t)s * P.ng + j1], shi);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// k_field helpers (the kernel itself is cooperative, see below); the 128-bit block scans and sums are block_ops.cuh's.
constexpr int kFieldThreads = 256;
constexpr int kFieldItems = 4;

// One pass of CTA b over its elements j in [j_lo, j_hi] (a sub-range of 1..jmax), in chunks of
// kFieldThreads * kFieldItems.  carryS = S_{j_lo-1}, carryT = T_{j_lo} on entry.  APPLY = false: only the sums
// (returns A = sum of R_j and C = sum of the local inclusive prefixes, so that T_{j_hi+1} = T_{j_lo} +
// len * S_{j_lo-1} + C); APPLY = true: writes phi_j and E_j.
template <bool APPLY>
__device__ void field_range(const Params& P, const long long* __restrict__ R_in, double Kphi, double KE, int j_lo,
                            int j_hi, i128 tot, i128 Tn, i128 carryS, i128 carryT, i128* s_warp, i128* outA,
                            i128* outC) {
  const int nc = P.nc, bc = P.bc;
  const i128 S0 = carryS;
  i128 accC = 0;
  for (int j0 = j_lo; j0 <= j_hi; j0 += kFieldThreads * kFieldItems) {
    const int jb = j0 + (int)threadIdx.x * kFieldItems;
    i128 R[kFieldItems], Sl[kFieldItems];
    i128 run = 0;
#pragma unroll
    for (int k = 0; k < kFieldItems; ++k) {
      const int j = jb + k;
      i128 r = 0;
      if (j <= j_hi) r = bc ? (i128)R_in[j] : (i128)nc * (i128)R_in[j] - tot;
      R[k] = r;
      run += r;
      Sl[k] = run;  // inclusive local
    }
    i128 chunkS;
    const i128 exS = carryS + block_exclusive_scan<i128>(run, s_warp, &chunkS);
    i128 tsumS = 0;
#pragma unroll
    for (int k = 0; k < kFieldItems; ++k) {
      const int j = jb + k;
      Sl[k] = exS + Sl[k];   // S_j
      if (j <= j_hi) tsumS += Sl[k];
    }
    i128 chunkSS;
    i128 T = carryT + block_exclusive_scan<i128>(tsumS, s_warp, &chunkSS);  // T at this thread's first element
    if (APPLY) {
#pragma unroll
      for (int k = 0; k < kFieldItems; ++k) {
        const int j = jb + k;
        if (j <= j_hi) {
          const i128 Sj = Sl[k], Sm = Sl[k] - R[k];
          P.phi[j] = Kphi * dbl128((i128)j * Tn - (i128)nc * T);
          if (bc) {
            if (j < nc) P.E[j] = KE * dbl128((i128)nc * (Sm + Sj) - 2 * Tn);
            else P.E[nc] = KE * dbl128(2 * (i128)nc * Sm - 2 * Tn + 2 * (i128)nc * (i128)R_in[nc]);
          } else {
            P.E[j] = KE * dbl128((i128)nc * (Sm + Sj) - 2 * Tn);
          }
          T += Sj;
        }
      }
    }
    carryS += chunkS;
    carryT += chunkSS;
    accC += chunkSS;
  }
  if (!APPLY) {
    // chunkSS sums S_j = S0 + local prefix: take the S0 part out again
    const int len = j_hi >= j_lo ? j_hi - j_lo + 1 : 0;
    *outA = carryS - S0;
    *outC = accC - (i128)len * S0;
  }
}

// k_field: cooperative launch.  rho = sum_s sign_s dens_s; exact integer double prefix sum -> phi, E
// (SURVEY 8(c) "P").  Phase A: rho and the two plain reductions (total charge, T_nc); phase B: every CTA sums its
// range of elements; phase C: carries from the CTAs before it, then phi and E.
__global__ void __launch_bounds__(kFieldThreads) k_field(const __grid_constant__ Params P, int commit_step) {
  __shared__ i128 s_warp[33];
  cg::grid_group grid = cg::this_grid();
  const int nc = P.nc, ng = P.ng, bc = P.bc;
  const int G = gridDim.x, b = blockIdx.x;
  DevState* st = P.st;
  if (st->stalled) return;
  i128* part = reinterpret_cast<i128*>(P.coop_scratch);  // [4][G]: tot, wsum, A, C
  // phase A: rho, then (NEXT-1, reading N1-a) `smooth` passes of the exact-integer 1-2-1 filter, then the two
  // plain reductions over the array the solve uses
  const int smooth = P.smooth;
  const long long* R = P.rho;
  double Kphi = P.Kphi, KE = P.KE;
  i128 tot = 0, wsum = 0;
  if (smooth > 0) {
    for (int j = b * kFieldThreads + (int)threadIdx.x; j < ng; j += G * kFieldThreads) {
      long long r = 0;
      for (int s = 0; s < P.ns; ++s) r += (long long)P.sp[s].sign * P.dens[(size_t)s * ng + j];
      P.rho[j] = r;
    }
    const long long* in = P.rho;
    for (int k = 0; k < smooth; ++k) {
      long long* out = ((smooth - 1 - k) & 1) ? P.rho_t : P.rho_s;   // the last pass lands in rho_s
      __threadfence();
      grid_or_cta_sync(grid);
      for (int j = b * kFieldThreads + (int)threadIdx.x; j < ng; j += G * kFieldThreads) {
        long long v;
        if (bc) {
          if (j == 0) v = 3 * in[0] + in[1];
          else if (j == nc) v = in[nc - 1] + 3 * in[nc];
          else v = in[j - 1] + 2 * in[j] + in[j + 1];
        } else {
          const int jm = j == 0 ? nc - 1 : j - 1, jp = j == nc - 1 ? 0 : j + 1;
          v = in[jm] + 2 * in[j] + in[jp];
        }
        out[j] = v;
      }
      in = out;
    }
    __threadfence();
    grid_or_cta_sync(grid);
    R = P.rho_s;
    const double scale = 1.0 / (double)(1ll << (2 * smooth));   // exact power of two
    Kphi = Kphi * scale;
    KE = KE * scale;
    for (int j = b * kFieldThreads + (int)threadIdx.x; j < ng; j += G * kFieldThreads) {
      const long long r = R[j];
      tot += (i128)r;
      if (j >= 1 && j <= nc - 1) wsum += (i128)(nc - j) * (i128)r;
    }
  } else {
    for (int j = b * kFieldThreads + (int)threadIdx.x; j < ng; j += G * kFieldThreads) {
      long long r = 0;
      for (int s = 0; s < P.ns; ++s) r += (long long)P.sp[s].sign * P.dens[(size_t)s * ng + j];
      P.rho[j] = r;
      tot += (i128)r;
      if (j >= 1 && j <= nc - 1) wsum += (i128)(nc - j) * (i128)r;
    }
  }
  tot = block_sum<i128>(tot, s_warp);
  wsum = block_sum<i128>(wsum, s_warp);
  if (G > 1) {   // (a one-CTA grid already holds the totals)
    if (threadIdx.x == 0) { part[b] = tot; part[G + b] = wsum; }
    __threadfence();
    grid_or_cta_sync(grid);
    tot = 0; wsum = 0;
    for (int i = threadIdx.x; i < G; i += kFieldThreads) { tot += part[i]; wsum += part[G + i]; }
    tot = block_sum<i128>(tot, s_warp);
    wsum = block_sum<i128>(wsum, s_warp);
  }
  if (b == 0 && threadIdx.x == 0) st->rho_total = (long long)(tot >> (2 * smooth));   // the filter conserves charge
  const bool frozen = st->freeze_field != 0;
  if (!frozen) {
    // periodic: R'_j = nc R_j - tot  =>  T_nc' = nc * wsum - tot * nc (nc - 1) / 2
    const i128 Tn = bc ? wsum : (i128)nc * wsum - tot * (((i128)nc * (i128)(nc - 1)) / 2);
    // elements j = 1..jmax, CTA b owns [j_lo, j_hi]
    const int jmax = bc ? nc : nc - 1;
    const int unit = kFieldThreads * kFieldItems;
    int per = (jmax + G - 1) / G;
    per = ((per + unit - 1) / unit) * unit;
    const int j_lo = min(1 + b * per, jmax + 1), j_hi = min(j_lo + per - 1, jmax);
    i128 carryS = 0, carryT = 0, Send = 0;
    if (G > 1) {
      // phase B
      i128 A = 0, C = 0;
      field_range<false>(P, R, Kphi, KE, j_lo, j_hi, tot, Tn, (i128)0, (i128)0, s_warp, &A, &C);
      if (threadIdx.x == 0) { part[2 * G + b] = A; part[3 * G + b] = C; }
      __threadfence();
      grid_or_cta_sync(grid);
      // phase C: S_{j_lo-1} = sum of A over earlier CTAs; T_{j_lo} = sum over earlier CTAs of (len * S_before + C)
      i128 myA = 0, myLen = 0, myC = 0;
      if ((int)threadIdx.x < G) {
        const int i = threadIdx.x;
        myA = part[2 * G + i];
        myC = part[3 * G + i];
        const int lo = min(1 + i * per, jmax + 1), hi = min(lo + per - 1, jmax);
        myLen = hi >= lo ? hi - lo + 1 : 0;
      }
      i128 dummy;
      const i128 Sbefore = block_exclusive_scan<i128>(myA, s_warp, &dummy);            // S at the start of CTA i
      const i128 term = ((int)threadIdx.x < b) ? myLen * Sbefore + myC : (i128)0;
      carryT = block_sum<i128>(term, s_warp);
      carryS = block_sum<i128>(((int)threadIdx.x < b) ? myA : (i128)0, s_warp);
      Send = block_sum<i128>(myA, s_warp);                                              // S_jmax
    } else if (!bc) {
      // one CTA owns every element: no carries; S_jmax = sum_{j=1}^{nc-1} (nc R_j - tot) = tot - nc R_0
      Send = tot - (i128)nc * (i128)R[0];
    }
    if (b == 0 && threadIdx.x == 0) {
      // node 0
      P.phi[0] = Kphi * dbl128((i128)0);
      if (bc) {
        P.E[0] = KE * dbl128(-2 * Tn - 2 * (i128)nc * (i128)R[0]);
      } else {
        // periodic: S_{-1} = S_{nc-1}, S_0 = 0; ghosts at nc
        P.E[0] = KE * dbl128((i128)nc * (Send + (i128)0) - 2 * Tn);
        P.E[nc] = P.E[0];
        P.phi[nc] = P.phi[0];
      }
    }
    field_range<true>(P, R, Kphi, KE, j_lo, j_hi, tot, Tn, carryS, carryT, s_warp, nullptr, nullptr);
  }
  if (b == 0 && threadIdx.x == 0) {
    st->n = st->n_next;
    if (commit_step) st->step += 1ull;
    st->ovf_count = 0;
    st->ovf_valid = 0;
    const unsigned Rn = P.R_fixed >= 0 ? (unsigned)P.R_fixed : st->R_next;
    st->R_cur = Rn < 1u && P.R_fixed < 0 ? 1u : Rn;
  }
}

// ---------------------------------------------------------------------------------------------
// k_average (NEXT-1, reading N1-b; PAPER.md:79-83 mvflag / mvStep): runs after k_field when averaging is armed.
// Step counter k (already advanced): r = k mod interval (0 read as interval); the step's dens and phi join the
// running sums when r > interval - window; at r == interval the sums are latched and cleared.
__global__ void __launch_bounds__(kAuxThreads) k_average(const __grid_constant__ Params P) {
  DevState* st = P.st;
  if (st->stalled) return;   // the step did not happen
  const unsigned long long I = (unsigned long long)P.avg_interval, W = (unsigned long long)P.avg_window;
  unsigned long long r = st->step % I;
  if (r == 0) r = I;
  const bool in_window = r > I - W, latch = r == I;
  if (!in_window && !latch) return;
  const size_t nd = (size_t)P.ns * (size_t)P.ng, gsz = (size_t)gridDim.x * blockDim.x;
  const size_t g0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (size_t i = g0; i < nd; i += gsz) {
    long long a = P.acc_dens[i];
    if (in_window) a += P.dens[i];
    if (latch) { P.avg_dens[i] = a; a = 0; }
    P.acc_dens[i] = a;
  }
  for (size_t j = g0; j <= (size_t)P.nc; j += gsz) {
    double a = P.acc_phi[j];
    if (in_window) a = a + P.phi[j];
    if (latch) { P.avg_phi[j] = a; a = 0.0; }
    P.acc_phi[j] = a;
  }
  if (g0 == 0) {
    unsigned long long c = st->acc_count + (in_window ? 1ull : 0ull);
    if (latch) { st->avg_count = c; st->avg_step = st->step; c = 0; }
    st->acc_count = c;
  }
}

// ---------------------------------------------------------------------------------------------
// host-side launchers
// SMs of the current device, asked once per device (grids are sized from it everywhere; step_kernels.h)
int sm_count() {
  constexpr int kMaxDev = 64, kB200Sms = 148;   // the fallback only if the attribute query itself fails
  static int cache[kMaxDev] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDev) return kB200Sms;
  if (cache[dev] <= 0) {
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return kB200Sms;
    cache[dev] = sms;
  }
  return cache[dev];
}

// persistent grid: kMinBlocks CTAs per SM (or one per tile when there are fewer tiles than that)
static int particle_grid(const Params& P) {
  const int want = sm_count() * kMinBlocks;
  return P.max_tiles < want ? (P.max_tiles > 0 ? P.max_tiles : 1) : want;
}

cudaError_t configure_kernels() {
  typedef PassSmem SM;
  cudaError_t e = cudaFuncSetAttribute(k_pass_a, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::a_total);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_pass_b, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::b_total);
}

#ifndef BIT1_ONE_CTA_CELLS
#define BIT1_ONE_CTA_CELLS 1024
#endif
static int coop_grid(int work_items, int per_cta) {
  // small grids: one CTA loops over its chunks with CTA barriers only, instead of a few CTAs meeting at grid barriers
  if (work_items <= BIT1_ONE_CTA_CELLS + 1) return 1;
  int g = (work_items + per_cta - 1) / per_cta;
  if (g < 1) g = 1;
  const int cap = sm_count() < kFieldThreads ? sm_count() : kFieldThreads;   // co-resident, and G <= threads
  return g < cap ? g : cap;
}

int launch_mid(const Params& P, const Particles& cur, int2* desc_out, int do_colscan, cudaStream_t s) {
  Params Pc = P;
  Particles pc = cur;
  int2* dout = desc_out;
  int dc = do_colscan;
  void* args[] = {&Pc, &pc, &dout, &dc};
  const int g = coop_grid(P.nc, kMidThreads);
  // a one-CTA grid synchronises with CTA barriers only (grid_or_cta_sync): a plain launch, without the cooperative
  // launch's residency bookkeeping on the stream
  if (g == 1) k_mid<<<1, kMidThreads, 0, s>>>(Pc, pc, dout, dc);
  else cudaLaunchCooperativeKernel((const void*)k_mid, dim3(g), dim3(kMidThreads), args, 0, s);
  return 1;
}

int launch_field(const Params& P, int commit_step, cudaStream_t s) {
  Params Pc = P;
  int cs = commit_step;
  void* args[] = {&Pc, &cs};
  const int g = coop_grid(P.ng, kFieldThreads * kFieldItems);
  if (g == 1) k_field<<<1, kFieldThreads, 0, s>>>(Pc, cs);
  else cudaLaunchCooperativeKernel((const void*)k_field, dim3(g), dim3(kFieldThreads), args, 0, s);
  return 1;
}

// time-averaged diagnostics of the step just taken (NEXT-1), when armed
int launch_average(const Params& P, cudaStream_t s) {
  if (P.avg_window <= 0) return 0;
  k_average<<<sm_count(), kAuxThreads, 0, s>>>(P);
  return 1;
}

int launch_step(const Params& P, const Particles& cur, const Particles& nxt, cudaStream_t s, cudaEvent_t* ev) {
  typedef PassSmem SM;
  const int g = particle_grid(P);
  if (ev) cudaEventRecord(ev[0], s);
  k_pass_a<<<g, kThreads, SM::a_total, s>>>(P, cur);
  if (ev) cudaEventRecord(ev[1], s);
  launch_mid(P, cur, nxt.desc, 1, s);
  if (ev) cudaEventRecord(ev[2], s);
  k_pass_b<<<g, kThreads, SM::b_total, s>>>(P, cur, nxt);
  if (ev) cudaEventRecord(ev[3], s);
  launch_field(P, 1, s);
  if (ev) cudaEventRecord(ev[4], s);
  return 4 + launch_average(P, s);
}

// load / restart: counts -> cell_start and tile descriptors, deposit, field (no push).  cur must be sorted by cell.
__global__ void __launch_bounds__(kAuxThreads) k_count_cells(const __grid_constant__ Params P, Particles cur) {
  const unsigned n = P.st->n;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i0 = (size_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u); i0 < n; i0 += stride) {
    const size_t i = i0 + (threadIdx.x & 31u);
    const bool have = i < n;
    const unsigned c = have ? (unsigned)cell_of(P, cur.x[i]) : (0x80000000u | (threadIdx.x & 31u));
    const unsigned m = __match_any_sync(0xffffffffu, c);
    if (have && (int)(threadIdx.x & 31u) == __ffs(m) - 1) atomicAdd(&P.cell_count[c], __popc(m));
  }
}
__global__ void k_clear_grids(const __grid_constant__ Params P) {
  const size_t tot = (size_t)P.ns * (size_t)P.ng;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < tot; i += (size_t)gridDim.x * blockDim.x)
    P.dens[i] = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)P.nc; i += (size_t)gridDim.x * blockDim.x) {
    P.cell_count[i] = 0;
    P.ovf_before[i] = 0;
  }
}

int launch_clear_grids(const Params& P, cudaStream_t s) {
  k_clear_grids<<<sm_count() * 4, 256, 0, s>>>(P);
  return 1;
}

int launch_deposit(const Params& P, const Particles& cur, const unsigned* n_ptr, cudaStream_t s) {
  k_deposit<<<sm_count() * 4, kAuxThreads, 0, s>>>(P, cur, n_ptr);
  return 1;
}

int launch_rebuild(const Params& P, const Particles& cur, cudaStream_t s) {
  launch_clear_grids(P, s);
  k_count_cells<<<sm_count() * 4, kAuxThreads, 0, s>>>(P, cur);
  launch_mid(P, cur, cur.desc, 0, s);   // ovf_count == 0: plain scan; n_next = n; no column scan (no tile rows yet)
  launch_deposit(P, cur, &P.st->n, s);
  launch_field(P, 0, s);  // commits n = n_next, leaves the step counter alone
  return 5;
}

}  // namespace bit1
