// The general path of one timestep: the same step as step_kernels.cu for inputs the banded single-scatter arranger
// cannot take -- a side list (far movers + births) longer than its capacity, i.e. a plasma so hot, so sparse or so
// violently accelerated that a sizeable fraction of the particles leaves its tile's sort window in one step.  It is
// SURVEY 8(d)'s "V0" written out: advance every particle in place, append the births behind the live slots in
// (parent, kind) order, stable radix sort of (new cell, slot) over the whole store, gather, deposit, field solve
// (SURVEY 8(c) "G .. P"; PAPER.md:111 mover then arranger).  Same arithmetic (advance()), same result bit for bit;
// about ten times the traffic of the fast path, so api.cu only comes here for steps that stalled
// (DevState::stalled) and for a bounded burst after repeated stalls.
#include "advance.cuh"
#include "aux_kernels.h"
#include "step_kernels.h"

namespace bit1 {

constexpr int kGenThreads = 256;

// births of one particle in kind order, without side effects
struct SinkCount {
  static constexpr bool kCounters = false, kBirths = true;
  unsigned mask;
  __device__ __forceinline__ void birth(const Params&, int kind, int, double, double, double, double, int) {
    mask |= 1u << kind;
  }
};
// as SinkStore, with the counters and diagnostics of the step (a step that pass A has not already counted)
struct SinkStoreCounted : SinkStore {
  static constexpr bool kCounters = true, kBirths = true;
};

// scratch words (unsigned) in front of the per-chunk counts
constexpr int kGenTotal = 0;   // births of the step
constexpr int kGenHeader = 64;

__global__ void k_gen_begin(const __grid_constant__ Params P, unsigned* hdr) {
  DevState* st = P.st;
  st->stalled = 0u;
  st->ovf_count = 0u;
  st->ovf_valid = 0u;
  st->general_steps += 1ull;
  hdr[kGenTotal] = 0u;
}

// pass 1: how many births does every chunk of kGenThreads consecutive particles produce
__global__ void __launch_bounds__(kGenThreads) k_gen_count(const __grid_constant__ Params P, Particles cur,
                                                           unsigned* hdr, unsigned* chunk_births) {
  __shared__ unsigned s_tot;
  const unsigned n = P.st->n;
  const unsigned long long step = P.st->step;
  const unsigned nchunks = (n + kGenThreads - 1) / kGenThreads;
  for (unsigned ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
    if (threadIdx.x == 0) s_tot = 0;
    __syncthreads();
    const unsigned i = ch * kGenThreads + threadIdx.x;
    if (i < n) {
      double x = cur.x[i], vx = cur.vx[i], vy = cur.vy[i], vz = cur.vz[i];
      int c = cell_of(P, x);
      SinkCount sink;
      sink.mask = 0;
      advance<SinkCount>(P, P.sp, step, P.E, (int)cur.sp[i], cur.pid[i], sink, x, vx, vy, vz, c);
      if (sink.mask) atomicAdd(&s_tot, (unsigned)__popc(sink.mask));
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      chunk_births[ch] = s_tot;
      if (s_tot) atomicAdd(&hdr[kGenTotal], s_tot);
    }
    __syncthreads();
  }
}

// pass 2: the step itself, in place; keys[slot] = new cell (nc: dead, nc + 1: unused slot), vals[slot] = slot
template <class SINK>
__global__ void __launch_bounds__(kGenThreads) k_gen_push(const __grid_constant__ Params P, Particles cur,
                                                          const unsigned* hdr, const unsigned* chunk_base,
                                                          unsigned* keys, unsigned* vals) {
  __shared__ unsigned s_warp[kGenThreads / 32];
  DevState* st = P.st;
  const unsigned n = st->n;
  const unsigned long long step = st->step;
  const unsigned room = P.capacity > n ? P.capacity - n : 0u;
  const unsigned births = hdr[kGenTotal];
  const unsigned created = births < room ? births : room;
  const unsigned next_pid = st->next_pid;
  const unsigned nchunks = (n + kGenThreads - 1) / kGenThreads;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (unsigned ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
    const unsigned i = ch * kGenThreads + threadIdx.x;
    SINK sink;
    sink.mask = 0;
    if (i < n) {
      double x = cur.x[i], vx = cur.vx[i], vy = cur.vy[i], vz = cur.vz[i];
      int c = cell_of(P, x);
      advance<SINK>(P, P.sp, step, P.E, (int)cur.sp[i], cur.pid[i], sink, x, vx, vy, vz, c);
      if (c >= 0) { cur.x[i] = x; cur.vx[i] = vx; cur.vy[i] = vy; cur.vz[i] = vz; }
      keys[i] = c >= 0 ? (unsigned)c : (unsigned)P.nc;
      vals[i] = i;
    }
    // rank of this particle's first birth among the step's births: chunk base + births of earlier threads
    const unsigned mine = (unsigned)__popc(sink.mask);
    unsigned inc = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const unsigned t = __shfl_up_sync(0xffffffffu, inc, d);
      if (lane >= d) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    unsigned before = chunk_base[ch] + inc - mine;
    for (int w = 0; w < warp; ++w) before += s_warp[w];
    __syncthreads();
    if (mine) {
      unsigned r = before;
#pragma unroll
      for (int kind = 0; kind < 4; ++kind) {
        if (!((sink.mask >> kind) & 1u)) continue;
        if (r < room) {   // reading R-W: the first capacity - N births in (parent, kind) order exist, the rest do not
          const unsigned slot = BIT1_CHECK(st, n + r, P.capacity);
          const BirthRec& b = sink.rec[kind];
          cur.x[slot] = b.x; cur.vx[slot] = b.vx; cur.vy[slot] = b.vy; cur.vz[slot] = b.vz;
          cur.pid[slot] = next_pid + r;
          cur.sp[slot] = (unsigned char)b.sp;
          keys[slot] = (unsigned)b.cell;
          vals[slot] = slot;
        }
        ++r;
      }
    }
  }
  // slots behind the births: sorted behind everything
  for (size_t s = (size_t)n + created + (size_t)blockIdx.x * kGenThreads + threadIdx.x; s < (size_t)P.capacity;
       s += (size_t)gridDim.x * kGenThreads) {
    keys[s] = (unsigned)P.nc + 1u;
    vals[s] = (unsigned)s;
  }
}

// after k_gen_push (its own launch, so that every CTA of the push has read next_pid): the births' bookkeeping
__global__ void k_gen_commit_births(const __grid_constant__ Params P, const unsigned* hdr) {
  DevState* st = P.st;
  const unsigned n = st->n;
  const unsigned room = P.capacity > n ? P.capacity - n : 0u;
  const unsigned births = hdr[kGenTotal];
  const unsigned created = births < room ? births : room;
  const unsigned next_pid = st->next_pid;
  if (next_pid + created < next_pid) st->flags |= kFlagPidWrap;
  st->next_pid = next_pid + created;
  st->births += created;
  if (births > room) st->flags |= kFlagCapacity;
}

// counts per cell from the sorted keys (dead and unused slots carry keys >= nc)
__global__ void __launch_bounds__(kGenThreads) k_gen_count_cells(const __grid_constant__ Params P,
                                                                 const unsigned* keys) {
  const size_t cap = P.capacity, stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i0 = (size_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u); i0 < cap; i0 += stride) {
    const size_t i = i0 + (threadIdx.x & 31u);
    const unsigned k = i < cap ? keys[i] : 0xffffffffu;
    const bool live = k < (unsigned)P.nc;
    const unsigned m = __match_any_sync(0xffffffffu, live ? k : (0x80000000u | (threadIdx.x & 31u)));
    if (live && (int)(threadIdx.x & 31u) == __ffs(m) - 1) atomicAdd(&P.cell_count[k], __popc(m));
  }
}

// the live particles in sorted order: nxt[i] = cur[perm[i]], i < n_next (from k_mid's scan of the counts)
__global__ void __launch_bounds__(kGenThreads) k_gen_gather(const __grid_constant__ Params P, Particles cur,
                                                            Particles nxt, const unsigned* perm) {
  const unsigned n = P.st->n_next;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const unsigned j = BIT1_CHECK(P.st, perm[i], P.capacity);
    nxt.x[i] = cur.x[j]; nxt.vx[i] = cur.vx[j]; nxt.vy[i] = cur.vy[j]; nxt.vz[i] = cur.vz[j];
    nxt.pid[i] = cur.pid[j]; nxt.sp[i] = cur.sp[j];
  }
}

size_t general_scratch_bytes(unsigned capacity) {
  const size_t nch = ((size_t)capacity + kGenThreads - 1) / kGenThreads;
  const size_t counts = (kGenHeader + nch + nch / 4096 + 8) * 4;
  return ((counts + 255) & ~(size_t)255) + load_scratch_bytes(capacity);
}

// One timestep by the general path.  count_side_effects = 0: the step stalled after pass A had already counted its
// wall hits, events and diagnostics; 1: a step the fast path never saw.
int launch_general_step(const Params& P, const Particles& cur, const Particles& nxt, int count_side_effects,
                        void* scratch, cudaStream_t s) {
  const size_t nch = ((size_t)P.capacity + kGenThreads - 1) / kGenThreads;
  unsigned* hdr = reinterpret_cast<unsigned*>(scratch);
  unsigned* chunk = hdr + kGenHeader;
  const size_t counts = (kGenHeader + nch + nch / 4096 + 8) * 4;
  char* sort_scratch = static_cast<char*>(scratch) + ((counts + 255) & ~(size_t)255);
  unsigned* k0 = reinterpret_cast<unsigned*>(sort_scratch);
  unsigned* v0 = k0 + P.capacity;
  int launches = 0;
  const int g = sm_count() * 8;
  k_gen_begin<<<1, 1, 0, s>>>(P, hdr);
  k_gen_count<<<g, kGenThreads, 0, s>>>(P, cur, hdr, chunk);
  launches += 2;
  launches += launch_scan_u32(chunk, nch, chunk + nch, s);
  if (count_side_effects) k_gen_push<SinkStoreCounted><<<g, kGenThreads, 0, s>>>(P, cur, hdr, chunk, k0, v0);
  else k_gen_push<SinkStore><<<g, kGenThreads, 0, s>>>(P, cur, hdr, chunk, k0, v0);
  k_gen_commit_births<<<1, 1, 0, s>>>(P, hdr);
  launches += 2;
  int bits = 0;
  while ((1ll << bits) < (long long)P.nc + 2) ++bits;
  unsigned *ks = nullptr, *vs = nullptr;
  launches += launch_radix_sort_u32(P.capacity, P.capacity, bits, sort_scratch, s, &ks, &vs);
  launches += launch_clear_grids(P, s);
  k_gen_count_cells<<<g, kGenThreads, 0, s>>>(P, ks);
  launches += 1;
  launches += launch_mid(P, cur, nxt.desc, 0, s);   // scan of the counts -> cell_start, n_next, tile descriptors
  k_gen_gather<<<g, kGenThreads, 0, s>>>(P, cur, nxt, vs);
  launches += 1;
  launches += launch_deposit(P, nxt, &P.st->n_next, s);
  launches += launch_field(P, 1, s);
  launches += launch_average(P, s);
  return launches;
}

}  // namespace bit1
