// Kernels off the per-step path: load (validate, cell index, general stable sort by cell), moments, export, and the
// cell-index fill (the store's cell array is cell_of(x) by construction and only materialised when asked for).
// The load-time sort is a multi-pass LSD radix sort (8-bit digits) on (cell, original index); it is the
// general counterpart of the banded single-scatter sort of the step kernels and is not timed.
#include "block_ops.cuh"
#include "aux_kernels.h"
#include "device_math.cuh"
#include "step_kernels.h"

namespace bit1 {

// grid of the grid-stride kernels below: 8 CTAs of 256 threads per SM of the current device
static int aux_grid() { return sm_count() * 8; }

// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_load_prepare(const __grid_constant__ Params P, Particles in, unsigned n,
                                                      int have_pid, unsigned* keys, unsigned* vals) {
  unsigned maxpid = 0;
  bool bad = false;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double x = in.x[i];
    const int s = in.sp[i];
    if (!(x >= 0.0 && x < P.L) || s >= P.ns) bad = true;
    const int c = cell_of(P, x);
    if (!have_pid) in.pid[i] = (unsigned)i;
    const unsigned pid = in.pid[i];
    maxpid = max(maxpid, pid + 1u);
    keys[i] = (unsigned)c;
    vals[i] = (unsigned)i;
  }
  for (int o = 16; o > 0; o >>= 1) maxpid = max(maxpid, __shfl_xor_sync(0xffffffffu, maxpid, o));
  if ((threadIdx.x & 31) == 0 && maxpid) atomicMax(&P.st->next_pid, maxpid);
  if (bad) atomicOr(&P.st->load_error, 1u);
}

// bit1_load_particles: every position inside [0, L), every species tag known -- checked before anything indexes by them
__global__ void __launch_bounds__(256) k_load_validate(const __grid_constant__ Params P, Particles in, unsigned n) {
  bool bad = false;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double x = in.x[i];
    if (!(x >= 0.0 && x < P.L) || (int)in.sp[i] >= P.ns) bad = true;
  }
  if (bad) atomicOr(&P.st->load_error, 1u);
}
int launch_load_validate(const Params& P, const Particles& in, unsigned n, cudaStream_t s) {
  if (n == 0) return 0;
  k_load_validate<<<aux_grid(), 256, 0, s>>>(P, in, n);
  return 1;
}
// bit1_restart: the same, and the positions must be in cell order (the blob's body is data from outside)
__global__ void __launch_bounds__(256) k_state_validate(const __grid_constant__ Params P, Particles p, unsigned n) {
  bool bad = false;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double x = p.x[i];
    if (!(x >= 0.0 && x < P.L) || (int)p.sp[i] >= P.ns) bad = true;
    else if (i > 0 && cell_of(P, p.x[i - 1]) > cell_of(P, x)) bad = true;
  }
  if (bad) atomicOr(&P.st->load_error, 1u);
}
int launch_state_validate(const Params& P, const Particles& p, unsigned n, cudaStream_t s) {
  if (n == 0) return 0;
  k_state_validate<<<aux_grid(), 256, 0, s>>>(P, p, n);
  return 1;
}

constexpr int kRadixItems = 8;
constexpr int kRadixChunk = 256 * kRadixItems;

__global__ void __launch_bounds__(256) k_radix_hist(const unsigned* keys, unsigned n, int shift, unsigned* blockhist,
                                                    unsigned nblocks) {
  __shared__ unsigned h[256];
  h[threadIdx.x] = 0;
  __syncthreads();
  const unsigned base = blockIdx.x * kRadixChunk;
  for (int r = 0; r < kRadixItems; ++r) {
    const unsigned i = base + r * 256 + threadIdx.x;
    if (i < n) atomicAdd(&h[(keys[i] >> shift) & 255u], 1u);
  }
  __syncthreads();
  blockhist[(size_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

// exclusive scan of a uint array by one CTA of 1024 threads (in place)
__global__ void __launch_bounds__(1024) k_scan_u32(unsigned* a, size_t n) {
  __shared__ unsigned s_warp[33];
  unsigned carry = 0;
  for (size_t i0 = 0; i0 < n; i0 += 4096) {
    const size_t i = i0 + (size_t)threadIdx.x * 4;
    unsigned v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = i + k < n ? a[i + k] : 0u;
    unsigned chunk;
    unsigned ex = carry + block_exclusive_scan<unsigned>(v[0] + v[1] + v[2] + v[3], s_warp, &chunk);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (i + k < n) a[i + k] = ex;
      ex += v[k];
    }
    carry += chunk;
  }
}

// Exclusive scan of a long uint array on many CTAs: sums of 4096-element chunks, scan of the sums (one CTA), then
// every chunk scanned with its carry.  (The one-CTA k_scan_u32 took 12 ms per radix pass at 2e8 particles.)
constexpr int kScanChunk = 4096;
__global__ void __launch_bounds__(1024) k_scan_chunk_sums(const unsigned* a, size_t n, unsigned* sums) {
  __shared__ unsigned s_warp[33];
  const size_t i = (size_t)blockIdx.x * kScanChunk + (size_t)threadIdx.x * 4;
  unsigned t = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) t += i + k < n ? a[i + k] : 0u;
  t = block_sum<unsigned>(t, s_warp);
  if (threadIdx.x == 0) sums[blockIdx.x] = t;
}
__global__ void __launch_bounds__(1024) k_scan_chunks(unsigned* a, size_t n, const unsigned* carry_in) {
  __shared__ unsigned s_warp[33];
  const size_t i = (size_t)blockIdx.x * kScanChunk + (size_t)threadIdx.x * 4;
  unsigned v[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) v[k] = i + k < n ? a[i + k] : 0u;
  unsigned chunk;
  unsigned ex = carry_in[blockIdx.x] + block_exclusive_scan<unsigned>(v[0] + v[1] + v[2] + v[3], s_warp, &chunk);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (i + k < n) a[i + k] = ex;
    ex += v[k];
  }
}
// tmp: (n / kScanChunk + 1) words
int launch_scan_u32(unsigned* a, size_t n, unsigned* tmp, cudaStream_t s) {
  if (n <= (size_t)4 * kScanChunk) {
    k_scan_u32<<<1, 1024, 0, s>>>(a, n);
    return 1;
  }
  const unsigned nb = (unsigned)((n + kScanChunk - 1) / kScanChunk);
  k_scan_chunk_sums<<<nb, 1024, 0, s>>>(a, n, tmp);
  k_scan_u32<<<1, 1024, 0, s>>>(tmp, nb);
  k_scan_chunks<<<nb, 1024, 0, s>>>(a, n, tmp);
  return 3;
}

__global__ void __launch_bounds__(256) k_radix_scatter(const unsigned* keys, const unsigned* vals, unsigned n, int shift,
                                                       const unsigned* blockhist, unsigned nblocks, unsigned* keys_out,
                                                       unsigned* vals_out) {
  __shared__ unsigned s_cnt[256 * 8];  // [digit][warp]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = lanemask_lt();
  for (int k = threadIdx.x; k < 256 * 8; k += 256) s_cnt[k] = 0;
  __syncthreads();
  const unsigned base = blockIdx.x * kRadixChunk + warp * (32 * kRadixItems);
  unsigned key[kRadixItems], val[kRadixItems], rank[kRadixItems];
#pragma unroll
  for (int r = 0; r < kRadixItems; ++r) {
    const unsigned i = base + r * 32 + lane;
    const bool have = i < n;
    key[r] = have ? keys[i] : 0u;
    val[r] = have ? vals[i] : 0u;
    const unsigned d = have ? ((key[r] >> shift) & 255u) : (0x80000000u | (unsigned)lane);
    const unsigned m = __match_any_sync(0xffffffffu, d);
    const int leader = __ffs(m) - 1;
    unsigned old = 0;
    if (have && lane == leader) {
      old = s_cnt[d * 8 + warp];
      s_cnt[d * 8 + warp] = old + (unsigned)__popc(m);
    }
    old = __shfl_sync(0xffffffffu, old, leader);
    rank[r] = have ? old + (unsigned)__popc(m & lt) : 0xffffffffu;
    __syncwarp();
  }
  __syncthreads();
  {
    const unsigned d = threadIdx.x;
    unsigned run = blockhist[(size_t)d * nblocks + blockIdx.x];
#pragma unroll
    for (int w = 0; w < 8; ++w) {
      const unsigned t = s_cnt[d * 8 + w];
      s_cnt[d * 8 + w] = run;
      run += t;
    }
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < kRadixItems; ++r) {
    if (rank[r] != 0xffffffffu) {
      const unsigned d = (key[r] >> shift) & 255u;
      const unsigned dst = s_cnt[d * 8 + warp] + rank[r];
      keys_out[dst] = key[r];
      vals_out[dst] = val[r];
    }
  }
}

// out[i] = in[perm[i]], split so that each velocity array can follow its own host-to-device copy: positions, ids and
// species (on the device before the sort starts) in one kernel, one kernel per velocity component
__global__ void __launch_bounds__(256) k_gather_keys(Particles in, Particles out, const unsigned* perm, unsigned n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const unsigned j = perm[i];
    out.x[i] = in.x[j]; out.pid[i] = in.pid[j]; out.sp[i] = in.sp[j];
  }
}
__global__ void __launch_bounds__(256) k_gather_f64(const double* __restrict__ in, double* __restrict__ out,
                                                    const unsigned* __restrict__ perm, unsigned n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    out[i] = in[perm[i]];
}

// Stable LSD radix sort (8-bit digits over key bits [0, bits)) of n (key, value) pairs of 32-bit words.
// scratch: [k0 | v0 | k1 | v1] of `stride` words each, then the per-block digit counts; the input pairs are in
// (k0, v0); *keys / *vals say which pair of arrays holds the result.
int launch_radix_sort_u32(unsigned n, unsigned stride, int bits, void* scratch, cudaStream_t s, unsigned** keys,
                          unsigned** vals) {
  unsigned* k0 = reinterpret_cast<unsigned*>(scratch);
  unsigned* v0 = k0 + stride;
  unsigned* k1 = v0 + stride;
  unsigned* v1 = k1 + stride;
  unsigned* bh = v1 + stride;
  int launches = 0;
  const unsigned nblocks = (n + kRadixChunk - 1) / kRadixChunk;
  for (int shift = 0; shift < bits && n > 0; shift += 8) {
    k_radix_hist<<<nblocks, 256, 0, s>>>(k0, n, shift, bh, nblocks);
    launches += launch_scan_u32(bh, (size_t)256 * nblocks, bh + (size_t)256 * nblocks, s);
    k_radix_scatter<<<nblocks, 256, 0, s>>>(k0, v0, n, shift, bh, nblocks, k1, v1);
    launches += 2;
    unsigned* t = k0; k0 = k1; k1 = t;
    t = v0; v0 = v1; v1 = t;
  }
  *keys = k0;
  *vals = v0;
  return launches;
}

int launch_load_sort(const Params& P, const Particles& in, const Particles& out, unsigned n, int have_pid,
                     void* scratch, cudaStream_t s, const cudaEvent_t* velocity_ready) {
  if (n == 0) return 0;
  int launches = 0;
  unsigned* k0 = reinterpret_cast<unsigned*>(scratch);
  unsigned* v0 = k0 + P.capacity;
  k_load_prepare<<<aux_grid(), 256, 0, s>>>(P, in, n, have_pid, k0, v0);
  ++launches;
  int bits = 0;
  while ((1ll << bits) < (long long)P.nc) ++bits;
  unsigned *ks = nullptr, *vs = nullptr;
  launches += launch_radix_sort_u32(n, P.capacity, bits, scratch, s, &ks, &vs);
  k_gather_keys<<<aux_grid(), 256, 0, s>>>(in, out, vs, n);
  // the velocity arrays arrive on another stream, one event each: a component is gathered as soon as it has landed
  const double* vin[3] = {in.vx, in.vy, in.vz};
  double* vout[3] = {out.vx, out.vy, out.vz};
  for (int k = 0; k < 3; ++k) {
    if (velocity_ready) cudaStreamWaitEvent(s, velocity_ready[k], 0);
    k_gather_f64<<<aux_grid(), 256, 0, s>>>(vin[k], vout[k], vs, n);
  }
  return launches + 4;
}

size_t load_scratch_bytes(unsigned capacity) {
  const size_t nblocks = ((size_t)capacity + kRadixChunk - 1) / kRadixChunk;
  return (size_t)capacity * 16 + nblocks * 256 * 4 + (nblocks * 256 / kScanChunk + 2) * 4 + 1024;
}

// ---------------------------------------------------------------------------------------------
// Moments: fixed-shape reduction, so the result is deterministic run to run.
constexpr int kMomBlocks = 1024;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(256) k_moments_partial(const __grid_constant__ Params P, Particles cur,
                                                         double* partial /* [blocks][ns][3] */) {
  __shared__ double s_red[8][kMaxSpecies * 3];
  const unsigned n = P.st->n;
  double acc[kMaxSpecies * 3];
#pragma unroll
  for (int k = 0; k < kMaxSpecies * 3; ++k) acc[k] = 0.0;
  const size_t per = ((size_t)n + gridDim.x - 1) / gridDim.x;
  const size_t lo = per * blockIdx.x, hi = min((size_t)n, lo + per);
  for (size_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
    const int s = cur.sp[i];
    const double vx = cur.vx[i], vy = cur.vy[i], vz = cur.vz[i];
    const double v2 = (vx * vx + vy * vy) + vz * vz;
#pragma unroll
    for (int k = 0; k < kMaxSpecies; ++k) {
      if (k == s) { acc[k * 3] += 1.0; acc[k * 3 + 1] += v2; acc[k * 3 + 2] += vx; }
    }
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int k = 0; k < P.ns * 3; ++k) {
    const double v = warp_sum(acc[k]);
    if (lane == 0) s_red[warp][k] = v;
  }
  __syncthreads();
  if ((int)threadIdx.x < P.ns * 3) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += s_red[w][threadIdx.x];
    partial[(size_t)blockIdx.x * (kMaxSpecies * 3) + threadIdx.x] = t;
  }
}

__global__ void __launch_bounds__(1024) k_moments_final(const __grid_constant__ Params P, const double* partial,
                                                        int nblocks, double* out /* [ns][3] then field */) {
  __shared__ double s_red[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int k = 0; k < P.ns * 3; ++k) {
    double v = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) v += partial[(size_t)b * (kMaxSpecies * 3) + k];
    v = warp_sum(v);
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    if (warp == 0) {
      double t = s_red[lane];
      t = warp_sum(t);
      if (lane == 0) out[k] = t;
    }
    __syncthreads();
  }
  // field energy sum g_j E_j^2
  double v = 0.0;
  for (int j = threadIdx.x; j < P.ng; j += blockDim.x) {
    const double g = (P.bc && (j == 0 || j == P.nc)) ? 0.5 : 1.0;
    const double e = P.E[j];
    v += g * (e * e);
  }
  v = warp_sum(v);
  if (lane == 0) s_red[warp] = v;
  __syncthreads();
  if (warp == 0) {
    double t = warp_sum(s_red[lane]);
    if (lane == 0) out[kMaxSpecies * 3] = t;
  }
}

// cell[i] = cell_of(x[i]) for the live particles (bit1_get_particles; a step never reads or writes the cell array)
__global__ void __launch_bounds__(256) k_fill_cells(const __grid_constant__ Params P, Particles cur) {
  const unsigned n = P.st->n;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    cur.cell[i] = cell_of(P, cur.x[i]);
}
int launch_fill_cells(const Params& P, const Particles& cur, cudaStream_t s) {
  k_fill_cells<<<aux_grid(), 256, 0, s>>>(P, cur);
  return 1;
}

#ifdef BIT1_CHECKED
__global__ void k_check_selftest(const __grid_constant__ Params P, int* sink) {
  int table[3] = {1, 2, 3};
  sink[0] = table[BIT1_CHECK(P.st, 5 + (int)threadIdx.x, 3)];   // out of range: caught, redirected to entry 0
}
void launch_check_selftest(const Params& P, cudaStream_t s) { k_check_selftest<<<1, 1, 0, s>>>(P, P.scan_part); }
#endif

int launch_moments(const Params& P, const Particles& cur, double* partial, double* out, cudaStream_t s) {
  k_moments_partial<<<kMomBlocks, 256, 0, s>>>(P, cur, partial);
  k_moments_final<<<1, 1024, 0, s>>>(P, partial, kMomBlocks, out);
  return 2;
}
size_t moments_scratch_bytes() { return ((size_t)kMomBlocks + 2) * kMaxSpecies * 3 * 8 + 256; }

}  // namespace bit1

// ---------------------------------------------------------------------------------------------
// Export of one species in the paper's checkpoint layout (per species, a counts-per-cell vector, then the
// position and velocity records in that order).  The store is sorted by cell, so the records of one
// species in cell order are a stable compaction: count per 1024-particle chunk, exclusive scan, scatter.
namespace bit1 {
constexpr int kExpChunk = 1024;

__global__ void __launch_bounds__(256) k_export_count(const __grid_constant__ Params P, Particles cur, int species,
                                                      unsigned* chunk_cnt, int* cell_cnt, unsigned long long* total) {
  __shared__ unsigned s_cnt;
  const unsigned n = P.st->n;
  const unsigned nchunks = (n + kExpChunk - 1) / kExpChunk;
  for (unsigned ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    unsigned mine = 0;
    for (int r = 0; r < kExpChunk / 256; ++r) {
      const unsigned i = ch * kExpChunk + r * 256 + threadIdx.x;
      const bool hit = i < n && cur.sp[i] == (unsigned char)species;
      // neighbours mostly share the cell: one atomic per run of the warp
      const unsigned key = hit ? (unsigned)cell_of(P, cur.x[i]) : 0xffffffffu - (threadIdx.x & 31);
      const unsigned m = __match_any_sync(0xffffffffu, key);
      if (hit) {
        mine++;
        if ((int)(threadIdx.x & 31) == __ffs(m) - 1) atomicAdd(&cell_cnt[key], __popc(m));
      }
    }
    if (mine) atomicAdd(&s_cnt, mine);
    __syncthreads();
    if (threadIdx.x == 0) {
      chunk_cnt[ch] = s_cnt;
      if (s_cnt) atomicAdd(total, (unsigned long long)s_cnt);
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(256) k_export_scatter(const __grid_constant__ Params P, Particles cur, Particles out,
                                                        int species, const unsigned* chunk_off) {
  __shared__ unsigned s_warp[8];
  __shared__ unsigned s_base;
  const unsigned n = P.st->n;
  const unsigned nchunks = (n + kExpChunk - 1) / kExpChunk;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (unsigned ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
    if (threadIdx.x == 0) s_base = chunk_off[ch];
    __syncthreads();
    for (int r = 0; r < kExpChunk / 256; ++r) {
      const unsigned i = ch * kExpChunk + r * 256 + threadIdx.x;
      const bool hit = i < n && cur.sp[i] == (unsigned char)species;
      const unsigned b = __ballot_sync(0xffffffffu, hit);
      if (lane == 0) s_warp[warp] = __popc(b);
      __syncthreads();
      unsigned before = 0, tot = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) {
        const unsigned c = s_warp[w];
        if (w < warp) before += c;
        tot += c;
      }
      if (hit) {
        const unsigned d = s_base + before + __popc(b & ((1u << lane) - 1u));
        out.x[d] = cur.x[i]; out.vx[d] = cur.vx[i]; out.vy[d] = cur.vy[i]; out.vz[d] = cur.vz[i];
        out.pid[d] = cur.pid[i];
      }
      __syncthreads();
      if (threadIdx.x == 0) s_base += tot;
      __syncthreads();
    }
  }
}

// scratch: [total u64 | pad to 256][cell_cnt int[nc]][chunk_cnt unsigned[nchunks]]
size_t export_scratch_bytes(int nc, unsigned capacity) {
  const size_t nch = ((size_t)capacity + kExpChunk - 1) / kExpChunk;
  return 256 + (((size_t)nc * 4 + 255) & ~(size_t)255) + (nch + nch / 4096 + 2) * 4 + 256;
}

int launch_export_count(const Params& P, const Particles& cur, int species, unsigned capacity, void* scratch,
                        cudaStream_t s) {
  char* b = static_cast<char*>(scratch);
  unsigned long long* total = reinterpret_cast<unsigned long long*>(b);
  int* cell_cnt = reinterpret_cast<int*>(b + 256);
  unsigned* chunk_cnt = reinterpret_cast<unsigned*>(b + 256 + (((size_t)P.nc * 4 + 255) & ~(size_t)255));
  const size_t nchunks_max = ((size_t)capacity + kExpChunk - 1) / kExpChunk;
  cudaMemsetAsync(b, 0, 256 + (((size_t)P.nc * 4 + 255) & ~(size_t)255) + nchunks_max * 4, s);
  k_export_count<<<aux_grid(), 256, 0, s>>>(P, cur, species, chunk_cnt, cell_cnt, total);
  return 1 + launch_scan_u32(chunk_cnt, nchunks_max, chunk_cnt + nchunks_max, s);
}

int launch_export_scatter(const Params& P, const Particles& cur, const Particles& out, int species, void* scratch,
                          cudaStream_t s) {
  char* b = static_cast<char*>(scratch);
  const unsigned* chunk_off = reinterpret_cast<const unsigned*>(b + 256 + (((size_t)P.nc * 4 + 255) & ~(size_t)255));
  k_export_scatter<<<aux_grid(), 256, 0, s>>>(P, cur, out, species, chunk_off);
  return 1;
}
}  // namespace bit1
