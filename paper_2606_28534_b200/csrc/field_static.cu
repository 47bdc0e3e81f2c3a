// bit1_field_solve_static (include/bit1.h): the field solve of one timestep -- optional 1-2-1 smoothing of rho, then the
// exact integer-scan Poisson solve for phi and E (PAPER.md:33 step (iii) "field solver" and "density smoothing";
// SURVEY 8(a) row a6, 8(f) NEXT-1) -- for callers that cannot allocate device memory.
//
// Who that is.  Everything else in libbit1 works out of a device workspace the caller allocates and hands to bit1_create.
// Some callers have nowhere to get one: code that runs inside a host program whose GPU memory is handed out by that
// program's own pool and is not open to plug-ins; a callback that runs while the host's allocator is locked or between
// the host's own cudaMalloc-free phases; a process whose memory budget was fixed at start-up.  They hold the arrays they
// were given (rho in, phi and E out) and nothing else, and cudaMalloc is either forbidden to them or would synchronise
// the whole device in the middle of somebody else's pipeline.
//
// What they get.  k_field_static is a variant of k_field (step_kernels.cu).  k_field keeps three things in the caller's
// workspace beyond its inputs and outputs: the per-CTA partial sums the CTAs exchange at the grid barriers and the two
// int64 arrays the smoothing passes alternate between.  Here the same three live in g_field_scratch below, a file-scope
// __device__ array that is part of the library image: the CUDA runtime places it on every GPU that loads libbit1 and
// frees it at process exit, so no call of ours (cudaMalloc, cudaFree, cudaMallocAsync, a library routine that allocates
// behind one's back) is needed -- and none is made.  The price is a fixed ceiling, BIT1_FIELD_STATIC_MAX_CELLS cells,
// and about 16 MiB of device memory per GPU whether or not the entry point is ever called.
//
// The arithmetic is k_field's, typed again for plain arguments (no Params / DevState): the results are the same bits.
#include <cooperative_groups.h>
#include <stdint.h>

#include <mutex>

#include "../../include/bit1.h"
#include "block_ops.cuh"

namespace cg = cooperative_groups;

namespace {

using bit1::block_exclusive_scan;
using bit1::block_sum;
using bit1::i128;

constexpr int kThreads = 256;        // k_field's geometry: the CTA count must not exceed the thread count (carry scan)
constexpr int kItems = 4;
constexpr int kMaxGrid = kThreads;
constexpr int kOneCtaNodes = 1025;   // up to here one CTA does the whole solve with CTA barriers only
constexpr int kMaxNodes = BIT1_FIELD_STATIC_MAX_CELLS + 1;   // bounded grids have nc + 1 nodes

constexpr double kEps0 = 8.8541878128e-12;     // F/m
constexpr double kTwoM40 = 9.094947017729282379150390625e-13;   // the fixed-point unit of rho, 2^-40 C

// Layout of the built-in scratch.  Every byte a call reads was written earlier in the same call (the partial sums of
// CTAs 0..G-1, nodes 0..ng-1 of the smoothing arrays), so nothing has to be cleared between calls; what the previous
// call left behind is simply overwritten or never looked at.
constexpr size_t kPartBytes = 4 * (size_t)kMaxGrid * sizeof(i128);                        // [4][kMaxGrid]: tot, wsum, A, C
constexpr size_t kRowBytes = (((size_t)kMaxNodes * sizeof(long long)) + 255) / 256 * 256;  // one smoothing array
constexpr size_t kScratchBytes = kPartBytes + 2 * kRowBytes;

// In host code the name below is only a handle for cudaGetSymbolAddress -- it is NOT a device address; handing
// `g_field_scratch` itself to a kernel would make the kernel read host memory (or fault).  device_setup() asks the
// runtime for the real address on the current device and the launch passes that.
static __device__ __align__(256) unsigned char g_field_scratch[kScratchBytes];

struct FieldStaticArgs {
  const long long* rho;   // ng, input
  double* phi;            // nc + 1, output
  double* E;              // nc + 1, output
  long long* tmp_s;       // scratch: the smoothing pass that the solve reads
  long long* tmp_t;       // scratch: the other one
  i128* part;             // scratch: [4][kMaxGrid]
  int nc, ng, bc, smooth;
  double Kphi, KE;
};

// magnitude first, then the sign: sign(n) * ((double)hi(|n|) * 2^64 + (double)lo(|n|))  (reading R-dbl)
__device__ __forceinline__ double to_double(i128 n) {
  const bool neg = n < 0;
  const unsigned __int128 a = neg ? (unsigned __int128)0 - (unsigned __int128)n : (unsigned __int128)n;
  const unsigned long long hi = (unsigned long long)(a >> 64), lo = (unsigned long long)a;
  const double d = (double)hi * 18446744073709551616.0 + (double)lo;
  return neg ? -d : d;
}

__device__ __forceinline__ void all_ctas_sync(cg::grid_group& grid) {
  if (gridDim.x == 1) __syncthreads();
  else { __threadfence(); grid.sync(); }
}

// Elements j in [j_lo, j_hi] of 1..jmax, in chunks of kThreads * kItems.  On entry carryS = S_{j_lo-1}, carryT = T_{j_lo}.
// APPLY = false returns A = sum of R_j and C = sum of the local inclusive prefixes; APPLY = true writes phi_j and E_j.
template <bool APPLY>
__device__ void solve_range(const FieldStaticArgs& a, const long long* __restrict__ R_in, double Kphi, double KE, int j_lo,
                            int j_hi, i128 tot, i128 Tn, i128 carryS, i128 carryT, i128* s_warp, i128* outA,
                            i128* outC) {
  const int nc = a.nc, bc = a.bc;
  const i128 S0 = carryS;
  i128 accC = 0;
  for (int j0 = j_lo; j0 <= j_hi; j0 += kThreads * kItems) {
    const int jb = j0 + (int)threadIdx.x * kItems;
    i128 R[kItems], Sl[kItems];
    i128 run = 0;
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
      const int j = jb + k;
      i128 r = 0;
      if (j <= j_hi) r = bc ? (i128)R_in[j] : (i128)nc * (i128)R_in[j] - tot;
      R[k] = r;
      run += r;
      Sl[k] = run;
    }
    i128 chunkS;
    const i128 exS = carryS + block_exclusive_scan<i128>(run, s_warp, &chunkS);
    i128 tsumS = 0;
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
      const int j = jb + k;
      Sl[k] = exS + Sl[k];   // S_j
      if (j <= j_hi) tsumS += Sl[k];
    }
    i128 chunkSS;
    i128 T = carryT + block_exclusive_scan<i128>(tsumS, s_warp, &chunkSS);
    if (APPLY) {
#pragma unroll
      for (int k = 0; k < kItems; ++k) {
        const int j = jb + k;
        if (j <= j_hi) {
          const i128 Sj = Sl[k], Sm = Sl[k] - R[k];
          a.phi[j] = Kphi * to_double((i128)j * Tn - (i128)nc * T);
          if (bc) {
            if (j < nc) a.E[j] = KE * to_double((i128)nc * (Sm + Sj) - 2 * Tn);
            else a.E[nc] = KE * to_double(2 * (i128)nc * Sm - 2 * Tn + 2 * (i128)nc * (i128)R_in[nc]);
          } else {
            a.E[j] = KE * to_double((i128)nc * (Sm + Sj) - 2 * Tn);
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
    const int len = j_hi >= j_lo ? j_hi - j_lo + 1 : 0;
    *outA = carryS - S0;
    *outC = accC - (i128)len * S0;
  }
}

// Cooperative launch when gridDim.x > 1.  Phase A: smoothing passes into the scratch arrays, total charge and T_nc;
// phase B: every CTA sums its range; phase C: carries from the CTAs before it, then phi and E.
__global__ void __launch_bounds__(kThreads) k_field_static(const __grid_constant__ FieldStaticArgs a) {
  __shared__ i128 s_warp[33];
  cg::grid_group grid = cg::this_grid();
  const int nc = a.nc, ng = a.ng, bc = a.bc, smooth = a.smooth;
  const int G = gridDim.x, b = blockIdx.x;
  i128* part = a.part;
  const long long* R = a.rho;
  double Kphi = a.Kphi, KE = a.KE;
  if (smooth > 0) {
    const long long* in = a.rho;
    for (int k = 0; k < smooth; ++k) {
      long long* out = ((smooth - 1 - k) & 1) ? a.tmp_t : a.tmp_s;   // the last pass lands in tmp_s
      if (k > 0) all_ctas_sync(grid);                                // pass k reads what every CTA wrote in pass k - 1
      for (int j = b * kThreads + (int)threadIdx.x; j < ng; j += G * kThreads) {
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
    all_ctas_sync(grid);
    R = a.tmp_s;
    const double scale = 1.0 / (double)(1ll << (2 * smooth));   // each pass carries a factor 4: an exact power of two
    Kphi = Kphi * scale;
    KE = KE * scale;
  }
  i128 tot = 0, wsum = 0;
  for (int j = b * kThreads + (int)threadIdx.x; j < ng; j += G * kThreads) {
    const long long r = R[j];
    tot += (i128)r;
    if (j >= 1 && j <= nc - 1) wsum += (i128)(nc - j) * (i128)r;
  }
  tot = block_sum<i128>(tot, s_warp);
  wsum = block_sum<i128>(wsum, s_warp);
  if (G > 1) {
    if (threadIdx.x == 0) { part[b] = tot; part[kMaxGrid + b] = wsum; }
    all_ctas_sync(grid);
    tot = 0; wsum = 0;
    for (int i = threadIdx.x; i < G; i += kThreads) { tot += part[i]; wsum += part[kMaxGrid + i]; }
    tot = block_sum<i128>(tot, s_warp);
    wsum = block_sum<i128>(wsum, s_warp);
  }
  // periodic: R'_j = nc R_j - tot  =>  T_nc' = nc * wsum - tot * nc (nc - 1) / 2
  const i128 Tn = bc ? wsum : (i128)nc * wsum - tot * (((i128)nc * (i128)(nc - 1)) / 2);
  const int jmax = bc ? nc : nc - 1;
  const int unit = kThreads * kItems;
  int per = (jmax + G - 1) / G;
  per = ((per + unit - 1) / unit) * unit;
  const int j_lo = min(1 + b * per, jmax + 1), j_hi = min(j_lo + per - 1, jmax);
  i128 carryS = 0, carryT = 0, Send = 0;
  if (G > 1) {
    i128 A = 0, C = 0;
    solve_range<false>(a, R, Kphi, KE, j_lo, j_hi, tot, Tn, (i128)0, (i128)0, s_warp, &A, &C);
    if (threadIdx.x == 0) { part[2 * kMaxGrid + b] = A; part[3 * kMaxGrid + b] = C; }
    all_ctas_sync(grid);
    i128 myA = 0, myLen = 0, myC = 0;
    if ((int)threadIdx.x < G) {
      const int i = threadIdx.x;
      myA = part[2 * kMaxGrid + i];
      myC = part[3 * kMaxGrid + i];
      const int lo = min(1 + i * per, jmax + 1), hi = min(lo + per - 1, jmax);
      myLen = hi >= lo ? hi - lo + 1 : 0;
    }
    i128 dummy;
    const i128 Sbefore = block_exclusive_scan<i128>(myA, s_warp, &dummy);
    const i128 term = ((int)threadIdx.x < b) ? myLen * Sbefore + myC : (i128)0;
    carryT = block_sum<i128>(term, s_warp);
    carryS = block_sum<i128>(((int)threadIdx.x < b) ? myA : (i128)0, s_warp);
    Send = block_sum<i128>(myA, s_warp);   // S_jmax
  } else if (!bc) {
    Send = tot - (i128)nc * (i128)R[0];    // sum_{j=1}^{nc-1} (nc R_j - tot)
  }
  if (b == 0 && threadIdx.x == 0) {
    a.phi[0] = Kphi * to_double((i128)0);
    if (bc) {
      a.E[0] = KE * to_double(-2 * Tn - 2 * (i128)nc * (i128)R[0]);
    } else {
      a.E[0] = KE * to_double((i128)nc * (Send + (i128)0) - 2 * Tn);
      a.E[nc] = a.E[0];
      a.phi[nc] = a.phi[0];
    }
  }
  solve_range<true>(a, R, Kphi, KE, j_lo, j_hi, tot, Tn, carryS, carryT, s_warp, nullptr, nullptr);
}

// Once per device: the device address of the built-in scratch and the SM count that bounds the cooperative grid.
struct DeviceSetup {
  bool done;
  unsigned char* scratch;
  int sms;
};
constexpr int kMaxDevices = 64;
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

// The device that is current for the calling thread must be the one the launch goes to.
cudaError_t device_setup(const DeviceSetup** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  DeviceSetup& s = g_setup[dev];
  if (!s.done) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_field_scratch);   // the name -> this device's copy of the array
    if (e != cudaSuccess) return e;
    if (p == nullptr || ((uintptr_t)p & 255u) != 0) return cudaErrorInvalidSymbol;
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    if (sms < 1) return cudaErrorInvalidDevice;
    s.scratch = static_cast<unsigned char*>(p);
    s.sms = sms;
    s.done = true;
  }
  *out = &s;
  return cudaSuccess;
}

}  // namespace

extern "C" bit1_status bit1_field_solve_static(const int64_t* rho_fixed, double* phi, double* E, int32_t nc, int32_t bc,
                                               double dx, double area, int32_t smoothing_passes, void* stream) {
  if (!rho_fixed || !phi || !E) return BIT1_ERR_INVALID_ARG;
  if (nc < 2 || (bc != 0 && bc != 1) || !(dx > 0.0) || !(area > 0.0)) return BIT1_ERR_INVALID_ARG;
  if (smoothing_passes < 0 || smoothing_passes > 8) return BIT1_ERR_INVALID_ARG;
  if (nc > BIT1_FIELD_STATIC_MAX_CELLS) return BIT1_ERR_STATIC_LIMIT;   // the built-in arrays end there
  const DeviceSetup* dev = nullptr;
  if (device_setup(&dev) != cudaSuccess) { cudaGetLastError(); return BIT1_ERR_CUDA; }

  FieldStaticArgs a;
  a.rho = reinterpret_cast<const long long*>(rho_fixed);
  a.phi = phi;
  a.E = E;
  a.part = reinterpret_cast<i128*>(dev->scratch);
  a.tmp_s = reinterpret_cast<long long*>(dev->scratch + kPartBytes);
  a.tmp_t = reinterpret_cast<long long*>(dev->scratch + kPartBytes + kRowBytes);
  a.nc = nc;
  a.ng = bc ? nc + 1 : nc;
  a.bc = bc;
  a.smooth = smoothing_passes;
  // the constants of bit1_create (api.cu), in the same order of operations
  a.Kphi = (kTwoM40 * dx) / ((area * kEps0) * (double)nc);
  a.KE = kTwoM40 / (((2.0 * (double)nc) * area) * kEps0);
  if (!bc) { a.Kphi = a.Kphi / (double)nc; a.KE = a.KE / (double)nc; }

  int g = 1;
  if (a.ng > kOneCtaNodes) {
    g = (a.ng + kThreads * kItems - 1) / (kThreads * kItems);
    const int cap = dev->sms < kMaxGrid ? dev->sms : kMaxGrid;   // every CTA resident at once, and G <= kThreads
    if (g > cap) g = cap;
  }
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  cudaError_t e;
  if (g == 1) {
    k_field_static<<<1, kThreads, 0, s>>>(a);
    e = cudaGetLastError();
  } else {
    void* args[] = {&a};
    e = cudaLaunchCooperativeKernel((const void*)k_field_static, dim3(g), dim3(kThreads), args, 0, s);
  }
  if (e != cudaSuccess) { cudaGetLastError(); return BIT1_ERR_CUDA; }
  return BIT1_OK;
}
