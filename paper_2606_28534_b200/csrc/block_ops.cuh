// CTA-wide exclusive scan and sum of one value per thread (int, unsigned, 128-bit integers), used by the scan
// kernels of step_kernels.cu (cell counts, Poisson prefix sums) and aux_kernels.cu (radix-sort offsets).  Two levels of
// warp shuffles with one word of shared memory per warp; every thread of the CTA must call, blockDim.x a multiple of
// 32 and at most 1024.  The caller supplies s_warp[33] of the value type.
#pragma once
#include <cuda_runtime.h>

namespace bit1 {

typedef __int128 i128;

template <class T>
__device__ __forceinline__ T shfl_up_t(T v, int d) { return __shfl_up_sync(0xffffffffu, v, d); }
template <class T>
__device__ __forceinline__ T shfl_xor_t(T v, int d) { return __shfl_xor_sync(0xffffffffu, v, d); }
template <>
__device__ __forceinline__ i128 shfl_up_t<i128>(i128 v, int d) {
  unsigned long long lo = (unsigned long long)v, hi = (unsigned long long)((unsigned __int128)v >> 64);
  lo = __shfl_up_sync(0xffffffffu, lo, d);
  hi = __shfl_up_sync(0xffffffffu, hi, d);
  return (i128)(((unsigned __int128)hi << 64) | (unsigned __int128)lo);
}
template <>
__device__ __forceinline__ i128 shfl_xor_t<i128>(i128 v, int d) {
  unsigned long long lo = (unsigned long long)v, hi = (unsigned long long)((unsigned __int128)v >> 64);
  lo = __shfl_xor_sync(0xffffffffu, lo, d);
  hi = __shfl_xor_sync(0xffffffffu, hi, d);
  return (i128)(((unsigned __int128)hi << 64) | (unsigned __int128)lo);
}

// exclusive scan over the CTA; *total = sum over the CTA.  Ends with a CTA barrier: s_warp may be reused at once.
template <class T>
__device__ T block_exclusive_scan(T v, T* s_warp, T* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  T inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const T t = shfl_up_t<T>(inc, d);
    if (lane >= d) inc += t;
  }
  if (lane == 31) s_warp[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    const T w = lane < (int)(blockDim.x >> 5) ? s_warp[lane] : (T)0;
    T winc = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const T t = shfl_up_t<T>(winc, d);
      if (lane >= d) winc += t;
    }
    s_warp[lane] = winc - w;
    if (lane == 31) s_warp[32] = winc;
  }
  __syncthreads();
  const T res = s_warp[warp] + inc - v;
  *total = s_warp[32];
  __syncthreads();
  return res;
}

// sum over the CTA (every thread gets it).  Ends with a CTA barrier.
template <class T>
__device__ T block_sum(T v, T* s_warp) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += shfl_xor_t<T>(v, o);
  if (lane == 0) s_warp[warp] = v;
  __syncthreads();
  if (warp == 0) {
    T t = lane < (int)(blockDim.x >> 5) ? s_warp[lane] : (T)0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += shfl_xor_t<T>(t, o);
    if (lane == 0) s_warp[32] = t;
  }
  __syncthreads();
  const T t = s_warp[32];
  __syncthreads();
  return t;
}

}  // namespace bit1
