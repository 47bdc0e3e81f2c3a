// Test-side probe (not product code): evaluates cuRAND's own device function curand_Philox4x32_10 on given
// counters/keys so that tests/test_gpu_philox_library.py can pin the oracle's and the library's Philox to it.
#include <cuda_runtime.h>
#include <curand_philox4x32_x.h>
#include <stdint.h>

__global__ void k_probe(const uint4* ctr, const uint2* key, uint4* out, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = curand_Philox4x32_10(ctr[i], key[i]);
}

extern "C" int curand_philox_probe(const uint32_t* ctr_host, const uint32_t* key_host, uint32_t* out_host, int n) {
  uint4 *c, *o;
  uint2* k;
  if (cudaMalloc(&c, n * 16) || cudaMalloc(&k, n * 8) || cudaMalloc(&o, n * 16)) return 1;
  cudaMemcpy(c, ctr_host, n * 16, cudaMemcpyHostToDevice);
  cudaMemcpy(k, key_host, n * 8, cudaMemcpyHostToDevice);
  k_probe<<<(n + 255) / 256, 256>>>(c, k, o, n);
  const int bad = cudaMemcpy(out_host, o, n * 16, cudaMemcpyDeviceToHost) != cudaSuccess;
  cudaFree(c); cudaFree(k); cudaFree(o);
  return bad;
}
