// Host-callable launchers of the load-time and diagnostic kernels (defined in aux_kernels.cu).
#pragma once
#include "common.cuh"

namespace bit1 {
// validate + cell index + general stable sort by cell of `in` (n particles) into `out`
// before_gather: NULL, or an event the final gather waits for (arrays other than x, sp, pid still being copied)
int launch_load_sort(const Params& P, const Particles& in, const Particles& out, unsigned n, int have_pid,
                     void* scratch, cudaStream_t s, cudaEvent_t before_gather);
size_t load_scratch_bytes(unsigned capacity);
// out: [kMaxSpecies*3] = (count, sum v^2, sum vx) per species, then sum g_j E_j^2
int launch_moments(const Params& P, const Particles& cur, double* partial, double* out, cudaStream_t s);
size_t moments_scratch_bytes();
}  // namespace bit1

namespace bit1 {
// NEXT-4: one species in the paper's checkpoint layout (counts per cell, then records in cell order)
size_t export_scratch_bytes(int nc, unsigned capacity);
// scratch afterwards: [0] total (u64), [256] cell_cnt int[nc], then exclusive chunk offsets
int launch_export_count(const Params& P, const Particles& cur, int species, unsigned capacity, void* scratch,
                        cudaStream_t s);
int launch_export_scatter(const Params& P, const Particles& cur, const Particles& out, int species, void* scratch,
                          cudaStream_t s);
}  // namespace bit1
