// Host-callable launchers of the load-time and diagnostic kernels (defined in aux_kernels.cu).
#pragma once
#include "common.cuh"

namespace bit1 {
// sets DevState::load_error when a position is outside [0, L) or a species tag is unknown (load) / additionally when
// the positions are not in cell order (restart)
int launch_load_validate(const Params& P, const Particles& in, unsigned n, cudaStream_t s);
int launch_state_validate(const Params& P, const Particles& p, unsigned n, cudaStream_t s);
// validate + cell index + general stable sort by cell of `in` (n particles) into `out`
// velocity_ready: NULL, or three events (vx, vy, vz still being copied on another stream): each component's gather waits
// for its own
int launch_load_sort(const Params& P, const Particles& in, const Particles& out, unsigned n, int have_pid,
                     void* scratch, cudaStream_t s, const cudaEvent_t* velocity_ready);
size_t load_scratch_bytes(unsigned capacity);
// exclusive scan of n words in place (tmp: n / 4096 + 2 words)
int launch_scan_u32(unsigned* a, size_t n, unsigned* tmp, cudaStream_t s);
// stable radix sort of n (key, value) word pairs laid out as load_scratch_bytes(stride) describes
int launch_radix_sort_u32(unsigned n, unsigned stride, int bits, void* scratch, cudaStream_t s, unsigned** keys,
                          unsigned** vals);
#ifdef BIT1_CHECKED
void launch_check_selftest(const Params& P, cudaStream_t s);
#endif
// cell[i] = cell_of(x[i]) for the live particles
int launch_fill_cells(const Params& P, const Particles& cur, cudaStream_t s);
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
