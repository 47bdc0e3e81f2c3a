// Host-callable launchers of the step kernels (defined in step_kernels.cu and general_kernels.cu).
#pragma once
#include "common.cuh"

namespace bit1 {
cudaError_t configure_kernels();
// SMs of the current device (cudaDevAttrMultiProcessorCount, remembered per device); every grid is sized from it
int sm_count();
// one timestep on stream s; returns the number of kernels launched
// ev: NULL, or 5 events recorded before/between/after the four kernels (per-kernel timing)
int launch_step(const Params& P, const Particles& cur, const Particles& nxt, cudaStream_t s, cudaEvent_t* ev);
// counts per cell -> cell_start, deposit, field solve for particles already sorted in cur
int launch_rebuild(const Params& P, const Particles& cur, cudaStream_t s);
// pieces of the above that the general path reuses
int launch_clear_grids(const Params& P, cudaStream_t s);
// desc_out: tile descriptors of the arrangement the scan describes (the store half it lives in)
int launch_mid(const Params& P, const Particles& cur, int2* desc_out, int do_colscan, cudaStream_t s);
int launch_deposit(const Params& P, const Particles& cur, const unsigned* n_ptr, cudaStream_t s);
int launch_field(const Params& P, int commit_step, cudaStream_t s);
int launch_average(const Params& P, cudaStream_t s);
// one timestep by the general path (general_kernels.cu); count_side_effects: see there
size_t general_scratch_bytes(unsigned capacity);
int launch_general_step(const Params& P, const Particles& cur, const Particles& nxt, int count_side_effects,
                        void* scratch, cudaStream_t s);
}  // namespace bit1
