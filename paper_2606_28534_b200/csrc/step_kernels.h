// Host-callable launchers of the step kernels (defined in step_kernels.cu).
#pragma once
#include "common.cuh"

namespace bit1 {
cudaError_t configure_kernels();
// one timestep on stream s; returns the number of kernels launched
// ev: NULL, or 5 events recorded before/between/after the kernels (per-kernel timing; k_mid + k_colscan share one)
int launch_step(const Params& P, const Particles& cur, const Particles& nxt, int variant, cudaStream_t s,
                cudaEvent_t* ev);
// counts per cell -> cell_start, deposit, field solve for particles already sorted in cur
int launch_rebuild(const Params& P, const Particles& cur, cudaStream_t s);
}  // namespace bit1
