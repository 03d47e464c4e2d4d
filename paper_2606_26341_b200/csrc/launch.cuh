// launch.cuh -- host-visible launchers of the slot kernel, one translation unit per family configuration
// (inst_*.cu) so that the four template instantiations compile in parallel.
#pragma once
#include "common.cuh"

namespace jipm {

struct LaunchInfo { int sm_doubles_per_warp; };

cudaError_t launch_pm(const Args& a, int warps_per_block, cudaStream_t st);
cudaError_t launch_q1(const Args& a, int warps_per_block, cudaStream_t st);
cudaError_t launch_q2(const Args& a, int warps_per_block, cudaStream_t st);
cudaError_t launch_q4(const Args& a, int warps_per_block, cudaStream_t st);
int sm_doubles_pm();
int sm_doubles_q1();
int sm_doubles_q2();
int sm_doubles_q4();
cudaError_t launch_fp64_peak(double* out, int blocks, int threads, int iters, cudaStream_t st);

}  // namespace jipm
