// launch.cuh -- host-visible launchers of the slot kernel, one translation unit per family configuration
// (inst_*.cu) so that the template instantiations compile in parallel.
#pragma once
#include "common.cuh"

namespace jipm {

// what the host needs to know about one instantiation
struct InstInfo {
    int nt;            // threads per problem slot (= CTA size: one team per CTA)
    int sm_fixed;      // fixed shared memory per team, doubles (tiles, staging, reduction scratch)
    int min_blocks;    // __launch_bounds__ min CTAs per SM the kernel was compiled for
    int hot_sm;        // 1: compiled assuming the hot layout group is shared-memory resident
};

typedef cudaError_t (*launch_fn)(const Args& a, cudaStream_t st);
struct Inst { InstInfo info; launch_fn launch; };

Inst inst_pm();
Inst inst_q1();
Inst inst_q1g();
Inst inst_q2();
Inst inst_q4();
Inst inst_qt();
cudaError_t launch_fp64_peak(double* out, int blocks, int threads, int iters, cudaStream_t st);

}  // namespace jipm
