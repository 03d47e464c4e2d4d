// inst.cuh -- body of one family instantiation (included by inst_*.cu with JIPM_INST_CFG / JIPM_INST_NAME set).
#pragma once
#include "kernel.cuh"
#include "launch.cuh"

namespace jipm {

template <class C>
static cudaError_t launch_cfg(const Args& a, int wpb, cudaStream_t st) {
    const size_t smem = (size_t)wpb * C::SM_TOTAL * sizeof(double);
    cudaError_t e = cudaFuncSetAttribute(jipm_slot_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int blocks = (a.n_slots + wpb - 1) / wpb;
    jipm_slot_kernel<C><<<blocks, wpb * 32, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace jipm
