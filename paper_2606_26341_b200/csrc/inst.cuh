// inst.cuh -- body of one family instantiation (included by inst_*.cu).
#pragma once
#include "kernel.cuh"
#include "launch.cuh"

namespace jipm {

template <class C, int MINB>
static cudaError_t launch_cfg(const Args& a, cudaStream_t st) {
    const size_t smem = (size_t)(C::SM_TOTAL + a.L.nsm) * sizeof(double);
    cudaError_t e = cudaFuncSetAttribute(jipm_slot_kernel<C, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyToSymbolAsync(g_A, &a, sizeof(Args), 0, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    jipm_slot_kernel<C, MINB><<<a.n_slots, C::NT, smem, st>>>();
    return cudaGetLastError();
}

template <class C, int MINB>
static Inst make_inst() {
    Inst i;
    i.info.nt = C::NT; i.info.sm_fixed = C::SM_TOTAL; i.info.min_blocks = MINB; i.info.hot_sm = C::HOT_SM ? 1 : 0;
    i.launch = &launch_cfg<C, MINB>;
    return i;
}

}  // namespace jipm
