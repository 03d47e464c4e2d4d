// inst_pm.cu -- slot kernel instantiation: PointmassDyn, 1 agent(s), 128 threads per problem slot, >= 4 CTA(s) per SM,
// hot layout group guaranteed shared-memory resident.
#include "inst.cuh"
namespace jipm {
Inst inst_pm() { return make_inst<Cfg<PointmassDyn, 1, 128, true>, 4>(); }
}  // namespace jipm

namespace jipm {
// dependent-free DFMA chains: the FP64 roofline denominator
__global__ void fp64_peak_kernel(double* out, int iters) {
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double b = 1.0000001, cc = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, b, cc); a1 = fma(a1, b, cc); a2 = fma(a2, b, cc); a3 = fma(a3, b, cc);
        a4 = fma(a4, b, cc); a5 = fma(a5, b, cc); a6 = fma(a6, b, cc); a7 = fma(a7, b, cc);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}

cudaError_t launch_fp64_peak(double* out, int blocks, int threads, int iters, cudaStream_t st) {
    fp64_peak_kernel<<<blocks, threads, 0, st>>>(out, iters);
    return cudaGetLastError();
}
}  // namespace jipm
