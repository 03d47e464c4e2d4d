// inst_q4.cu -- slot kernel instantiation: Cfg<QuadDyn, 4>.
#include "inst.cuh"
namespace jipm {
using C_ = Cfg<QuadDyn, 4>;
cudaError_t launch_q4(const Args& a, int wpb, cudaStream_t st) { return launch_cfg<C_>(a, wpb, st); }
int sm_doubles_q4() { return C_::SM_TOTAL; }
}  // namespace jipm
