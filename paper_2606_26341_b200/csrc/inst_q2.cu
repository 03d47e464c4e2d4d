// inst_q2.cu -- slot kernel instantiation: Cfg<QuadDyn, 2>.
#include "inst.cuh"
namespace jipm {
using C_ = Cfg<QuadDyn, 2>;
cudaError_t launch_q2(const Args& a, int wpb, cudaStream_t st) { return launch_cfg<C_>(a, wpb, st); }
int sm_doubles_q2() { return C_::SM_TOTAL; }
}  // namespace jipm
