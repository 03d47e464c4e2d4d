// inst_q1.cu -- slot kernel instantiation: Cfg<QuadDyn, 1>.
#include "inst.cuh"
namespace jipm {
using C_ = Cfg<QuadDyn, 1>;
cudaError_t launch_q1(const Args& a, int wpb, cudaStream_t st) { return launch_cfg<C_>(a, wpb, st); }
int sm_doubles_q1() { return C_::SM_TOTAL; }
}  // namespace jipm
