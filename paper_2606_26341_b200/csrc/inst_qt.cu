// inst_qt.cu -- slot kernel instantiation: QuatDyn (the paper's 13-state quaternion quadrotor), 1 agent,
// 256 threads per problem slot, >= 1 CTA per SM, layout arrays wherever they fit (at the paper's horizon of 30 knots the
// factor blocks, J and W exceed one SM's shared memory).
#include "inst.cuh"
namespace jipm {
Inst inst_qt() { return make_inst<Cfg<QuatDyn, 1, 256, false>, 1>(); }
}  // namespace jipm
