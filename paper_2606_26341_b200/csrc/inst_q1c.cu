// inst_q1c.cu -- slot kernel instantiation: QuadDyn, 1 agent, 64 threads per problem slot, >= 4 CTAs per SM,
// layout arrays wherever they fit (generic loads).
#include "inst.cuh"
namespace jipm {
Inst inst_q1c() { return make_inst<Cfg<QuadDyn, 1, 64, false>, 4>(); }
}  // namespace jipm
