// inst_q1b.cu -- slot kernel instantiation: QuadDyn, 1 agent, 128 threads per problem slot, >= 2 CTAs per SM,
// layout arrays wherever they fit (generic loads).
#include "inst.cuh"
namespace jipm {
Inst inst_q1b() { return make_inst<Cfg<QuadDyn, 1, 128, false>, 2>(); }
}  // namespace jipm
