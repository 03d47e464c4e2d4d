// inst_q2.cu -- slot kernel instantiation: QuadDyn, 2 agent(s), 256 threads per problem slot, >= 1 CTA(s) per SM,
// hot layout group wherever it fits (generic loads).
#include "inst.cuh"
namespace jipm {
Inst inst_q2() { return make_inst<Cfg<QuadDyn, 2, 256, false>, 1>(); }
}  // namespace jipm
