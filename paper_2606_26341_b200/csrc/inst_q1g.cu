// inst_q1g.cu -- slot kernel instantiation: QuadDyn, 1 agent(s), 256 threads per problem slot, >= 1 CTA(s) per SM,
// hot layout group wherever it fits (generic loads).
#include "inst.cuh"
namespace jipm {
Inst inst_q1g() { return make_inst<Cfg<QuadDyn, 1, 256, false>, 1>(); }
}  // namespace jipm
