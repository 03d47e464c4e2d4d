// inst_q4.cu -- slot kernel instantiation: QuadDyn, 4 agent(s), 256 threads per problem slot, >= 1 CTA(s) per SM,
// hot layout group wherever it fits (generic loads).
#include "inst.cuh"
namespace jipm {
Inst inst_q4() { return make_inst<Cfg<QuadDyn, 4, 256, false>, 1>(); }
}  // namespace jipm
