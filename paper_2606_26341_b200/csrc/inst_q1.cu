// inst_q1.cu -- slot kernel instantiation: QuadDyn, 1 agent(s), 256 threads per problem slot, >= 1 CTA(s) per SM,
// hot layout group guaranteed shared-memory resident.
#include "inst.cuh"
namespace jipm {
Inst inst_q1() { return make_inst<Cfg<QuadDyn, 1, 256, true>, 1>(); }
}  // namespace jipm
