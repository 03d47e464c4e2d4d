// inst_q2.cu -- slot kernel instantiation: QuadDyn, 2 agent(s), 128 threads per problem slot, >= 2 CTA(s) per SM.
#include "inst.cuh"
namespace jipm {
Inst inst_q2() { return make_inst<Cfg<QuadDyn, 2, 128>, 2>(); }
}  // namespace jipm
