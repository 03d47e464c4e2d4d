// inst_q1.cu -- slot kernel instantiation: QuadDyn, 1 agent(s), 128 threads per problem slot, >= 3 CTA(s) per SM.
#include "inst.cuh"
namespace jipm {
Inst inst_q1() { return make_inst<Cfg<QuadDyn, 1, 128>, 3>(); }
}  // namespace jipm
