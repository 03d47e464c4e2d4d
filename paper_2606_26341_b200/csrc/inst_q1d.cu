// inst_q1d.cu -- experimental slot kernel instantiations of the single-quadrotor families.
#include "inst.cuh"
namespace jipm {
Inst inst_q1d() { return make_inst<Cfg<QuadDyn, 1, 256, false>, 2>(); }
Inst inst_q1e() { return make_inst<Cfg<QuadDyn, 1, 128, false>, 4>(); }
// 128 registers per thread but the whole shared memory of the SM (one CTA per SM): isolates the cost of the register cap
Inst inst_q1h() { Inst i = make_inst<Cfg<QuadDyn, 1, 256, true>, 2>(); i.info.min_blocks = 1; return i; }
}  // namespace jipm
