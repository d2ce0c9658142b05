// avm_transport_inst.cu — instantiations of transport_kernel for ONE (field kind, B) pair: compiled six times by build.py
// with -DAVM_INST_FK=0|1|2 -DAVM_INST_B=0|1 (parallel translation units; the kernel is ~10 s of ptxas per variant).
// Tallies are always kept in the hot loop (three per-thread counters); AVM_RUN_NO_TALLIES only skips their publication.
#include "avm_transport.cuh"

#ifndef AVM_INST_FK
#error "compile with -DAVM_INST_FK=0|1|2 -DAVM_INST_B=0|1"
#endif

namespace avm {
namespace {
template <int FK, bool B, int T, bool TPB, bool BANDED>
TransportFn pick4(bool smemtab, bool signal) {
  if (signal) return smemtab ? transport_kernel<FK, B, true, true, T, TPB, BANDED, true> : nullptr;
  return smemtab ? transport_kernel<FK, B, true, true, T, TPB, BANDED, false> : transport_kernel<FK, B, true, false, T, TPB, BANDED, false>;
}
template <int FK, bool B, int T, bool TPB>
TransportFn pick3(bool smemtab, bool banded, bool signal) {
  return banded ? pick4<FK, B, T, TPB, true>(smemtab, signal) : pick4<FK, B, T, TPB, false>(smemtab, signal);
}
}  // namespace

template <>
TransportFn pick_transport_inst<AVM_INST_FK, (AVM_INST_B != 0)>(bool smemtab, bool wide, bool banded, bool signal) {
  constexpr int FK = AVM_INST_FK;
  constexpr bool B = AVM_INST_B != 0;
  return wide ? pick3<FK, B, kThreadsWide, false>(smemtab, banded, signal) : pick3<FK, B, kThreads, true>(smemtab, banded, signal);
}

}  // namespace avm
