// Instantiation of every kernel for the AoSoA32 track layout (the mapping is a
// compile-time choice).  One translation unit per layout so that the three build in parallel.
#include "step_impl.cuh"

namespace adept {
const LayoutOps kOpsAoSoA32 = OpsImpl<L_AOSOA32>::make();
}  // namespace adept
