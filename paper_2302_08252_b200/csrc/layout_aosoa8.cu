// Instantiation of every kernel for the AoSoA8 track layout (the paper tried
// several AoSoA lane counts).
#include "step_impl.cuh"

namespace adept {
const LayoutOps kOpsAoSoA8 = OpsImpl<L_AOSOA8>::make();
}  // namespace adept
