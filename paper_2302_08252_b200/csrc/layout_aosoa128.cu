// Instantiation of every kernel for the AoSoA128 track layout (the paper tried
// several AoSoA lane counts).
#include "step_impl.cuh"

namespace adept {
const LayoutOps kOpsAoSoA128 = OpsImpl<L_AOSOA128>::make();
}  // namespace adept
