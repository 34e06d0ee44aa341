// Instantiation of every kernel for the AoSoA64 track layout ("AoSoA64 with the dense
// double buffer" was the paper's fastest variant).
#include "step_impl.cuh"

namespace adept {
const LayoutOps kOpsAoSoA64 = OpsImpl<L_AOSOA64>::make();
}  // namespace adept
