// Instantiation of every kernel for the SoA-of-16-byte-groups track layout (
// BASELINE.json north_star: "coalesced, vectorised 16-byte loads of SoA fields").
#include "step_impl.cuh"

namespace adept {
const LayoutOps kOpsSoA16 = OpsImpl<L_SOA16>::make();
}  // namespace adept
