// Instantiation of every kernel for the SoA track layout (the mapping is a
// compile-time choice).  One translation unit per layout so that the three build in parallel.
#include "step_impl.cuh"

namespace adept {
const LayoutOps kOpsSoA = OpsImpl<L_SOA>::make();
}  // namespace adept
