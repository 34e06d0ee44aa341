// Instantiation of every kernel for the HC16 track layout: hot/cold split with per-kind grouping
// (layout.cuh Mapping<L_HC16>).  One translation unit per layout so that they build in parallel.
#include "step_impl.cuh"

namespace adept {
const LayoutOps kOpsHC16 = OpsImpl<L_HC16>::make();
}  // namespace adept
