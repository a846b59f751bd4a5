// step_bf16.cu -- step_kernel instantiations: gradients bf16, bf16 working copy off.
#include "step_dispatch.cuh"

namespace hadpsgd {
LaunchPlan plan_bf16(int G, bool exact, bool diag, int mode, int wmode) {
    return pick_G<true, false>(G, exact, diag, mode, wmode);
}
}  // namespace hadpsgd
