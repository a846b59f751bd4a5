// step_bf16_emit.cu -- step_kernel instantiations: gradients bf16, bf16 working copy emitted.
#include "step_dispatch.cuh"

namespace hadpsgd {
LaunchPlan plan_bf16_emit(int G, bool exact, bool diag, int mode, int wmode) {
    return pick_G<true, true>(G, exact, diag, mode, wmode);
}
}  // namespace hadpsgd
