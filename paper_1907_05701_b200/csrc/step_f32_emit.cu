// step_f32_emit.cu -- step_kernel instantiations: gradients fp32, bf16 working copy emitted.
#include "step_dispatch.cuh"

namespace hadpsgd {
LaunchPlan plan_f32_emit(int G, bool exact, bool diag, int mode, int wmode) {
    return pick_G<false, true>(G, exact, diag, mode, wmode);
}
}  // namespace hadpsgd
