// step_f32.cu -- step_kernel instantiations: gradients fp32, bf16 working copy off.
#include "step_dispatch.cuh"

namespace hadpsgd {
LaunchPlan plan_f32(int G, bool exact, bool diag, int mode, int wmode) {
    return pick_G<false, false>(G, exact, diag, mode, wmode);
}
}  // namespace hadpsgd
