// step_dispatch.cuh -- maps run-time (G, flags, mode) to one instantiation of step_kernel and
// its launch shape.  The instantiations are spread over four translation units
// (step_{f32,bf16}{,_emit}.cu), one per (gradient dtype, bf16 working copy) so they build in
// parallel; each defines one plan_* function declared here.
#pragma once
#include "step_kernel.cuh"

namespace hadpsgd {

struct LaunchPlan { const void* fn; int threads; int tile_units; int blocks_per_sm; };

// shared: pair members share weight slots (kPair only; ignored for the other modes)
LaunchPlan plan_f32(int G, bool exact, bool diag, int mode, bool shared);
LaunchPlan plan_bf16(int G, bool exact, bool diag, int mode, bool shared);
LaunchPlan plan_f32_emit(int G, bool exact, bool diag, int mode, bool shared);
LaunchPlan plan_bf16_emit(int G, bool exact, bool diag, int mode, bool shared);

// Launch shape: 256 threads, ONE resident block per SM, and
// enough 32-byte loads per thread (>= 12) that ~96 KB per SM are in flight.  More resident
// warps than that measured slower on this path (more DRAM pages open at once).
template <int G, bool BF16, bool EXACT, bool DIAG, int MODE, bool EMIT, bool SHARED>
LaunchPlan plan_for() {
    static_assert(!SHARED || MODE == kPair, "slots are shared by the members of a kPair item only");
    constexpr int members = (MODE == kSingle) ? 1 : 2;
    constexpr int loads_per_unit = members * ((G > 0 ? G : 4) + (BF16 ? 4 : 2));
    constexpr int U = loads_per_unit <= 6 ? 2 : 1;
    // measured: 12 loads x 256 threads and 20 loads x 160 threads
    // (both ~100 KB in flight per SM) are the best shapes for fp32 G=4 and G=8; 8 loads x 256
    // threads x 1 block beats both 2 blocks/SM and U=2 for G=2.
    constexpr int THREADS = (!BF16 && G > 0 && U * loads_per_unit >= 20) ? 160 : 256;
    constexpr int in_flight = THREADS * U * loads_per_unit * 32;           // bytes per block
    constexpr int BPS = in_flight >= 48 * 1024 ? 1 : 2;
    return {reinterpret_cast<const void*>(&step_kernel<G, BF16, EXACT, DIAG, MODE, EMIT, SHARED, U, THREADS, 1>),
            THREADS, THREADS * U, BPS};
}

template <int G, bool BF16, bool EXACT, bool DIAG, bool EMIT>
LaunchPlan pick_mode(int mode, bool shared) {
    switch (mode) {
        case kPair: return shared ? plan_for<G, BF16, EXACT, DIAG, kPair, EMIT, true>()
                                  : plan_for<G, BF16, EXACT, DIAG, kPair, EMIT, false>();
        case kSingle: return plan_for<G, BF16, EXACT, DIAG, kSingle, EMIT, false>();
        default: return plan_for<G, BF16, EXACT, DIAG, kPairEq7, EMIT, false>();
    }
}
template <int G, bool BF16, bool EMIT>
LaunchPlan pick_flags(bool exact, bool diag, int mode, bool shared) {
    if (exact) return diag ? pick_mode<G, BF16, true, true, EMIT>(mode, shared) : pick_mode<G, BF16, true, false, EMIT>(mode, shared);
    return diag ? pick_mode<G, BF16, false, true, EMIT>(mode, shared) : pick_mode<G, BF16, false, false, EMIT>(mode, shared);
}
template <bool BF16, bool EMIT>
LaunchPlan pick_G(int G, bool exact, bool diag, int mode, bool shared) {
    switch (G) {
        case 1: return pick_flags<1, BF16, EMIT>(exact, diag, mode, shared);
        case 2: return pick_flags<2, BF16, EMIT>(exact, diag, mode, shared);
        case 4: return pick_flags<4, BF16, EMIT>(exact, diag, mode, shared);
        case 8: return pick_flags<8, BF16, EMIT>(exact, diag, mode, shared);
        default: return pick_flags<0, BF16, EMIT>(exact, diag, mode, shared);  // runtime learner count
    }
}

}  // namespace hadpsgd
