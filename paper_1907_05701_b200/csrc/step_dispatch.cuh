// step_dispatch.cuh -- maps run-time (G, flags, mode) to one instantiation of step_kernel and
// its launch shape.  The instantiations are spread over four translation units
// (step_{f32,bf16}{,_emit}.cu), one per (gradient dtype, bf16 working copy) so they build in
// parallel; each defines one plan_* function declared here.
#pragma once
#include "internal.h"
#include "step_kernel.cuh"

namespace hadpsgd {

struct LaunchPlan { const void* fn; int threads; int tile_units; int blocks_per_sm; int wmode; };

// wmode: kOwn | kSlots (kPair only) | kPeer (kPair and kSingle, no bf16 working copy).  A
// combination that is not instantiated returns fn == nullptr.
LaunchPlan plan_f32(int G, bool exact, bool diag, int mode, int wmode);
LaunchPlan plan_bf16(int G, bool exact, bool diag, int mode, int wmode);
LaunchPlan plan_f32_emit(int G, bool exact, bool diag, int mode, int wmode);
LaunchPlan plan_bf16_emit(int G, bool exact, bool diag, int mode, int wmode);

// Launch shape: 256 threads, ONE resident block per SM, and
// enough 32-byte loads per thread (>= 12) that ~96 KB per SM are in flight.  More resident
// warps than that measured slower on this path (more DRAM pages open at once).
template <int G, bool BF16, bool EXACT, bool DIAG, int MODE, bool EMIT, int WMODE>
LaunchPlan plan_for() {
    static_assert((WMODE != kSlots && WMODE != kChain) || MODE == kPair, "slots are shared by the members of a kPair item only");
    static_assert(kInlineItems == kMaxItemsPerLaunch, "host and kernel disagree on the items per launch");
    constexpr int members = (MODE == kSingle) ? 1 : 2;
    constexpr int loads_per_unit = members * ((G > 0 ? G : 4) + (BF16 ? 4 : 2));
    constexpr int U = loads_per_unit <= 6 ? 2 : 1;
    // measured: 12 loads x 256 threads and 20 loads x 160 threads
    // (both ~100 KB in flight per SM) are the best shapes for fp32 G=4 and G=8; 8 loads x 256
    // threads x 1 block beats both 2 blocks/SM and U=2 for G=2.
    // Threads per block (one resident block per SM), measured per family:
    //  fp32 gradients, 20 loads per thread (G = 8 pairs): 160 -- 256 puts 164 KB in flight, too many
    //  a bf16 working copy (6 write streams per pair instead of 4): 192 (3-4 % faster than 256)
    //  bf16 gradients, G = 8 pairs: 224
    constexpr bool heavy_f32 = !BF16 && G > 0 && U * loads_per_unit >= 20;
    constexpr int THREADS = heavy_f32 ? 160 : (EMIT && MODE != kSingle) ? 192 : (BF16 && G == 8 && MODE != kSingle) ? 224 : 256;
    constexpr int in_flight = THREADS * U * loads_per_unit * 32;           // bytes per block
    constexpr int BPS = in_flight >= 48 * 1024 ? 1 : 2;
    // fp32 pair kernels with <= 12 loads per unit need 128-133 registers: capped at 128 so that TWO blocks
    // fit an SM -- not for the persistent grid (one block per SM) but so that the next step's blocks can
    // be resident behind the programmatic dependent launch and a one-wave problem can use 2 x #SMs blocks
    constexpr int MINB = (!BF16 && G >= 1 && G <= 4 && U == 1 && MODE != kSingle && WMODE == kOwn && !EMIT && THREADS == 256) ? 2 : 1;
    return {reinterpret_cast<const void*>(&step_kernel<G, BF16, EXACT, DIAG, MODE, EMIT, WMODE, U, THREADS, MINB>),
            THREADS, THREADS * U, BPS, WMODE};
}

template <int G, bool BF16, bool EXACT, bool DIAG, bool EMIT>
LaunchPlan pick_mode(int mode, int wmode) {
    const LaunchPlan none = {nullptr, 0, 0, 0, 0};
    // shared slots: the CHAIN walk where it measured faster (<= 12 loads per pair unit: fp32 G <= 4)
    constexpr bool chain = !BF16 && G >= 1 && G <= 4;
    if (wmode == kPeer) {
        if constexpr (EMIT) return none;
        else {
            if (mode == kPair) return plan_for<G, BF16, EXACT, DIAG, kPair, false, kPeer>();
            if (mode == kSingle) return plan_for<G, BF16, EXACT, DIAG, kSingle, false, kPeer>();
            return none;
        }
    }
    switch (mode) {
        case kPair: return wmode == kSlots ? plan_for<G, BF16, EXACT, DIAG, kPair, EMIT, chain ? kChain : kSlots>()
                                           : plan_for<G, BF16, EXACT, DIAG, kPair, EMIT, kOwn>();
        case kSingle: return plan_for<G, BF16, EXACT, DIAG, kSingle, EMIT, kOwn>();
        default: return wmode == kOwn ? plan_for<G, BF16, EXACT, DIAG, kPairEq7, EMIT, kOwn>() : none;
    }
}
template <int G, bool BF16, bool EMIT>
LaunchPlan pick_flags(bool exact, bool diag, int mode, int wmode) {
    if (exact) return diag ? pick_mode<G, BF16, true, true, EMIT>(mode, wmode) : pick_mode<G, BF16, true, false, EMIT>(mode, wmode);
    return diag ? pick_mode<G, BF16, false, true, EMIT>(mode, wmode) : pick_mode<G, BF16, false, false, EMIT>(mode, wmode);
}
template <bool BF16, bool EMIT>
LaunchPlan pick_G(int G, bool exact, bool diag, int mode, int wmode) {
    switch (G) {
        case 1: return pick_flags<1, BF16, EMIT>(exact, diag, mode, wmode);
        case 2: return pick_flags<2, BF16, EMIT>(exact, diag, mode, wmode);
        case 4: return pick_flags<4, BF16, EMIT>(exact, diag, mode, wmode);
        case 8: return pick_flags<8, BF16, EMIT>(exact, diag, mode, wmode);
        default: return pick_flags<0, BF16, EMIT>(exact, diag, mode, wmode);  // runtime learner count
    }
}

}  // namespace hadpsgd
