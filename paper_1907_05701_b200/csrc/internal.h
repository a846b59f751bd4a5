// internal.h -- shared between the host runtime (allocator.cpp, scheduler.cpp) and the
// CUDA translation unit (hadpsgd.cu).  Product code only: nothing under oracle/ sees this.
#pragma once
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/hadpsgd.h"

namespace hadpsgd {

constexpr size_t kRegionAlign = 256;  // byte alignment of every buffer start inside the arena

// a0: where everything lives.  All buffers have P_padded elements; segment k of every
// buffer starts at seg_offset[k] (multiple of HADPSGD_SEG_ALIGN_ELEMS).
struct Layout {
    int S = 0, G = 0, n_seg = 0;
    int grad_dtype = HADPSGD_F32;
    int working_dtype = HADPSGD_F32;         // HADPSGD_BF16: a bf16 copy of the weights is emitted
    int peer_stage = 0;                      // 1: two stage weight buffers per super-learner follow the S main ones
    int64_t P_padded = 0;
    std::vector<int64_t> seg_len, seg_offset;
    size_t w_off = 0, v_off = 0, g_off = 0;  // byte offsets inside the arena
    size_t stage_off = 0;                    // = w_off + S weight buffers: [2][S] stage buffers (peer_stage only)
    size_t epoch_off = 0;                    // = stage_off + 2 S buffers: this handle's 32-bit epoch word on a 256 B line of
                                             // its own (peer_stage only); peers find it from the stage pointer they attached
    size_t wb_off = 0;                       // bf16 working copies (S x P_padded x 2 B), if any
    size_t aux_off = 0, aux_bytes = 0;       // diagnostics scratch: tagged partials | plain scratch | results
    size_t partials_bytes = 0, scratch_bytes = 0;
    size_t total_bytes = 0;
    size_t grad_elem_bytes() const { return grad_dtype == HADPSGD_BF16 ? 2 : 4; }
    size_t w_stride_bytes() const { return static_cast<size_t>(P_padded) * 4; }
    size_t g_stride_bytes() const { return static_cast<size_t>(P_padded) * grad_elem_bytes(); }
};

// Upper bound on the persistent grid of the step kernel (sizes the partials scratch; grids are
// clamped to it).  Not tied to an SM count: the grid itself is #SMs of the device x blocks/SM.
constexpr int kMaxGridBlocks = 3072;
constexpr int kMaxItemsPerLaunch = 32;   // == kInlineItems of step_kernel.cuh (static_assert there)
constexpr int kMaxDiagQuantities = 9;    // per work item: gsq_s, gsq_p, wsq_s, wsq_p, gap (+4 in peer mode)
constexpr int kDiagArrays = 5;           // device result: gsq | wsq | gap | pend_wsq | pend_gap, S doubles each

// Returns HADPSGD_OK or HADPSGD_INVALID_ARG; err gets a human-readable reason.
int compute_layout(int S, int G, const int64_t* seg_len, int n_seg, hadpsgd_dtypes dt,
                   Layout* out, std::string* err);

// a1: work list for one step.  Each item is a pair (s, p) to average, or s == p (unmixed).
// ws / wp: weight SLOT (buffer index 0..S-1) that currently holds w_s / w_p; wo_s / wo_p: slot the
// new weights of s / p are written to.  Without HADPSGD_SHARE_PAIR_WEIGHTS every slot is the
// member's own index.  With it both members of a pair share ONE slot (wo_s == wo_p), because
// they hold identical bits after the step (R3): one weight write instead of two.
// b_s / b_p (peer mode): 0, or 1 + index into the handle's peer pointer table of the stage buffer
// whose average with ws / wp IS the member's weight (a mix left pending by the previous step).
struct WorkItem { int32_t s, p, ws, wp, wo_s, wo_p, b_s, b_p; };
struct SlotCopy { int32_t src, dst; };   // "copy weight slot src to slot dst" (un-sharing)

int ring_partner(int S, uint64_t step_k, int32_t* partner);  // even/odd ring pairing
int validate_matching(int S, const int32_t* partner);        // partner[partner[s]] == s

// Turns a matching into pair items (s < p) and single items (s == p), ascending s, and assigns
// weight slots.  w_slot[s] (in/out, [S]) = slot holding w_s before / after the step.
//   share == false: slots are the identity, w_slot is left untouched.
//   share == true : (1) if the matching has unmixed members while some slot is shared, the shared
//                   slots are first split again (copies: src -> a free slot);
//                   (2) every pair writes to ONE slot that no other item of this step reads:
//                   in place if one member's current slot is referenced by nobody outside the
//                   pair, else the lowest-numbered slot that is free at the start of the step.
// A free slot always exists when needed: S slots, S members, so the number of free slots equals
// the number of shared ones, and a pair needs a free slot only if both its members come out of
// two different shared slots.
void plan_step(int S, const int32_t* partner, bool share, std::vector<int32_t>* w_slot,
               std::vector<WorkItem>* pairs, std::vector<WorkItem>* singles,
               std::vector<SlotCopy>* copies);
// Splits every shared slot (copies: src -> free slot); afterwards w_slot is injective.
void plan_unshare(int S, std::vector<int32_t>* w_slot, std::vector<SlotCopy>* copies);

// Super-learner partition over `world` handles (row f4; Fig. 3).  Rank r owns the
// global super-learners [rank_begin[r], rank_begin[r+1]); rank_begin[world] = S_global.  `partner`
// is a matching of the S_global members.  pending (in/out, [S_local]): global index of the partner
// whose stage buffer completes this member's weights (w = 1/2 (own stage + partner stage)), or -1.
// Weight buffer indices of the items: main s, stage (parity e, s) = S_local * (1 + e) + s; b refers
// to peer-table entry e * S_global + global index.  A pair with both members here is an ordinary
// pair item; a member whose partner lives elsewhere becomes a single item that writes its u into
// stage[epoch & 1] and is left pending; pending members read stage[(epoch - 1) & 1].
int plan_peer_step(int world, int rank, const int32_t* rank_begin, const int32_t* partner, uint64_t epoch,
                   std::vector<int32_t>* pending, std::vector<WorkItem>* pairs, std::vector<WorkItem>* singles);

}  // namespace hadpsgd
