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
    int64_t P_padded = 0;
    std::vector<int64_t> seg_len, seg_offset;
    size_t w_off = 0, v_off = 0, g_off = 0;  // byte offsets inside the arena
    size_t wb_off = 0;                       // bf16 working copies (S x P_padded x 2 B), if any
    size_t aux_off = 0, aux_bytes = 0;       // diagnostics scratch (partials, results, ticket)
    size_t total_bytes = 0;
    size_t grad_elem_bytes() const { return grad_dtype == HADPSGD_BF16 ? 2 : 4; }
    size_t w_stride_bytes() const { return static_cast<size_t>(P_padded) * 4; }
    size_t g_stride_bytes() const { return static_cast<size_t>(P_padded) * grad_elem_bytes(); }
};

// Upper bound on persistent blocks the step kernel may launch (sizes the partials scratch).
constexpr int kMaxGridBlocks = 148 * 16;
constexpr int kDiagQuantities = 5;  // per work item: gsq_s, gsq_p, wsq_s, wsq_p, gap

// Returns HADPSGD_OK or HADPSGD_INVALID_ARG; err gets a human-readable reason.
int compute_layout(int S, int G, const int64_t* seg_len, int n_seg, hadpsgd_dtypes dt,
                   Layout* out, std::string* err);

// a1: work list for one step.  Each item is (a, b): a pair to average, or a == b (unmixed).
struct WorkItem { int32_t a, b; };
int ring_partner(int S, uint64_t step_k, int32_t* partner);  // even/odd ring pairing
int validate_matching(int S, const int32_t* partner);        // partner[partner[s]] == s
// Splits a matching into pair items (a < b) and single items (a == b), in ascending a.
void matching_to_work(int S, const int32_t* partner, std::vector<WorkItem>* pairs,
                      std::vector<WorkItem>* singles);

}  // namespace hadpsgd
