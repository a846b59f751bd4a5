// allocator.cpp -- a0, the replica allocator (host only).
//
// Lays out S weight buffers, S momentum buffers and S*G learner gradient buffers in one
// arena, flat (n_seg == 1) or as a ragged per-tensor segment table whose segment starts are
// aligned to HADPSGD_SEG_ALIGN_ELEMS elements in every buffer (
// north_star (a)).  One weight + one momentum copy per SUPER-learner: the G learners of a
// super-learner have staleness 0, so their replicas are identical and are
// collapsed (R18).  With dtypes.working_dtype == BF16 a fourth region holds S bf16
// working copies of the weights (row f2).  With dtypes.peer_stage the weight region also holds two
// stage buffers per super-learner, in which the halves of a mix between two arenas wait (row f4).
#include "internal.h"

namespace hadpsgd {

static size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int compute_layout(int S, int G, const int64_t* seg_len, int n_seg, hadpsgd_dtypes dt,
                   Layout* out, std::string* err) {
    auto fail = [&](const char* m) { if (err) *err = m; return HADPSGD_INVALID_ARG; };
    if (S < 1) return fail("S must be >= 1");
    if (S > HADPSGD_MAX_S) return fail("S exceeds HADPSGD_MAX_S");
    if (G < 1) return fail("G must be >= 1");
    if (n_seg < 1 || !seg_len) return fail("segment table must have at least one segment");
    if (dt.grad_dtype != HADPSGD_F32 && dt.grad_dtype != HADPSGD_BF16) return fail("grad_dtype must be F32 or BF16");
    if (dt.master_dtype != HADPSGD_F32) return fail("master_dtype must be F32");
    if (dt.working_dtype != HADPSGD_F32 && dt.working_dtype != HADPSGD_BF16) return fail("working_dtype must be F32 (none) or BF16");
    if (dt.peer_stage != 0 && dt.peer_stage != 1) return fail("peer_stage must be 0 or 1");
    if (dt.peer_stage && dt.working_dtype != HADPSGD_F32) return fail("peer_stage (HADPSGD_PEER) has no bf16 working copy");

    Layout L;
    L.S = S; L.G = G; L.n_seg = n_seg; L.grad_dtype = dt.grad_dtype; L.working_dtype = dt.working_dtype;
    L.peer_stage = dt.peer_stage;
    L.seg_len.assign(seg_len, seg_len + n_seg);
    L.seg_offset.resize(n_seg);
    int64_t off = 0;
    for (int k = 0; k < n_seg; ++k) {
        if (seg_len[k] < 1) return fail("every segment length must be >= 1");
        L.seg_offset[k] = off;
        int64_t padded = (seg_len[k] + HADPSGD_SEG_ALIGN_ELEMS - 1) / HADPSGD_SEG_ALIGN_ELEMS *
                         HADPSGD_SEG_ALIGN_ELEMS;
        if (off > INT64_MAX / 8 - padded) return fail("segment table too large");
        off += padded;
    }
    L.P_padded = off;

    size_t cur = 0;
    // weights: S main buffers, then (peer_stage) 2 x S stage buffers, contiguous: buffer x = w_off + x * P * 4
    L.w_off = cur;
    L.stage_off = cur + static_cast<size_t>(S) * L.w_stride_bytes();
    cur = round_up(cur + static_cast<size_t>(S) * (L.peer_stage ? 3 : 1) * L.w_stride_bytes(), kRegionAlign);
    if (L.peer_stage) {   // the epoch word of the neighbour handshake, directly behind the stage buffers (a buffer is a
        L.epoch_off = L.stage_off + static_cast<size_t>(2) * S * L.w_stride_bytes();   // multiple of 256 B, so no gap)
        cur = L.epoch_off + kRegionAlign;
    }
    L.v_off = cur; cur = round_up(cur + static_cast<size_t>(S) * L.w_stride_bytes(), kRegionAlign);
    L.g_off = cur; cur = round_up(cur + static_cast<size_t>(S) * G * L.g_stride_bytes(), kRegionAlign);
    L.wb_off = cur;
    if (L.working_dtype == HADPSGD_BF16) cur = round_up(cur + static_cast<size_t>(S) * L.P_padded * 2, kRegionAlign);
    // aux: per-block partial sums of the step kernel [kMaxGridBlocks][items per launch x quantities], 16 B
    // each (a double with its launch tag, step_kernel.cuh); a plain scratch of doubles for the consensus
    // and flush kernels; the results (kDiagArrays x S doubles)
    const int items = S < kMaxItemsPerLaunch ? S : kMaxItemsPerLaunch;
    L.aux_off = cur;
    L.partials_bytes = round_up(static_cast<size_t>(items) * kMaxDiagQuantities * kMaxGridBlocks * 16, kRegionAlign);
    L.scratch_bytes = round_up(static_cast<size_t>(kMaxGridBlocks) * kMaxItemsPerLaunch * 2 * sizeof(double), kRegionAlign);
    L.aux_bytes = L.partials_bytes + L.scratch_bytes +
                  round_up(static_cast<size_t>(kDiagArrays * S) * sizeof(double) + 256, kRegionAlign);
    cur += L.aux_bytes;
    L.total_bytes = cur;
    *out = L;
    return HADPSGD_OK;
}

}  // namespace hadpsgd

extern "C" int hadpsgd_required_bytes(int S, int G, const int64_t* seg_len, int n_seg,
                                      hadpsgd_dtypes dt, size_t* out_bytes) {
    if (!out_bytes) return HADPSGD_INVALID_ARG;
    hadpsgd::Layout L;
    int rc = hadpsgd::compute_layout(S, G, seg_len, n_seg, dt, &L, nullptr);
    if (rc != HADPSGD_OK) return rc;
    *out_bytes = L.total_bytes;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_layout(int S, int G, const int64_t* seg_len, int n_seg, hadpsgd_dtypes dt,
                              int64_t* seg_offset, int64_t* P_padded, size_t* w_off, size_t* v_off,
                              size_t* g_off, size_t* wb_off) {
    hadpsgd::Layout L;
    int rc = hadpsgd::compute_layout(S, G, seg_len, n_seg, dt, &L, nullptr);
    if (rc != HADPSGD_OK) return rc;
    if (seg_offset) for (int k = 0; k < n_seg; ++k) seg_offset[k] = L.seg_offset[k];
    if (P_padded) *P_padded = L.P_padded;
    if (w_off) *w_off = L.w_off;
    if (v_off) *v_off = L.v_off;
    if (g_off) *g_off = L.g_off;
    if (wb_off) *wb_off = L.wb_off;
    return HADPSGD_OK;
}
