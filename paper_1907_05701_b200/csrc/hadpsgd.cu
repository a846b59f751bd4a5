// hadpsgd.cu -- B2/B1: the C ABI of include/hadpsgd.h over the fused step kernel.
// sm_100a only: hadpsgd_create() refuses any device whose compute capability is not 10.x.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "internal.h"
#include "step_dispatch.cuh"

using namespace hadpsgd;

struct hadpsgd_ctx {
    Layout L;
    uint32_t flags = 0;
    int device = 0;
    int num_sms = 0;
    cudaStream_t stream = nullptr;
    cudaStream_t copy_stream = nullptr;   // host path: H2D copies overlap the kernel
    std::vector<cudaEvent_t> chunk_events;
    std::vector<std::pair<const void*, int>> occupancy;   // per kernel instantiation, queried once
    std::vector<std::pair<const void*, size_t>> smem_optin; // largest dynamic smem opted in per kernel
    std::vector<int32_t> w_slot;                           // slot (buffer index) that holds w_s right now
    char* arena = nullptr;
    bool owns_arena = false;
    double* d_partials = nullptr;
    double* d_diag = nullptr;
    unsigned int* d_ticket = nullptr;
    uint64_t last_step_k = 0;
    int last_n_pairs = 0;
    uint64_t launches = 0;
    int blocks_per_sm = 0;   // tuning override of the persistent grid (0 = the plan's default)
    std::string err;
};

static thread_local std::string g_create_error;

#define CUDA_TRY(h, call)                                                                   \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess) {                                                            \
            (h)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                  \
            return HADPSGD_CUDA;                                                            \
        }                                                                                   \
    } while (0)

// ---- kernel dispatch -------------------------------------------------------------------
namespace {

// Entry points that enqueue work make the handle's device current for their duration, so a
// process that drives several GPUs may call them from any current device.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int want) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != want) switched = cudaSetDevice(want) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

int launch_chunk(hadpsgd_ctx* h, const WorkItem* items, int n_items, int mode, bool shared_slots, float lr, float mu,
                 int64_t elem_begin, int64_t elem_end, bool accumulate) {
    const bool bf16 = h->L.grad_dtype == HADPSGD_BF16;
    const bool exact = h->flags & HADPSGD_DETERMINISTIC;
    const bool diag = !(h->flags & HADPSGD_NO_DIAG);
    const bool emit = h->L.working_dtype == HADPSGD_BF16;
    const bool shared = shared_slots && mode == kPair;   // pair members share weight slots
    LaunchPlan plan = emit ? (bf16 ? plan_bf16_emit(h->L.G, exact, diag, mode, shared) : plan_f32_emit(h->L.G, exact, diag, mode, shared))
                           : (bf16 ? plan_bf16(h->L.G, exact, diag, mode, shared) : plan_f32(h->L.G, exact, diag, mode, shared));

    const int unit = bf16 ? 16 : 8;   // elements per 32-byte gradient vector
    StepArgs a;
    a.w = reinterpret_cast<float*>(h->arena + h->L.w_off);
    a.v = reinterpret_cast<float*>(h->arena + h->L.v_off);
    a.g = h->arena + h->L.g_off;
    a.wb = emit ? h->arena + h->L.wb_off : nullptr;
    a.P = h->L.P_padded;
    a.unit_begin = elem_begin / unit;
    a.unit_end = elem_end / unit;
    a.G = h->L.G;
    a.n_work = n_items;
    a.lr = lr; a.mu = mu;
    a.invG = 1.0f / static_cast<float>(h->L.G);   // fp32 reciprocal, exact for G = 1,2,4,8 (R5)
    a.accumulate_diag = accumulate ? 1 : 0;
    a.S = h->L.S;
    a.partials = h->d_partials; a.diag = h->d_diag; a.ticket = h->d_ticket;
    for (int j = 0; j < n_items; ++j)
        a.work[j] = pack_item(items[j].s, items[j].p, items[j].ws, items[j].wp, items[j].wo_s, items[j].wo_p);

    int occ = 0;
    for (const auto& kv : h->occupancy) if (kv.first == plan.fn) occ = kv.second;
    if (occ == 0) {
        CUDA_TRY(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, plan.fn, plan.threads, 0));
        if (occ < 1) occ = 1;
        h->occupancy.emplace_back(plan.fn, occ);
    }
    // per-warp diagnostic accumulators: [warps][items][5] doubles of dynamic shared memory
    const size_t smem = diag ? static_cast<size_t>(plan.threads / 32) * n_items * kDiagQuantities * sizeof(double) : 0;
    if (smem > 48 * 1024) {
        size_t have = 0;
        for (const auto& kv : h->smem_optin) if (kv.first == plan.fn) have = kv.second;
        if (have < smem) {
            CUDA_TRY(h, cudaFuncSetAttribute(plan.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
            h->smem_optin.emplace_back(plan.fn, smem);
        }
    }
    int bps = h->blocks_per_sm > 0 ? h->blocks_per_sm : plan.blocks_per_sm;
    if (bps > occ) bps = occ;                      // persistent grid: never more than fit at once
    long long n_units = a.unit_end - a.unit_begin;
    long long want = (n_units + plan.tile_units - 1) / plan.tile_units * a.n_work;   // (item, tile) pairs
    long long grid = static_cast<long long>(h->num_sms) * bps;
    if (grid > want) grid = want;
    if (grid > kMaxGridBlocks) grid = kMaxGridBlocks;
    if (grid < 1) grid = 1;

    void* params[] = {&a};
    CUDA_TRY(h, cudaLaunchKernel(plan.fn, dim3(static_cast<unsigned>(grid)), dim3(plan.threads), params, smem, h->stream));
    h->launches++;
    return HADPSGD_OK;
}

// All items of one mode over [elem_begin, elem_end); more than kMaxWork items (S > 480 unmixed
// super-learners) take several launches.
int launch_items(hadpsgd_ctx* h, const std::vector<WorkItem>& items, int mode, bool shared_slots, float lr, float mu,
                 int64_t elem_begin, int64_t elem_end, bool accumulate) {
    if (elem_end <= elem_begin) return HADPSGD_OK;
    for (size_t first = 0; first < items.size(); first += kMaxWork) {
        const int n = static_cast<int>(items.size() - first < static_cast<size_t>(kMaxWork) ? items.size() - first : kMaxWork);
        int rc = launch_chunk(h, items.data() + first, n, mode, shared_slots, lr, mu, elem_begin, elem_end, accumulate);
        if (rc != HADPSGD_OK) return rc;
    }
    return HADPSGD_OK;
}

// The launches of one step over the element range [elem_begin, elem_end).
struct StepPlan { std::vector<WorkItem> pairs, singles; bool shared = false; };

int step_range(hadpsgd_ctx* h, const StepPlan& sp, float lr, float mu, int64_t elem_begin, int64_t elem_end,
               bool accumulate) {
    const int pair_mode = (h->flags & HADPSGD_EQ7_LITERAL) ? kPairEq7 : kPair;
    int rc = launch_items(h, sp.pairs, pair_mode, sp.shared, lr, mu, elem_begin, elem_end, accumulate);
    if (rc != HADPSGD_OK) return rc;
    // unmixed super-learners (S == 1, NO_MIX, or partner[s] == s in a custom matching)
    return launch_items(h, sp.singles, kSingle, false, lr, mu, elem_begin, elem_end, accumulate);
}

// Copies weight slot src to slot dst (and the bf16 working copy with it) on the handle's stream.
int copy_slots(hadpsgd_ctx* h, const std::vector<SlotCopy>& copies) {
    for (const SlotCopy& c : copies) {
        char* wbase = h->arena + h->L.w_off;
        CUDA_TRY(h, cudaMemcpyAsync(wbase + static_cast<size_t>(c.dst) * h->L.w_stride_bytes(),
                                    wbase + static_cast<size_t>(c.src) * h->L.w_stride_bytes(), h->L.w_stride_bytes(),
                                    cudaMemcpyDeviceToDevice, h->stream));
        if (h->L.working_dtype == HADPSGD_BF16) {
            char* bbase = h->arena + h->L.wb_off;
            const size_t nb = static_cast<size_t>(h->L.P_padded) * 2;
            CUDA_TRY(h, cudaMemcpyAsync(bbase + c.dst * nb, bbase + c.src * nb, nb, cudaMemcpyDeviceToDevice, h->stream));
        }
    }
    return HADPSGD_OK;
}

// Matching -> work items with weight slots (updates h->w_slot) and enqueues any un-sharing copies.
int plan_and_prepare(hadpsgd_ctx* h, const int32_t* partner, StepPlan* sp) {
    const bool share = h->flags & HADPSGD_SHARE_PAIR_WEIGHTS;
    std::vector<SlotCopy> copies;
    plan_step(h->L.S, partner, share, &h->w_slot, &sp->pairs, &sp->singles, &copies);
    sp->shared = share;
    h->last_n_pairs = static_cast<int>(sp->pairs.size());
    return copy_slots(h, copies);
}

int build_partner(hadpsgd_ctx* h, uint64_t step_k, const int32_t* custom, std::vector<int32_t>* partner) {
    const int S = h->L.S;
    partner->resize(S);
    if (custom) {
        if (validate_matching(S, custom) != HADPSGD_OK) { h->err = "partner[] is not a matching"; return HADPSGD_INVALID_ARG; }
        std::memcpy(partner->data(), custom, sizeof(int32_t) * S);
    } else if (h->flags & HADPSGD_NO_MIX) {
        for (int s = 0; s < S; ++s) (*partner)[s] = s;
    } else if (ring_partner(S, step_k, partner->data()) != HADPSGD_OK) {
        h->err = "odd S > 1 has no perfect ring matching (PAPER.md:66 needs two 0.5s per row): use "
                 "hadpsgd_step_matching with an unpaired member (T_ii = 1) or HADPSGD_NO_MIX";
        return HADPSGD_INVALID_ARG;
    }
    return HADPSGD_OK;
}

}  // namespace

// ---- C ABI -----------------------------------------------------------------------------

extern "C" int hadpsgd_create(int S, int G, const int64_t* seg_len, int n_seg, hadpsgd_dtypes dt,
                              const hadpsgd_opts* opts, hadpsgd_handle* out) {
    if (!out) { g_create_error = "out handle is NULL"; return HADPSGD_INVALID_ARG; }
    *out = nullptr;
    Layout L;
    std::string why;
    int rc = compute_layout(S, G, seg_len, n_seg, dt, &L, &why);
    if (rc != HADPSGD_OK) { g_create_error = why; return rc; }
    const uint32_t flags = opts ? opts->flags : 0u;
    int dev = (opts && opts->device >= 0) ? opts->device : -1;
    cudaError_t e;
    if (dev < 0) {
        e = cudaGetDevice(&dev);
        if (e != cudaSuccess) { g_create_error = std::string("no CUDA device: ") + cudaGetErrorString(e); return HADPSGD_CUDA; }
    }
    DeviceGuard guard(dev);   // the caller's current device is restored on return
    int now = -1;
    e = cudaGetDevice(&now);
    if (e != cudaSuccess || now != dev) {
        g_create_error = "cannot select CUDA device " + std::to_string(dev) + (e != cudaSuccess ? std::string(": ") + cudaGetErrorString(e) : "");
        cudaGetLastError();
        return HADPSGD_CUDA;
    }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) { g_create_error = cudaGetErrorString(e); return HADPSGD_CUDA; }
    if (prop.major != 10) {
        g_create_error = "libhadpsgd is built for sm_100a only; device is sm_" + std::to_string(prop.major) + std::to_string(prop.minor);
        return HADPSGD_UNSUPPORTED_DEVICE;
    }

    if ((flags & HADPSGD_SHARE_PAIR_WEIGHTS) && (flags & (HADPSGD_NO_MIX | HADPSGD_EQ7_LITERAL))) {
        g_create_error = "HADPSGD_SHARE_PAIR_WEIGHTS needs pair members that end a step with identical weights: "
                         "not with NO_MIX or EQ7_LITERAL";
        return HADPSGD_INVALID_ARG;
    }
    hadpsgd_ctx* h = new hadpsgd_ctx();
    h->w_slot.resize(S);
    for (int s = 0; s < S; ++s) h->w_slot[s] = s;
    h->L = L; h->flags = flags; h->device = dev; h->num_sms = prop.multiProcessorCount;
    h->stream = opts ? static_cast<cudaStream_t>(opts->stream) : nullptr;
    if (opts && opts->arena) {
        if (opts->arena_bytes < L.total_bytes || (reinterpret_cast<uintptr_t>(opts->arena) % kRegionAlign) != 0) {
            g_create_error = "arena too small or not 256 B aligned"; delete h; return HADPSGD_OUT_OF_MEMORY;
        }
        h->arena = static_cast<char*>(opts->arena);
    } else {
        void* p = nullptr;
        e = cudaMalloc(&p, L.total_bytes);
        if (e != cudaSuccess) { g_create_error = std::string("cudaMalloc: ") + cudaGetErrorString(e); delete h; return HADPSGD_OUT_OF_MEMORY; }
        h->arena = static_cast<char*>(p); h->owns_arena = true;
    }
    e = cudaMemsetAsync(h->arena, 0, L.total_bytes, h->stream);   // zero w, v, grads, padding, scratch
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking);
    if (e != cudaSuccess) {
        g_create_error = std::string("init: ") + cudaGetErrorString(e);
        if (h->owns_arena) cudaFree(h->arena);
        delete h; return HADPSGD_CUDA;
    }
    char* aux = h->arena + L.aux_off;
    h->d_partials = reinterpret_cast<double*>(aux);
    h->d_diag = h->d_partials + static_cast<size_t>(S) * kDiagQuantities * kMaxGridBlocks;
    h->d_ticket = reinterpret_cast<unsigned int*>(h->d_diag + 3 * S);
    *out = h;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_destroy(hadpsgd_handle h) {
    if (!h) return HADPSGD_INVALID_ARG;
    DeviceGuard guard(h->device);
    cudaStreamSynchronize(h->stream);
    for (cudaEvent_t ev : h->chunk_events) cudaEventDestroy(ev);
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    if (h->owns_arena) cudaFree(h->arena);
    delete h;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_step(hadpsgd_handle h, float lr, float momentum, uint64_t step_k) {
    return hadpsgd_step_matching(h, lr, momentum, step_k, nullptr);
}

extern "C" int hadpsgd_step_matching(hadpsgd_handle h, float lr, float momentum, uint64_t step_k,
                                     const int32_t* partner) {
    if (!h) return HADPSGD_INVALID_ARG;
    DeviceGuard guard(h->device);
    std::vector<int32_t> pt;
    int rc = build_partner(h, step_k, partner, &pt);
    if (rc != HADPSGD_OK) return rc;
    h->last_step_k = step_k;
    StepPlan sp;
    rc = plan_and_prepare(h, pt.data(), &sp);
    if (rc != HADPSGD_OK) return rc;
    return step_range(h, sp, lr, momentum, 0, h->L.P_padded, false);
}

extern "C" int hadpsgd_step_host(hadpsgd_handle h, const void* const* host_grads, float lr,
                                 float momentum, uint64_t step_k, hadpsgd_diag* diag_out) {
    if (!h || !host_grads) return HADPSGD_INVALID_ARG;
    DeviceGuard guard(h->device);
    std::vector<int32_t> pt;
    int rc = build_partner(h, step_k, nullptr, &pt);
    if (rc != HADPSGD_OK) return rc;
    h->last_step_k = step_k;
    const int n_buf = h->L.S * h->L.G;
    for (int b = 0; b < n_buf; ++b) if (!host_grads[b]) { h->err = "host_grads[] has a NULL entry"; return HADPSGD_INVALID_ARG; }

    StepPlan sp;                      // one slot plan for the whole step, shared by all chunks
    rc = plan_and_prepare(h, pt.data(), &sp);
    if (rc != HADPSGD_OK) return rc;

    // Chunk the element range so the H2D copy of chunk c+1 overlaps the kernel on chunk c.
    const int64_t P = h->L.P_padded;
    const size_t eb = h->L.grad_elem_bytes();
    int64_t chunk = (int64_t(8) << 20);                       // 8 Mi elements per learner per chunk
    chunk = chunk / HADPSGD_SEG_ALIGN_ELEMS * HADPSGD_SEG_ALIGN_ELEMS;
    const int n_chunks = static_cast<int>((P + chunk - 1) / chunk);
    while (static_cast<int>(h->chunk_events.size()) < n_chunks + 1) {
        cudaEvent_t ev;
        CUDA_TRY(h, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        h->chunk_events.push_back(ev);
    }
    // the copy stream must not overwrite gradients an earlier step on h->stream still reads
    CUDA_TRY(h, cudaEventRecord(h->chunk_events[n_chunks], h->stream));
    CUDA_TRY(h, cudaStreamWaitEvent(h->copy_stream, h->chunk_events[n_chunks], 0));
    char* gdev = h->arena + h->L.g_off;
    for (int c = 0; c < n_chunks; ++c) {
        const int64_t e0 = c * chunk, e1 = (e0 + chunk < P) ? e0 + chunk : P;
        for (int b = 0; b < n_buf; ++b)
            CUDA_TRY(h, cudaMemcpyAsync(gdev + static_cast<size_t>(b) * h->L.g_stride_bytes() + e0 * eb,
                                        static_cast<const char*>(host_grads[b]) + e0 * eb,
                                        static_cast<size_t>(e1 - e0) * eb, cudaMemcpyHostToDevice, h->copy_stream));
        CUDA_TRY(h, cudaEventRecord(h->chunk_events[c], h->copy_stream));
        CUDA_TRY(h, cudaStreamWaitEvent(h->stream, h->chunk_events[c], 0));
        rc = step_range(h, sp, lr, momentum, e0, e1, c > 0);
        if (rc != HADPSGD_OK) return rc;
    }
    if (diag_out) return hadpsgd_diagnostics(h, diag_out);
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return HADPSGD_OK;
}

extern "C" int hadpsgd_weights(hadpsgd_handle h, int s, float** dev_ptr) {
    if (!h || !dev_ptr || s < 0 || s >= h->L.S) return HADPSGD_INVALID_ARG;
    *dev_ptr = reinterpret_cast<float*>(h->arena + h->L.w_off + static_cast<size_t>(h->w_slot[s]) * h->L.w_stride_bytes());
    return HADPSGD_OK;
}
extern "C" int hadpsgd_momentum(hadpsgd_handle h, int s, float** dev_ptr) {
    if (!h || !dev_ptr || s < 0 || s >= h->L.S) return HADPSGD_INVALID_ARG;
    *dev_ptr = reinterpret_cast<float*>(h->arena + h->L.v_off + static_cast<size_t>(s) * h->L.w_stride_bytes());
    return HADPSGD_OK;
}
extern "C" int hadpsgd_weights_bf16(hadpsgd_handle h, int s, void** dev_ptr) {
    if (!h || !dev_ptr || s < 0 || s >= h->L.S) return HADPSGD_INVALID_ARG;
    if (h->L.working_dtype != HADPSGD_BF16) { h->err = "handle was created without a bf16 working copy (dtypes.working_dtype)"; return HADPSGD_INVALID_ARG; }
    *dev_ptr = h->arena + h->L.wb_off + static_cast<size_t>(h->w_slot[s]) * static_cast<size_t>(h->L.P_padded) * 2;
    return HADPSGD_OK;
}
extern "C" int hadpsgd_grads(hadpsgd_handle h, int s, int g, void** dev_ptr) {
    if (!h || !dev_ptr || s < 0 || s >= h->L.S || g < 0 || g >= h->L.G) return HADPSGD_INVALID_ARG;
    *dev_ptr = h->arena + h->L.g_off + (static_cast<size_t>(s) * h->L.G + g) * h->L.g_stride_bytes();
    return HADPSGD_OK;
}
extern "C" int hadpsgd_segment(hadpsgd_handle h, int seg, int64_t* elem_offset, int64_t* elem_len) {
    if (!h || seg < 0 || seg >= h->L.n_seg) return HADPSGD_INVALID_ARG;
    if (elem_offset) *elem_offset = h->L.seg_offset[seg];
    if (elem_len) *elem_len = h->L.seg_len[seg];
    return HADPSGD_OK;
}
extern "C" int hadpsgd_padded_len(hadpsgd_handle h, int64_t* P_padded) {
    if (!h || !P_padded) return HADPSGD_INVALID_ARG;
    *P_padded = h->L.P_padded;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_diagnostics(hadpsgd_handle h, hadpsgd_diag* host_out) {
    if (!h || !host_out) return HADPSGD_INVALID_ARG;
    if (h->flags & HADPSGD_NO_DIAG) { h->err = "handle was created with HADPSGD_NO_DIAG"; return HADPSGD_INVALID_ARG; }
    DeviceGuard guard(h->device);
    const int S = h->L.S;
    std::vector<double> tmp(3 * S);
    CUDA_TRY(h, cudaMemcpyAsync(tmp.data(), h->d_diag, sizeof(double) * 3 * S, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    host_out->S = S; host_out->n_pairs = h->last_n_pairs; host_out->step_k = h->last_step_k;
    std::memcpy(host_out->gsq, tmp.data(), sizeof(double) * S);
    std::memcpy(host_out->wsq, tmp.data() + S, sizeof(double) * S);
    std::memcpy(host_out->gap, tmp.data() + 2 * S, sizeof(double) * S);
    return HADPSGD_OK;
}

namespace hadpsgd {
int launch_consensus(const float* w, long long P_padded, int S, const int32_t* w_slot, int num_sms,
                     double* block_out, cudaStream_t stream, cudaError_t* err);   // consensus.cu
}

extern "C" int hadpsgd_unshare(hadpsgd_handle h) {
    if (!h) return HADPSGD_INVALID_ARG;
    DeviceGuard guard(h->device);
    std::vector<SlotCopy> copies;
    plan_unshare(h->L.S, &h->w_slot, &copies);
    return copy_slots(h, copies);
}

extern "C" int hadpsgd_consensus(hadpsgd_handle h, double* D_out) {
    if (!h || !D_out) return HADPSGD_INVALID_ARG;
    DeviceGuard guard(h->device);
    // the partials scratch is free between steps: everything is ordered on h->stream
    cudaError_t e = cudaSuccess;
    const int grid = launch_consensus(reinterpret_cast<const float*>(h->arena + h->L.w_off), h->L.P_padded, h->L.S,
                                      h->w_slot.data(), h->num_sms, h->d_partials, h->stream, &e);
    CUDA_TRY(h, e);
    h->launches++;
    std::vector<double> part(grid);
    CUDA_TRY(h, cudaMemcpyAsync(part.data(), h->d_partials, sizeof(double) * grid, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    double D = 0.;
    for (int b = 0; b < grid; ++b) D += part[b];   // fixed order: run-to-run deterministic
    *D_out = D;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_set_launch(hadpsgd_handle h, int blocks_per_sm) {
    if (!h || blocks_per_sm < 0 || blocks_per_sm > 16) return HADPSGD_INVALID_ARG;
    h->blocks_per_sm = blocks_per_sm;
    return HADPSGD_OK;
}
extern "C" int hadpsgd_launch_count(hadpsgd_handle h, uint64_t* out) {
    if (!h || !out) return HADPSGD_INVALID_ARG;
    *out = h->launches;
    return HADPSGD_OK;
}

extern "C" const char* hadpsgd_error_string(int code) {
    switch (code) {
        case HADPSGD_OK: return "ok";
        case HADPSGD_INVALID_ARG: return "invalid argument";
        case HADPSGD_OUT_OF_MEMORY: return "out of device memory";
        case HADPSGD_CUDA: return "CUDA error";
        case HADPSGD_UNSUPPORTED_DEVICE: return "unsupported device (sm_100a required)";
        default: return "unknown status";
    }
}
extern "C" const char* hadpsgd_last_error(hadpsgd_handle h) {
    return h ? h->err.c_str() : g_create_error.c_str();
}
