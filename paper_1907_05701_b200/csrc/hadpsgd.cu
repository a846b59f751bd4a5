// hadpsgd.cu -- B2/B1: the C ABI of include/hadpsgd.h over the fused step kernel.
// sm_100a only: hadpsgd_create() refuses any device whose compute capability is not 10.x.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "internal.h"
#include "step_dispatch.cuh"

using namespace hadpsgd;

// The launches of one step: pair items, then unmixed / publishing single items.
struct StepPlan { std::vector<WorkItem> pairs, singles; bool shared = false; };

struct hadpsgd_ctx {
    Layout L;
    uint32_t flags = 0;
    int device = 0;
    int num_sms = 0;
    cudaStream_t stream = nullptr;
    cudaStream_t copy_stream = nullptr;   // host path: H2D copies overlap the kernel
    std::vector<cudaEvent_t> chunk_events;
    std::vector<std::pair<const void*, int>> occupancy;   // per kernel instantiation, queried once
    std::vector<int32_t> w_slot;                           // slot (buffer index) that holds w_s right now
    char* arena = nullptr;
    bool owns_arena = false;
    TaggedDouble* d_partials = nullptr;   // step kernel: block partials with their launch tag
    double* d_scratch = nullptr;           // consensus / flush kernels: block partials, plain doubles
    double* d_diag = nullptr;
    bool walk_reverse = false;             // direction of the kernel's walk; flips with every step (L2 reuse)
    const bool serpentine = true;          // fixed choices of the build: nothing is read from the environment
    const size_t keep_bytes = size_t(64) << 20;  // bytes stored at the end of a step's walk that stay in L2
    bool in_host_step = false;             // hadpsgd_step_host is enqueuing (its launches follow event waits)
    const bool use_pdl = true;             // launch steps with programmatic stream serialization
    uint32_t diag_tag = 0;                 // tag of the block partials of the most recent launch (never 0)
    uint64_t last_step_k = 0;
    int last_n_pairs = 0;
    uint64_t launches = 0;
    int blocks_per_sm = 0;   // tuning override of the persistent grid (0 = the plan's default)
    bool diag_on = true;     // hadpsgd_set_diagnostics: a5 computed by the steps that follow (never with NO_DIAG)
    uint64_t diag_step_k = 0;   // step_k of the most recent step that computed diagnostics
    // scratch of the step calls: sized by the first step, reused afterwards (no host allocation per step)
    std::vector<int32_t> partner, new_slot, new_pending;
    std::vector<SlotCopy> copies;
    std::vector<double> diag_host;      // hadpsgd_diagnostics: landing buffer of the device results
    std::vector<WorkItem> part[2][2];   // peer mode: [pairs | singles][plain | pending]
    StepPlan plan;
    // super-learner partition (HADPSGD_PEER)
    bool peer_init = false, peer_table_dirty = true;
    int rank = 0, world = 1, S_global = 0;
    std::vector<int32_t> rank_begin;
    std::vector<const float*> stage_of_rank;   // [world] stage regions as seen from this process
    std::vector<int32_t> pending;              // [S] global partner whose stage completes w_s, or -1
    uint64_t epoch = 0;
    const float** d_peer = nullptr;            // device table [2][S_global]
    // neighbour-only epoch handshake: war_until[parity][q] = value rank q's epoch word must have reached before this
    // handle overwrites its stage buffers of that parity again (0: no reader outstanding)
    std::vector<uint32_t> war_until[2], wait_value;
    std::vector<void*> ipc_mapped;             // [world] the cudaIpcOpenMemHandle mapping of rank r (nullptr: none); closed on re-attach and at destroy
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

namespace hadpsgd {
int launch_consensus(const float* w, long long P_padded, int S, const int32_t* w_slot, int num_sms,
                     double* block_out, cudaStream_t stream, cudaError_t* err);   // consensus.cu
int launch_peer_flush(float* w_main, const float* a_stage, const float* const* peer, const int32_t* members,
                      int n_members, long long P_padded, int S, int num_sms, double* partials, double* diag,
                      cudaStream_t stream, cudaError_t* err);                     // peer_flush.cu
}

// ---- kernel dispatch -------------------------------------------------------------------
namespace {

constexpr size_t kKeepMaxStepBytes = size_t(2) << 30;

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

bool is_peer(const hadpsgd_ctx* h) { return (h->flags & HADPSGD_PEER) != 0; }

int launch_chunk(hadpsgd_ctx* h, const WorkItem* items, int n_items, int mode, int wmode_req, float lr, float mu,
                 int64_t elem_begin, int64_t elem_end, bool accumulate) {
    const bool bf16 = h->L.grad_dtype == HADPSGD_BF16;
    const bool exact = h->flags & HADPSGD_DETERMINISTIC;
    const bool diag = !(h->flags & HADPSGD_NO_DIAG) && h->diag_on;
    const bool emit = h->L.working_dtype == HADPSGD_BF16;
    const int wmode = (wmode_req == kSlots && mode != kPair) ? kOwn : wmode_req;
    LaunchPlan plan = emit ? (bf16 ? plan_bf16_emit(h->L.G, exact, diag, mode, wmode) : plan_f32_emit(h->L.G, exact, diag, mode, wmode))
                           : (bf16 ? plan_bf16(h->L.G, exact, diag, mode, wmode) : plan_f32(h->L.G, exact, diag, mode, wmode));
    if (!plan.fn) { h->err = "this combination of flags has no kernel"; return HADPSGD_INVALID_ARG; }

    const int unit = bf16 ? 16 : 8;   // elements per 32-byte gradient vector
    StepArgs a;
    a.w = reinterpret_cast<float*>(h->arena + h->L.w_off);
    a.v = reinterpret_cast<float*>(h->arena + h->L.v_off);
    a.g = h->arena + h->L.g_off;
    a.wb = emit ? h->arena + h->L.wb_off : nullptr;
    a.peer = h->d_peer;
    a.P = h->L.P_padded;
    a.unit_begin = elem_begin / unit;
    a.unit_end = elem_end / unit;
    a.G = h->L.G;
    a.n_work = n_items;
    a.lr = lr; a.mu = mu;
    a.invG = 1.0f / static_cast<float>(h->L.G);   // fp32 reciprocal, exact for G = 1,2,4,8 (R5)
    a.accumulate_diag = accumulate ? 1 : 0;
    a.reverse = h->walk_reverse ? 1 : 0;
    a.S = h->L.S;
    a.partials = h->d_partials; a.diag = h->d_diag;
    a.timeout_flag = reinterpret_cast<unsigned int*>(h->d_diag + kDiagArrays * h->L.S);   // first spare word behind the results
    if (++h->diag_tag == 0) h->diag_tag = 1;   // a tag is never 0 (zero = empty slot)
    a.tag = h->diag_tag;
    for (int j = 0; j < n_items; ++j) {
        const WorkItem& it = items[j];
        a.items[j] = {static_cast<unsigned short>(it.s), static_cast<unsigned short>(it.p),
                      static_cast<unsigned short>(it.ws), static_cast<unsigned short>(it.wp),
                      static_cast<unsigned short>(it.wo_s), static_cast<unsigned short>(it.wo_p),
                      static_cast<unsigned short>(it.b_s), static_cast<unsigned short>(it.b_p)};
    }

    // per-warp diagnostic accumulators [warps][items][quantities].  At most 18 KB: no opt-in needed.
    const int nq = plan.wmode == kPeer ? kNQPeer : kNQ;
    const size_t smem = diag ? static_cast<size_t>(plan.threads / 32) * n_items * nq * sizeof(double) : 0;
    int occ = 0;
    for (const auto& kv : h->occupancy) if (kv.first == plan.fn) occ = kv.second;
    if (occ == 0) {   // with the largest shared-memory footprint this kernel can be launched with
        const size_t worst = diag ? static_cast<size_t>(plan.threads / 32) * kInlineItems * nq * sizeof(double) : 0;
        CUDA_TRY(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, plan.fn, plan.threads, worst));
        if (occ < 1) occ = 1;
        h->occupancy.emplace_back(plan.fn, occ);
    }
    int bps = h->blocks_per_sm > 0 ? h->blocks_per_sm : plan.blocks_per_sm;
    if (bps > occ) bps = occ;                      // persistent grid: never more than fit at once
    long long n_units = a.unit_end - a.unit_begin;
    const long long n_tiles = (n_units + plan.tile_units - 1) / plan.tile_units;
    // shared slots: a block owns whole tiles (and walks every item of each); else (item, tile) pairs
    long long want = plan.wmode == kChain ? n_tiles : n_tiles * a.n_work;
    long long grid = static_cast<long long>(h->num_sms) * bps;
    // a problem that fits ONE wave of resident blocks runs as one wave (every block exactly one tile,
    // all tiles in flight at once) instead of some blocks walking two tiles one after the other:
    // 2^18 parameters x 4 x 4 fp32 takes 5.9 instead of 7.2 us per step
    if (h->blocks_per_sm == 0 && want <= static_cast<long long>(h->num_sms) * occ) grid = want;
    if (grid > want) grid = want;
    if (grid > kMaxGridBlocks) grid = kMaxGridBlocks;
    if (grid < 1) grid = 1;
    // how many blocks work on any one item (the collecting block sums exactly their partials)
    long long per = grid;
    if (plan.wmode == kSlots) {                      // tile-major walk: blocks (i * n_work + j) mod grid
        long long x = a.n_work, y = grid;
        while (y) { const long long t = x % y; x = y; y = t; }   // x = gcd(n_work, grid)
        per = grid / x;
    }
    // Stores of the last part of the walk keep the default L2 policy -- the next step, walking the other
    // way, begins with them -- everything before is evict_first.  The budget is in bytes STORED (a share
    // of the 126 MB L2; where all of w and v fit they never travel to HBM at all); a step that moves
    // more than kKeepMaxStepBytes gains nothing and loses 2-4 % (the kept lines shrink the L2 left for
    // streaming), so it keeps nothing.
    {
        const long long walk_len = plan.wmode == kChain ? n_tiles : n_tiles * a.n_work;
        const size_t members = mode == kSingle ? 1 : 2;
        const size_t per_walk_pos = static_cast<size_t>(plan.tile_units) * 32 * members * (plan.wmode == kChain ? a.n_work : 1);
        const size_t store_bytes = per_walk_pos * (bf16 ? 4 : 2) + (emit ? per_walk_pos * (bf16 ? 2 : 1) / 2 : 0);   // w, v (+ the bf16 copy of w)
        const size_t all_bytes = per_walk_pos * (h->L.G + (bf16 ? 8 : 4));
        long long keep_tiles = 0;
        if (h->serpentine && all_bytes * static_cast<size_t>(walk_len) < kKeepMaxStepBytes)
            keep_tiles = static_cast<long long>(h->keep_bytes / (store_bytes ? store_bytes : 1));
        if (keep_tiles > walk_len) keep_tiles = walk_len;
        a.keep_from = walk_len - keep_tiles;
    }
    a.touch_count = static_cast<int>(plan.wmode == kChain ? grid : (n_tiles < per ? n_tiles : per));
    void* params[] = {&a};
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(grid));
    cfg.blockDim = dim3(plan.threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = h->stream;
    // programmatic dependent launch: the kernel itself waits (griddepcontrol.wait) for the launch before it
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = (h->use_pdl && !h->in_host_step) ? 1 : 0;   // chunk launches wait on copy events: plain launches
    CUDA_TRY(h, cudaLaunchKernelExC(&cfg, plan.fn, params));
    h->launches++;
    return HADPSGD_OK;
}

// All items of one mode over [elem_begin, elem_end); more than kInlineItems items (S > 64 paired or
// S > 32 unmixed super-learners) take several launches.
int launch_items(hadpsgd_ctx* h, const std::vector<WorkItem>& items, int mode, int wmode, float lr, float mu,
                 int64_t elem_begin, int64_t elem_end, bool accumulate) {
    if (elem_end <= elem_begin) return HADPSGD_OK;
    for (size_t first = 0; first < items.size(); first += kInlineItems) {
        const int n = static_cast<int>(items.size() - first < static_cast<size_t>(kInlineItems) ? items.size() - first : kInlineItems);
        int rc = launch_chunk(h, items.data() + first, n, mode, wmode, lr, mu, elem_begin, elem_end, accumulate);
        if (rc != HADPSGD_OK) return rc;
    }
    return HADPSGD_OK;
}

// The launches of one step over the element range [elem_begin, elem_end).
int step_range(hadpsgd_ctx* h, const StepPlan& sp, float lr, float mu, int64_t elem_begin, int64_t elem_end,
               bool accumulate) {
    const int pair_mode = (h->flags & HADPSGD_EQ7_LITERAL) ? kPairEq7 : kPair;
    if (!is_peer(h)) {
        int rc = launch_items(h, sp.pairs, pair_mode, sp.shared ? kSlots : kOwn, lr, mu, elem_begin, elem_end, accumulate);
        if (rc != HADPSGD_OK) return rc;
        // unmixed super-learners (S == 1, NO_MIX, or partner[s] == s in a custom matching)
        return launch_items(h, sp.singles, kSingle, kOwn, lr, mu, elem_begin, elem_end, accumulate);
    }
    // Peer mode.  Only items that first have to resolve a pending mix need the kPeer kernel (two more
    // loads per member, more registers).  A pair without one reads and writes its members' main
    // buffers -- exactly the kOwn pair kernel -- and a single without one (unmixed, or publishing u for
    // a partner in another arena) is the ordinary kSingle kernel, which addresses weights through the
    // item's buffer indices anyway.  Each kernel writes pend_wsq / pend_gap of its own members (the plain
    // ones write 0), so the up to four launches of a step follow one another with nothing in between.
    for (auto& row : h->part) for (auto& v : row) v.clear();   // [pairs | singles][plain | pending]
    for (const WorkItem& it : sp.pairs) h->part[0][(it.b_s || it.b_p) ? 1 : 0].push_back(it);
    for (const WorkItem& it : sp.singles) h->part[1][it.b_s ? 1 : 0].push_back(it);
    for (int kind = 0; kind < 2; ++kind)
        for (int pend = 0; pend < 2; ++pend) {
            int rc = launch_items(h, h->part[kind][pend], kind == 0 ? kPair : kSingle, pend ? kPeer : kOwn, lr, mu,
                                  elem_begin, elem_end, accumulate);
            if (rc != HADPSGD_OK) return rc;
        }
    return HADPSGD_OK;
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

// (Re)builds the device table of stage-buffer pointers: entry e * S_global + s_global.
int upload_peer_table(hadpsgd_ctx* h) {
    if (!h->peer_table_dirty) return HADPSGD_OK;
    for (int r = 0; r < h->world; ++r)
        if (!h->stage_of_rank[r]) { h->err = "rank " + std::to_string(r) + " is not attached (hadpsgd_peer_attach)"; return HADPSGD_INVALID_ARG; }
    std::vector<const float*> tab(static_cast<size_t>(2) * h->S_global);
    for (int r = 0; r < h->world; ++r) {
        const int n = h->rank_begin[r + 1] - h->rank_begin[r];
        for (int e = 0; e < 2; ++e)
            for (int s = 0; s < n; ++s)
                tab[static_cast<size_t>(e) * h->S_global + h->rank_begin[r] + s] =
                    h->stage_of_rank[r] + (static_cast<size_t>(e) * n + s) * h->L.P_padded;
    }
    if (!h->d_peer) CUDA_TRY(h, cudaMalloc(reinterpret_cast<void**>(&h->d_peer), tab.size() * sizeof(float*)));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));   // no launch may still read the old table
    CUDA_TRY(h, cudaMemcpy(h->d_peer, tab.data(), tab.size() * sizeof(float*), cudaMemcpyHostToDevice));
    h->peer_table_dirty = false;
    return HADPSGD_OK;
}

// ---- neighbour-only epoch handshake (HADPSGD_PEER) -------------------------------------------------
// Every handle owns one 32-bit EPOCH WORD behind its stage buffers (Layout::epoch_off; inside the arena,
// so it is reachable wherever the stage region is: same device, peer device, CUDA IPC mapping).  After the
// last launch of its step number e (e = 0, 1, ...) a handle writes e + 1 there with a stream memory
// operation; before the first launch of a step it makes its stream wait (>=) on the words of exactly the
// ranks it exchanges stage buffers with:
//   RAW  a member whose mix with a partner in rank q is pending reads q's stage buffer of step e - 1:
//        wait word_q >= e.  (hadpsgd_peer_flush: the same.)
//   WAR  a handle that published u for a partner in rank q at step e0 must not overwrite that stage
//        parity (step e0 + 2 at the earliest) before q has read it, which q does in its step e0 + 1 (or
//        in a flush enqueued before that step): wait word_q >= e0 + 2.
// These are stream operations (cuStreamWaitValue32 / cuStreamWriteValue32): no kernel spins, nothing
// occupies an SM while waiting, so ranks that share one GPU cannot starve each other, and no rank ever
// waits for a rank that is not its partner -- there is no global barrier.
using stream_memop_fn = int (*)(cudaStream_t, unsigned long long, uint32_t, unsigned int);
struct StreamMemOps { stream_memop_fn write = nullptr, wait = nullptr; };

int get_stream_memops(hadpsgd_ctx* h, StreamMemOps* out) {
    static StreamMemOps ops;      // resolved once per process (benign race: both threads store the same pointers)
    if (!ops.write || !ops.wait) {
        void* fw = nullptr; void* fq = nullptr;
        cudaDriverEntryPointQueryResult qr;
        CUDA_TRY(h, cudaGetDriverEntryPoint("cuStreamWriteValue32", &fw, cudaEnableDefault, &qr));
        if (!fw || qr != cudaDriverEntryPointSuccess) { h->err = "cuStreamWriteValue32 is unavailable"; return HADPSGD_CUDA; }
        CUDA_TRY(h, cudaGetDriverEntryPoint("cuStreamWaitValue32", &fq, cudaEnableDefault, &qr));
        if (!fq || qr != cudaDriverEntryPointSuccess) { h->err = "cuStreamWaitValue32 is unavailable"; return HADPSGD_CUDA; }
        ops.write = reinterpret_cast<stream_memop_fn>(fw);
        ops.wait = reinterpret_cast<stream_memop_fn>(fq);
    }
    *out = ops;
    return HADPSGD_OK;
}

int owner_rank(const hadpsgd_ctx* h, int global_member) {
    int r = 0;
    while (r + 1 < h->world && global_member >= h->rank_begin[r + 1]) ++r;
    return r;
}

// Device address of rank r's epoch word, from the stage region this process attached for it.
unsigned long long epoch_word_of(const hadpsgd_ctx* h, int r) {
    const size_t n = static_cast<size_t>(h->rank_begin[r + 1] - h->rank_begin[r]);
    return reinterpret_cast<unsigned long long>(h->stage_of_rank[r]) + 2 * n * h->L.w_stride_bytes();
}

// Enqueues the waits a step (for_step) or a flush needs before its first launch.
int epoch_wait(hadpsgd_ctx* h, bool for_step) {
    if (h->world < 2) return HADPSGD_OK;
    const uint32_t e = static_cast<uint32_t>(h->epoch);
    std::vector<uint32_t>& need = h->wait_value;
    need.assign(h->world, 0);
    for (int s = 0; s < h->L.S; ++s)
        if (h->pending[s] >= 0) need[owner_rank(h, h->pending[s])] = e;                       // RAW
    if (for_step) {
        std::vector<uint32_t>& war = h->war_until[e & 1];
        for (int q = 0; q < h->world; ++q) { if (war[q] > need[q]) need[q] = war[q]; war[q] = 0; }   // WAR
    }
    StreamMemOps ops;
    for (int q = 0; q < h->world; ++q) {
        if (!need[q] || q == h->rank) continue;
        if (!ops.wait) { const int rc = get_stream_memops(h, &ops); if (rc != HADPSGD_OK) return rc; }
        if (ops.wait(h->stream, epoch_word_of(h, q), need[q], 0u /* CU_STREAM_WAIT_VALUE_GEQ */) != 0) {
            h->err = "cuStreamWaitValue32 on the epoch word of rank " + std::to_string(q) + " failed";
            return HADPSGD_CUDA;
        }
    }
    return HADPSGD_OK;
}

// After the last launch of step `epoch`: publish epoch + 1, and remember who must have read what this
// step published before its stage parity is written again.
int epoch_signal(hadpsgd_ctx* h, const std::vector<int32_t>& new_pending) {
    if (h->world < 2) return HADPSGD_OK;
    const uint32_t e = static_cast<uint32_t>(h->epoch);
    StreamMemOps ops;
    const int rc = get_stream_memops(h, &ops);
    if (rc != HADPSGD_OK) return rc;
    if (ops.write(h->stream, reinterpret_cast<unsigned long long>(h->arena + h->L.epoch_off), e + 1u, 0u) != 0) {
        h->err = "cuStreamWriteValue32 on the epoch word failed";
        return HADPSGD_CUDA;
    }
    for (int s = 0; s < h->L.S; ++s)
        if (new_pending[s] >= 0) h->war_until[e & 1][owner_rank(h, new_pending[s])] = e + 2u;
    return HADPSGD_OK;
}

// Matching -> work items with weight buffers.  Nothing of the handle's state is committed here: the
// caller commits `new_slot` / `new_pending` once every launch of the step has been enqueued.
int plan_and_prepare(hadpsgd_ctx* h, const int32_t* partner, StepPlan* sp, std::vector<int32_t>* new_slot,
                     std::vector<int32_t>* new_pending) {
    if (is_peer(h)) {
        int rc = upload_peer_table(h);
        if (rc != HADPSGD_OK) return rc;
        *new_pending = h->pending;
        rc = plan_peer_step(h->world, h->rank, h->rank_begin.data(), partner, h->epoch, new_pending, &sp->pairs, &sp->singles);
        if (rc != HADPSGD_OK) { h->err = "peer plan failed: partner[] is not a matching of the S_global members"; return rc; }
        sp->shared = false;
        return HADPSGD_OK;
    }
    const bool share = h->flags & HADPSGD_SHARE_PAIR_WEIGHTS;
    h->copies.clear();
    *new_slot = h->w_slot;
    plan_step(h->L.S, partner, share, new_slot, &sp->pairs, &sp->singles, &h->copies);
    sp->shared = share;
    return copy_slots(h, h->copies);
}

void commit_plan(hadpsgd_ctx* h, const StepPlan& sp, const std::vector<int32_t>& new_slot,
                 const std::vector<int32_t>& new_pending, uint64_t step_k) {
    h->last_step_k = step_k;
    if (h->serpentine) h->walk_reverse = !h->walk_reverse;
    if (h->diag_on) h->diag_step_k = step_k;
    h->last_n_pairs = static_cast<int>(sp.pairs.size());
    if (is_peer(h)) { h->pending = new_pending; h->epoch++; }
    else h->w_slot = new_slot;
}

int build_partner(hadpsgd_ctx* h, uint64_t step_k, const int32_t* custom, std::vector<int32_t>* partner) {
    const int S = is_peer(h) ? h->S_global : h->L.S;
    if (is_peer(h) && !h->peer_init) { h->err = "HADPSGD_PEER handle: call hadpsgd_peer_init first"; return HADPSGD_INVALID_ARG; }
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
    if (flags & HADPSGD_PEER) {
        if (flags & (HADPSGD_SHARE_PAIR_WEIGHTS | HADPSGD_EQ7_LITERAL)) {
            g_create_error = "HADPSGD_PEER cannot be combined with SHARE_PAIR_WEIGHTS or EQ7_LITERAL";
            return HADPSGD_INVALID_ARG;
        }
        if (!dt.peer_stage) { g_create_error = "HADPSGD_PEER needs dtypes.peer_stage = 1 (the stage buffers)"; return HADPSGD_INVALID_ARG; }
    }
    hadpsgd_ctx* h = new hadpsgd_ctx();
    h->w_slot.resize(S);
    for (int s = 0; s < S; ++s) h->w_slot[s] = s;
    h->pending.assign(S, -1);
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
    h->d_partials = reinterpret_cast<TaggedDouble*>(aux);
    h->d_scratch = reinterpret_cast<double*>(aux + L.partials_bytes);
    h->d_diag = reinterpret_cast<double*>(aux + L.partials_bytes + L.scratch_bytes);
    *out = h;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_destroy(hadpsgd_handle h) {
    if (!h) return HADPSGD_INVALID_ARG;
    DeviceGuard guard(h->device);
    cudaStreamSynchronize(h->stream);
    for (cudaEvent_t ev : h->chunk_events) cudaEventDestroy(ev);
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    if (h->d_peer) cudaFree(h->d_peer);
    for (void* p : h->ipc_mapped) if (p) cudaIpcCloseMemHandle(p);
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
    int rc = build_partner(h, step_k, partner, &h->partner);
    if (rc != HADPSGD_OK) return rc;
    rc = plan_and_prepare(h, h->partner.data(), &h->plan, &h->new_slot, &h->new_pending);
    if (rc != HADPSGD_OK) return rc;
    if (is_peer(h)) { rc = epoch_wait(h, true); if (rc != HADPSGD_OK) return rc; }   // neighbours only, on the stream
    rc = step_range(h, h->plan, lr, momentum, 0, h->L.P_padded, false);
    if (rc != HADPSGD_OK) return rc;
    if (is_peer(h)) { rc = epoch_signal(h, h->new_pending); if (rc != HADPSGD_OK) return rc; }
    commit_plan(h, h->plan, h->new_slot, h->new_pending, step_k);   // only now: every launch is enqueued
    return HADPSGD_OK;
}

extern "C" int hadpsgd_step_host(hadpsgd_handle h, const void* const* host_grads, float lr,
                                 float momentum, uint64_t step_k, hadpsgd_diag* diag_out) {
    if (!h || !host_grads) return HADPSGD_INVALID_ARG;
    if (is_peer(h)) { h->err = "hadpsgd_step_host is not available on a HADPSGD_PEER handle"; return HADPSGD_INVALID_ARG; }
    DeviceGuard guard(h->device);
    int rc = build_partner(h, step_k, nullptr, &h->partner);
    if (rc != HADPSGD_OK) return rc;
    const int n_buf = h->L.S * h->L.G;
    for (int b = 0; b < n_buf; ++b) if (!host_grads[b]) { h->err = "host_grads[] has a NULL entry"; return HADPSGD_INVALID_ARG; }

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

    std::vector<int32_t>& new_slot = h->new_slot;  // one slot plan for the whole step, shared by all chunks
    std::vector<int32_t>& new_pending = h->new_pending;
    rc = plan_and_prepare(h, h->partner.data(), &h->plan, &new_slot, &new_pending);
    if (rc != HADPSGD_OK) return rc;

    // On an error after this point copies from the caller's buffers may still be in flight and part of
    // the step has run: drain both streams before reporting it, so the caller may free its buffers.
    auto fail = [&](int code) {
        cudaStreamSynchronize(h->copy_stream);
        cudaStreamSynchronize(h->stream);
        return code;
    };
#define CUDA_TRY_DRAIN(call)                                                                \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess) {                                                            \
            h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                    \
            return fail(HADPSGD_CUDA);                                                      \
        }                                                                                   \
    } while (0)
    // the copy stream must not overwrite gradients an earlier step on h->stream still reads
    CUDA_TRY_DRAIN(cudaEventRecord(h->chunk_events[n_chunks], h->stream));
    CUDA_TRY_DRAIN(cudaStreamWaitEvent(h->copy_stream, h->chunk_events[n_chunks], 0));
    char* gdev = h->arena + h->L.g_off;
    struct HostStepScope { hadpsgd_ctx* h; ~HostStepScope() { h->in_host_step = false; } } scope{h};
    h->in_host_step = true;
    for (int c = 0; c < n_chunks; ++c) {
        const int64_t e0 = c * chunk, e1 = (e0 + chunk < P) ? e0 + chunk : P;
        for (int b = 0; b < n_buf; ++b)
            CUDA_TRY_DRAIN(cudaMemcpyAsync(gdev + static_cast<size_t>(b) * h->L.g_stride_bytes() + e0 * eb,
                                           static_cast<const char*>(host_grads[b]) + e0 * eb,
                                           static_cast<size_t>(e1 - e0) * eb, cudaMemcpyHostToDevice, h->copy_stream));
        CUDA_TRY_DRAIN(cudaEventRecord(h->chunk_events[c], h->copy_stream));
        CUDA_TRY_DRAIN(cudaStreamWaitEvent(h->stream, h->chunk_events[c], 0));
        rc = step_range(h, h->plan, lr, momentum, e0, e1, c > 0);
        if (rc != HADPSGD_OK) return fail(rc);
    }
#undef CUDA_TRY_DRAIN
    commit_plan(h, h->plan, new_slot, new_pending, step_k);
    if (diag_out) return hadpsgd_diagnostics(h, diag_out);
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return HADPSGD_OK;
}

extern "C" int hadpsgd_weights(hadpsgd_handle h, int s, float** dev_ptr) {
    if (!h || !dev_ptr || s < 0 || s >= h->L.S) return HADPSGD_INVALID_ARG;
    if (is_peer(h) && h->pending[s] >= 0) {
        h->err = "the mix of this super-learner with its partner in another arena is pending: call hadpsgd_peer_flush";
        return HADPSGD_INVALID_ARG;
    }
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
    std::vector<double>& tmp = h->diag_host;
    tmp.resize(kDiagArrays * S + 1);              // + the word a collector sets when it gave up waiting
    CUDA_TRY(h, cudaMemcpyAsync(tmp.data(), h->d_diag, sizeof(double) * (kDiagArrays * S + 1), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    uint32_t timed_out = 0;
    std::memcpy(&timed_out, &tmp[kDiagArrays * S], sizeof timed_out);
    if (timed_out) {
        CUDA_TRY(h, cudaMemsetAsync(h->d_diag + kDiagArrays * S, 0, sizeof(double), h->stream));   // report once
        h->err = "a step's diagnostics hand-over timed out (the blocks of its grid were not scheduled in order while the "
                 "device was shared): the diagnostics of that step are NaN; weights and momenta are not affected";
        return HADPSGD_DIAG_TIMEOUT;
    }
    host_out->S = S; host_out->n_pairs = h->last_n_pairs; host_out->step_k = h->diag_step_k;
    std::memcpy(host_out->gsq, tmp.data(), sizeof(double) * S);
    std::memcpy(host_out->wsq, tmp.data() + S, sizeof(double) * S);
    std::memcpy(host_out->gap, tmp.data() + 2 * S, sizeof(double) * S);
    std::memcpy(host_out->pend_wsq, tmp.data() + 3 * S, sizeof(double) * S);
    std::memcpy(host_out->pend_gap, tmp.data() + 4 * S, sizeof(double) * S);
    for (int s = 0; s < S; ++s) host_out->pending[s] = (is_peer(h) && h->pending[s] >= 0) ? 1 : 0;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_unshare(hadpsgd_handle h) {
    if (!h) return HADPSGD_INVALID_ARG;
    DeviceGuard guard(h->device);
    std::vector<SlotCopy> copies;
    std::vector<int32_t> slot = h->w_slot;
    plan_unshare(h->L.S, &slot, &copies);
    int rc = copy_slots(h, copies);
    if (rc == HADPSGD_OK) h->w_slot = slot;
    return rc;
}

extern "C" int hadpsgd_consensus(hadpsgd_handle h, double* D_out) {
    if (!h || !D_out) return HADPSGD_INVALID_ARG;
    if (is_peer(h)) { h->err = "hadpsgd_consensus needs all S_global weight columns in one arena: not on a HADPSGD_PEER handle"; return HADPSGD_INVALID_ARG; }
    DeviceGuard guard(h->device);
    // the scratch is free between steps: everything is ordered on h->stream
    cudaError_t e = cudaSuccess;
    const int grid = launch_consensus(reinterpret_cast<const float*>(h->arena + h->L.w_off), h->L.P_padded, h->L.S,
                                      h->w_slot.data(), h->num_sms, h->d_scratch, h->stream, &e);
    CUDA_TRY(h, e);
    h->launches++;
    std::vector<double> part(grid);
    CUDA_TRY(h, cudaMemcpyAsync(part.data(), h->d_scratch, sizeof(double) * grid, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    double D = 0.;
    for (int b = 0; b < grid; ++b) D += part[b];   // fixed order: run-to-run deterministic
    *D_out = D;
    return HADPSGD_OK;
}

// ---- super-learner partition (row f4) ----------------------------------------------------

extern "C" int hadpsgd_peer_init(hadpsgd_handle h, int rank, int world, const int32_t* rank_begin) {
    if (!h || !rank_begin || world < 1 || rank < 0 || rank >= world) return HADPSGD_INVALID_ARG;
    if (!is_peer(h)) { h->err = "handle was created without HADPSGD_PEER"; return HADPSGD_INVALID_ARG; }
    if (h->epoch != 0) { h->err = "hadpsgd_peer_init after the first step"; return HADPSGD_INVALID_ARG; }
    if (rank_begin[0] != 0) { h->err = "rank_begin[0] must be 0"; return HADPSGD_INVALID_ARG; }
    for (int r = 0; r < world; ++r)
        if (rank_begin[r + 1] <= rank_begin[r]) { h->err = "rank_begin must be increasing"; return HADPSGD_INVALID_ARG; }
    if (rank_begin[world] > HADPSGD_MAX_S) { h->err = "S_global exceeds HADPSGD_MAX_S"; return HADPSGD_INVALID_ARG; }
    if (rank_begin[rank + 1] - rank_begin[rank] != h->L.S) {
        h->err = "this handle holds S = " + std::to_string(h->L.S) + " super-learners but rank_begin gives it " +
                 std::to_string(rank_begin[rank + 1] - rank_begin[rank]);
        return HADPSGD_INVALID_ARG;
    }
    for (void* p : h->ipc_mapped) if (p) cudaIpcCloseMemHandle(p);   // a repeated init (before the first step) starts over
    h->ipc_mapped.assign(world, nullptr);
    h->war_until[0].assign(world, 0);
    h->war_until[1].assign(world, 0);
    // the epoch word (zeroed with the arena at create, on the stream) must be zero before any peer can learn
    // its address, which it does through calls that follow this one
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    h->rank = rank; h->world = world; h->S_global = rank_begin[world];
    h->rank_begin.assign(rank_begin, rank_begin + world + 1);
    h->stage_of_rank.assign(world, nullptr);
    h->stage_of_rank[rank] = reinterpret_cast<const float*>(h->arena + h->L.stage_off);
    h->peer_table_dirty = true;
    h->peer_init = true;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_peer_stage(hadpsgd_handle h, float** dev_ptr) {
    if (!h || !dev_ptr) return HADPSGD_INVALID_ARG;
    if (!is_peer(h)) { h->err = "handle was created without HADPSGD_PEER"; return HADPSGD_INVALID_ARG; }
    *dev_ptr = reinterpret_cast<float*>(h->arena + h->L.stage_off);
    return HADPSGD_OK;
}

extern "C" int hadpsgd_peer_attach(hadpsgd_handle h, int r, const float* stage_region) {
    if (!h || !stage_region) return HADPSGD_INVALID_ARG;
    if (!is_peer(h) || !h->peer_init) { h->err = "call hadpsgd_peer_init first"; return HADPSGD_INVALID_ARG; }
    if (r < 0 || r >= h->world || r == h->rank) { h->err = "rank out of range (or the handle's own rank)"; return HADPSGD_INVALID_ARG; }
    h->stage_of_rank[r] = stage_region;
    h->peer_table_dirty = true;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_peer_ipc_export(hadpsgd_handle h, void* ipc_handle_out, uint64_t* stage_offset_out) {
    if (!h || !ipc_handle_out || !stage_offset_out) return HADPSGD_INVALID_ARG;
    if (!is_peer(h)) { h->err = "handle was created without HADPSGD_PEER"; return HADPSGD_INVALID_ARG; }
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "the ABI promises a 64-byte IPC handle");
    DeviceGuard guard(h->device);
    // The IPC handle names the whole ALLOCATION the arena lives in (a caller-supplied arena may be a
    // slice of a larger one): find its base so that the importer can add the right offset.
    void* base = nullptr;
    {
        using get_range_t = int (*)(unsigned long long*, size_t*, unsigned long long);
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        CUDA_TRY(h, cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qr));
        if (!fn || qr != cudaDriverEntryPointSuccess) { h->err = "cuMemGetAddressRange is unavailable"; return HADPSGD_CUDA; }
        unsigned long long b = 0; size_t sz = 0;
        if (reinterpret_cast<get_range_t>(fn)(&b, &sz, reinterpret_cast<unsigned long long>(h->arena)) != 0) {
            h->err = "cuMemGetAddressRange failed on the arena"; return HADPSGD_CUDA;
        }
        base = reinterpret_cast<void*>(b);
    }
    cudaIpcMemHandle_t ipc;
    CUDA_TRY(h, cudaIpcGetMemHandle(&ipc, base));
    std::memcpy(ipc_handle_out, &ipc, sizeof ipc);
    *stage_offset_out = static_cast<uint64_t>(h->arena - static_cast<char*>(base)) + h->L.stage_off;
    return HADPSGD_OK;
}

extern "C" int hadpsgd_peer_ipc_attach(hadpsgd_handle h, int r, const void* ipc_handle, uint64_t stage_offset) {
    if (!h || !ipc_handle) return HADPSGD_INVALID_ARG;
    if (!is_peer(h) || !h->peer_init) { h->err = "call hadpsgd_peer_init first"; return HADPSGD_INVALID_ARG; }
    if (r < 0 || r >= h->world || r == h->rank) { h->err = "rank out of range (or the handle's own rank)"; return HADPSGD_INVALID_ARG; }
    DeviceGuard guard(h->device);
    if (h->ipc_mapped[r]) {
        // re-attach: one mapping per rank.  No launch may still read through the old one.
        CUDA_TRY(h, cudaStreamSynchronize(h->stream));
        void* old_base = h->ipc_mapped[r];
        h->ipc_mapped[r] = nullptr;
        h->stage_of_rank[r] = nullptr;
        h->peer_table_dirty = true;
        CUDA_TRY(h, cudaIpcCloseMemHandle(old_base));
    }
    cudaIpcMemHandle_t ipc;
    std::memcpy(&ipc, ipc_handle, sizeof ipc);
    void* base = nullptr;
    CUDA_TRY(h, cudaIpcOpenMemHandle(&base, ipc, cudaIpcMemLazyEnablePeerAccess));
    h->ipc_mapped[r] = base;
    return hadpsgd_peer_attach(h, r, reinterpret_cast<const float*>(static_cast<char*>(base) + stage_offset));
}

extern "C" int hadpsgd_peer_flush(hadpsgd_handle h) {
    if (!h) return HADPSGD_INVALID_ARG;
    if (!is_peer(h) || !h->peer_init) { h->err = "call hadpsgd_peer_init first"; return HADPSGD_INVALID_ARG; }
    DeviceGuard guard(h->device);
    std::vector<int32_t> members;   // (local member, peer-table entry of the partner's stage buffer)
    const int rd = static_cast<int>((h->epoch + 1) & 1);
    for (int s = 0; s < h->L.S; ++s)
        if (h->pending[s] >= 0) { members.push_back(s); members.push_back(rd * h->S_global + h->pending[s]); }
    if (members.empty()) return HADPSGD_OK;
    int rc = upload_peer_table(h);
    if (rc != HADPSGD_OK) return rc;
    rc = epoch_wait(h, false);          // the partners' publishing step must have completed
    if (rc != HADPSGD_OK) return rc;
    cudaError_t e = cudaSuccess;
    const float* a_stage = reinterpret_cast<const float*>(h->arena + h->L.stage_off) + static_cast<size_t>(rd) * h->L.S * h->L.P_padded;
    launch_peer_flush(reinterpret_cast<float*>(h->arena + h->L.w_off), a_stage, h->d_peer, members.data(),
                      static_cast<int>(members.size() / 2), h->L.P_padded, h->L.S, h->num_sms,
                      ((h->flags & HADPSGD_NO_DIAG) || !h->diag_on) ? nullptr : h->d_scratch, h->d_diag, h->stream, &e);
    CUDA_TRY(h, e);
    h->launches++;
    h->pending.assign(h->L.S, -1);
    return HADPSGD_OK;
}

extern "C" int hadpsgd_set_diagnostics(hadpsgd_handle h, int enable) {
    if (!h) return HADPSGD_INVALID_ARG;
    if (enable && (h->flags & HADPSGD_NO_DIAG)) { h->err = "handle was created with HADPSGD_NO_DIAG"; return HADPSGD_INVALID_ARG; }
    h->diag_on = enable != 0;
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
        case HADPSGD_DIAG_TIMEOUT: return "diagnostics hand-over timed out";
        default: return "unknown status";
    }
}
extern "C" const char* hadpsgd_last_error(hadpsgd_handle h) {
    return h ? h->err.c_str() : g_create_error.c_str();
}
