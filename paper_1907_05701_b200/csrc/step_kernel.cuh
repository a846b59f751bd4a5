// step_kernel.cuh -- B0: the fused H-ADPSGD step kernel for sm_100a.
//
// One launch per step, one pass over HBM.  For each work item
// (a pair (s,p) of super-learners, or a single s when unmixed) and each unit of parameters
// (8 for fp32 gradients, 16 for bf16 gradients = one 32-byte gradient vector), a thread
//   * streams the G gradient vectors of s and of p, w_s, v_s, w_p, v_p
//                                        [2G+4 (fp32) / 2G+8 (bf16) independent 32 B loads in flight]
//   * reduces the G gradients left to right in fp32 registers (eq. (6))
//   * v <- mu v + gbar ; u = w - lr v                       (eq. (3), + momentum)
//   * w_s = w_p = 1/2 (u_s + u_p)                           (eq. (7))
//   * writes v_s, v_p, w_s, w_p (32 B stores), optionally a bf16 copy of w' (EMIT), and
//     accumulates the a5 diagnostics.
// The path is HBM-bound (0.3 flop/B): no tensor cores, no shared-memory staging of data --
// each byte is touched exactly once, so the design goal is only "the right amount of coalesced
// 32 B requests in flight per SM" (~100 KB) and full-sector writes.
//
// Weight addressing (WMODE): every work item names, per member, the weight buffer it READS (a),
// the buffer it WRITES (o) and -- in peer mode -- a second buffer b whose average with a IS the
// member's weight: w = 1/2 (a + b).  That is how a pair whose members live in two arenas (two
// GPUs; Fig. 3: one super-learner per node) is mixed without any kernel waiting
// on another: at step k each side writes its u into a stage buffer instead of averaging, and
// the launch of step k+1 forms 1/2 (u_own + u_partner) on the fly, reading the partner's stage
// buffer through a peer pointer (NVLink) -- 4 B per parameter, inside this same fused pass.
//
// Diagnostics: per tile, per-thread sums -> warp shuffle tree -> the warp's own accumulator of
// that work item in shared memory (no atomics, no block barrier per tile) -> at the end one block
// partial per item in a fixed slot of global scratch, tagged with the launch's number -> the last
// block of the grid polls the tags and adds the partials in a fixed order (no fence, no atomics).  Results are therefore run-to-run deterministic.  A launch of a
// single block skips the scratch round trip and reduces straight from shared memory.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace hadpsgd {

constexpr int kInlineItems = 32;   // work items per launch (16 B each, inside the kernel parameter)
constexpr int kNQ = 5;             // gsq_a, gsq_b, wsq_a, wsq_b, gap
constexpr int kNQPeer = 9;         // ... + pend_wsq_a, pend_wsq_b, pend_gap_a, pend_gap_b (peer mode)

enum Mode : int { kPair = 0, kSingle = 1, kPairEq7 = 2 };
// kOwn: member s reads and writes weight buffer s.  kSlots: read buffer a, write buffer o (pair
// members may share one buffer: HADPSGD_SHARE_PAIR_WEIGHTS).  kPeer: a, o and the pending-mix
// partner buffer b (super-learner partition over several arenas / GPUs).
// kChain: kSlots with the CHAIN walk (below); the dispatcher picks it for the kernels it measured faster on.
enum WMode : int { kOwn = 0, kSlots = 1, kPeer = 2, kChain = 3 };

// Work item: super-learner indices s, p of the pair inside THIS handle (momentum and gradients
// are always the member's own buffers); a_*: weight buffer index read; o_*: weight buffer index
// written; b_*: 0, or 1 + index into StepArgs::peer of the buffer to average with a_* first.
// Weight buffer index x addresses arena weights + x * P (main buffers 0..S-1, then -- peer mode
// -- the 2S stage buffers).
struct Item { unsigned short s, p, a_s, a_p, o_s, o_p, b_s, b_p; };

// A block partial on its way to the collecting block: lo = (tag << 32) | low half of the double,
// hi = (tag << 32) | high half.  Each word is one 64-bit access, so a reader that finds the tag of
// THIS launch in both words holds the value -- the flag travels with the data and no fence is needed.
// A tag is never 0, the scratch is zero at create, and the reader zeroes every slot it has consumed,
// so between launches the scratch is all zero: a launch replayed with the same tag (a CUDA graph) is
// safe, and the host still changes the tag with every launch it enqueues.
struct __align__(16) TaggedDouble { unsigned long long lo, hi; };

struct StepArgs {
    float* w;             // weight buffers (main, then stage) of P floats each
    float* v;             // S buffers of P floats
    const void* g;        // S*G buffers of P grad elements
    void* wb;             // EMIT only: S buffers of P bf16, the working copy of the new weights
    const float* const* peer;  // kPeer: device table of stage-buffer pointers (own and remote)
    long long P;          // padded elements per buffer
    long long unit_begin; // first vector unit of this launch
    long long unit_end;   // one past the last vector unit
    TaggedDouble* partials;   // [gridDim.x][n_work * NQ]
    double* diag;         // gsq[S] | wsq[S] | gap[S] | pend_wsq[S] | pend_gap[S]
    unsigned int tag;     // never 0; the host changes it with every launch it enqueues
    int G;
    int n_work;
    int S;
    int accumulate_diag;  // 0: diag = result ; 1: diag += result (chunked host path)
    int touch_count;      // blocks that work on any one item (host: from n_tiles, grid, walk order)
    int reverse;          // 1: walk the (item, tile) space backwards
    unsigned int* timeout_flag;   // set to 1 by a collector that gave up waiting (hadpsgd_diagnostics reports it)
    long long keep_from;  // walk position ((item, tile) index; CHAIN: tile index) from which stores stay in L2
    float lr, mu, invG;
    Item items[kInlineItems];
};

// ---- memory access helpers -------------------------------------------------------------
// Every byte is touched once per step, so all traffic is issued as 32-byte vector accesses
// (ld/st.global.v8.b32, new on sm_100) carrying L2::evict_first: a warp covers 1 KB of each
// stream per request, which measured ~6 % faster than 16-byte accesses on this path
// because fewer, longer DRAM bursts are in flight per stream.  (Selecting
// the policy at run time -- evict_normal when one step's working set fits L2 -- measured no
// faster at any L2-resident size and 0.4 % slower at full size, so the hint is a literal.)
struct Raw8 { unsigned u[8]; };
__device__ __forceinline__ Raw8 ld_stream32(const void* p) {
    Raw8 r;
    asm volatile("ld.global.L1::no_allocate.L2::evict_first.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r.u[0]), "=r"(r.u[1]), "=r"(r.u[2]), "=r"(r.u[3]), "=r"(r.u[4]), "=r"(r.u[5]), "=r"(r.u[6]), "=r"(r.u[7])
                 : "l"(p));
    return r;
}
// keep == false: L2::evict_first -- the line is written back and dropped as soon as possible (a step
// of a large problem never sees it again before it would have been evicted anyway; measured 6 %
// faster than evict_normal at >= 2 GB per step).  keep == true (block-uniform): the line stays in L2
// like any other -- used for the last part of a step's walk, which the NEXT step, walking in the
// opposite direction, reads and overwrites first (10-15 % at 0.2-0.8 GB per step).
__device__ __forceinline__ void st_stream32(void* p, const Raw8& r, bool keep) {
    if (keep)
        asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                     :: "l"(p), "r"(r.u[0]), "r"(r.u[1]), "r"(r.u[2]), "r"(r.u[3]), "r"(r.u[4]), "r"(r.u[5]), "r"(r.u[6]), "r"(r.u[7])
                     : "memory");
    else
        asm volatile("st.global.L1::no_allocate.L2::evict_first.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                     :: "l"(p), "r"(r.u[0]), "r"(r.u[1]), "r"(r.u[2]), "r"(r.u[3]), "r"(r.u[4]), "r"(r.u[5]), "r"(r.u[6]), "r"(r.u[7])
                     : "memory");
}

template <bool EXACT> __device__ __forceinline__ float add_(float a, float b) { return EXACT ? __fadd_rn(a, b) : a + b; }
template <bool EXACT> __device__ __forceinline__ float mul_(float a, float b) { return EXACT ? __fmul_rn(a, b) : a * b; }
// v' = mu*v + gbar : EXACT = mul then add (two roundings, as the oracle), else one FMA
template <bool EXACT> __device__ __forceinline__ float vupd_(float mu, float v, float gbar) {
    return EXACT ? __fadd_rn(__fmul_rn(mu, v), gbar) : fmaf(mu, v, gbar);
}
// u = w - lr*v'
template <bool EXACT> __device__ __forceinline__ float wupd_(float lr, float vn, float w) {
    return EXACT ? __fsub_rn(w, __fmul_rn(lr, vn)) : fmaf(-lr, vn, w);
}

// One super-learner's vector unit: UNIT consecutive parameters (8 for fp32 gradients, 16 for
// bf16 gradients, so that a gradient unit is always ONE 32-byte load).
template <int UNIT> struct Vec { float x[UNIT]; };

// Widen one 32-byte gradient load to UNIT floats.  bf16 -> fp32 is exact: a bf16 is the top
// half of an fp32.
template <bool BF16, int UNIT>
__device__ __forceinline__ void widen(const Raw8& raw, Vec<UNIT>& out) {
    if constexpr (BF16) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            out.x[2 * q] = __uint_as_float(raw.u[q] << 16);
            out.x[2 * q + 1] = __uint_as_float(raw.u[q] & 0xFFFF0000u);
        }
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) out.x[q] = __uint_as_float(raw.u[q]);
    }
}

// Issue the G learner-gradient loads of super-learner s for one unit (a2); raw registers.
template <int G, bool BF16>
__device__ __forceinline__ void load_grads(const char* gbase, long long P, long long off0, Raw8 (&gr)[G]) {
    constexpr int EB = BF16 ? 2 : 4;   // off0 = element offset inside learner 0's buffer of this super-learner
#pragma unroll
    for (int k = 0; k < G; ++k) gr[k] = ld_stream32(gbase + (off0 + k * P) * EB);
}

template <int UNIT>
__device__ __forceinline__ void load_state(const float* base, long long off, Vec<UNIT>& out) {
#pragma unroll
    for (int q = 0; q < UNIT / 8; ++q) {
        Raw8 t = ld_stream32(base + off + 8 * q);
#pragma unroll
        for (int e = 0; e < 8; ++e) out.x[8 * q + e] = __uint_as_float(t.u[e]);
    }
}
template <int UNIT>
__device__ __forceinline__ void store_state(float* base, long long off, const Vec<UNIT>& in, bool keep) {
#pragma unroll
    for (int q = 0; q < UNIT / 8; ++q) {
        Raw8 t;
#pragma unroll
        for (int e = 0; e < 8; ++e) t.u[e] = __float_as_uint(in.x[8 * q + e]);
        st_stream32(base + off + 8 * q, t, keep);
    }
}

// EMIT: bf16 (round-to-nearest-even) copy of the new weights for mixed-precision learners
// (SURVEY.md 8(f) row f2).  16 floats -> one 32 B store.  8 floats are only 16 B, so two
// neighbouring lanes pair up: the even lane fetches its neighbour's four packed registers by
// shuffle and stores 32 B for both (units come in even numbers -- P_padded and every sub-range are
// multiples of 64 elements -- so an even lane's unit and the next are live or dead together).
// Must be called by all 32 lanes of the warp; `live` predicates the store only.
template <int UNIT>
__device__ __forceinline__ void store_bf16(void* base, long long off, const Vec<UNIT>& in, bool live, bool keep) {
    unsigned pk[UNIT / 2];
#pragma unroll
    for (int q = 0; q < UNIT / 2; ++q) {
        __nv_bfloat162 h = __floats2bfloat162_rn(in.x[2 * q], in.x[2 * q + 1]);   // .x = low half
        pk[q] = *reinterpret_cast<unsigned*>(&h);
    }
    __nv_bfloat16* dst = static_cast<__nv_bfloat16*>(base) + off;
    Raw8 r;
    if constexpr (UNIT == 16) {
#pragma unroll
        for (int q = 0; q < 8; ++q) r.u[q] = pk[q];
        if (live) st_stream32(dst, r, keep);
    } else {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            r.u[q] = pk[q];
            r.u[4 + q] = __shfl_down_sync(0xffffffffu, pk[q], 1);
        }
        if (live && (threadIdx.x & 1) == 0) st_stream32(dst, r, keep);
    }
}

// Sum of the G learner gradients of one unit, left to right (a2); gradients already in registers.
template <int G, bool BF16, bool EXACT, int UNIT>
__device__ __forceinline__ void sum_grads(const Raw8 (&gr)[G], Vec<UNIT>& acc) {
    widen<BF16, UNIT>(gr[0], acc);
#pragma unroll
    for (int k = 1; k < G; ++k) {   // fixed learner order g = 0..G-1
        Vec<UNIT> t;
        widen<BF16, UNIT>(gr[k], t);
#pragma unroll
        for (int e = 0; e < UNIT; ++e) acc.x[e] = add_<EXACT>(acc.x[e], t.x[e]);
    }
}

// Runtime-G sum (any G >= 1): learners are streamed in batches of 4 loads, left to right.
template <bool BF16, bool EXACT, int UNIT>
__device__ __forceinline__ void sum_grads_runtime(const char* gbase, long long P, int G, long long off0,
                                                  Vec<UNIT>& acc) {
    constexpr int EB = BF16 ? 2 : 4;
    const char* p0 = gbase + off0 * EB;
    const long long stride = P * EB;
    widen<BF16, UNIT>(ld_stream32(p0), acc);
    int k = 1;
    for (; k + 4 <= G; k += 4) {
        Raw8 b[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) b[j] = ld_stream32(p0 + (k + j) * stride);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            Vec<UNIT> t;
            widen<BF16, UNIT>(b[j], t);
#pragma unroll
            for (int e = 0; e < UNIT; ++e) acc.x[e] = add_<EXACT>(acc.x[e], t.x[e]);
        }
    }
    for (; k < G; ++k) {
        Vec<UNIT> t;
        widen<BF16, UNIT>(ld_stream32(p0 + k * stride), t);
#pragma unroll
        for (int e = 0; e < UNIT; ++e) acc.x[e] = add_<EXACT>(acc.x[e], t.x[e]);
    }
}

// gbar = acc/G (a2), then v' = mu v + gbar, u = w - lr v' (a3).  acc is overwritten by gbar.
template <bool EXACT, int UNIT>
__device__ __forceinline__ void apply_update(Vec<UNIT>& acc, float invG, float mu, float lr,
                                             const Vec<UNIT>& w, Vec<UNIT>& v, Vec<UNIT>& u) {
#pragma unroll
    for (int e = 0; e < UNIT; ++e) {
        float gb = mul_<EXACT>(acc.x[e], invG);
        float vn = vupd_<EXACT>(mu, v.x[e], gb);
        acc.x[e] = gb;
        v.x[e] = vn;
        u.x[e] = wupd_<EXACT>(lr, vn, w.x[e]);
    }
}

template <int UNIT> __device__ __forceinline__ float sumsq(const Vec<UNIT>& a) {
    float s = 0.f;
#pragma unroll
    for (int e = 0; e < UNIT; ++e) s = fmaf(a.x[e], a.x[e], s);
    return s;
}

// Peer mode: the member's weight is the pending mix 1/2 (a + b) of its own stage buffer (already
// in w) and its partner's (b, possibly in another GPU's memory); this IS phase 2 of the previous
// step, 0.5f * (u_s + u_p).  Adds the two diagnostics that step still owes: sum m^2, sum (a-b)^2.
template <bool EXACT, bool DIAG, int UNIT>
__device__ __forceinline__ void resolve_pending(Vec<UNIT>& w, const Vec<UNIT>& b, double& d_wsq, double& d_gap) {
    float sw = 0.f, sg = 0.f;
#pragma unroll
    for (int e = 0; e < UNIT; ++e) {
        const float a = w.x[e];
        const float m = mul_<EXACT>(0.5f, add_<EXACT>(a, b.x[e]));
        if constexpr (DIAG) {
            const float d = a - b.x[e];
            sg = fmaf(d, d, sg);
            sw = fmaf(m, m, sw);
        }
        w.x[e] = m;
    }
    if constexpr (DIAG) { d_wsq += static_cast<double>(sw); d_gap += static_cast<double>(sg); }
}

__device__ __forceinline__ void st_tagged(TaggedDouble* p, double x, unsigned tag) {
    const unsigned long long b = static_cast<unsigned long long>(__double_as_longlong(x));
    const unsigned long long t = static_cast<unsigned long long>(tag) << 32;
    asm volatile("st.volatile.global.v2.u64 [%0], {%1,%2};" :: "l"(p), "l"(t | (b & 0xffffffffull)), "l"(t | (b >> 32)) : "memory");
}
__device__ __forceinline__ TaggedDouble ld_tagged(const TaggedDouble* p) {
    TaggedDouble r;
    asm volatile("ld.volatile.global.v2.u64 {%0,%1}, [%2];" : "=l"(r.lo), "=l"(r.hi) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void clear_tagged(TaggedDouble* p) {
    asm volatile("st.volatile.global.v2.u64 [%0], {%1,%1};" :: "l"(p), "l"(0ull) : "memory");
}
// Value of a partial already loaded once (t); re-polls until both words carry `tag`.  The writer is a
// block of the same grid with a LOWER block id (see the collector below), i.e. one that was handed to
// an SM before this block was: it is running or finished, so the wait is short.  That rests on the
// hardware dispatching the blocks of a grid in block-id order, which every NVIDIA GPU so far does but
// CUDA does not promise; should it ever not hold while the SMs are shared with other work, a bounded
// spin turns the stall into NaN diagnostics PLUS a flag that hadpsgd_diagnostics reports as
// HADPSGD_DIAG_TIMEOUT, instead of a hung GPU or a silent NaN (w and v never depend on this).
__device__ __forceinline__ double wait_tagged(const TaggedDouble* p, TaggedDouble t, unsigned tag, unsigned int* timeout_flag) {
    unsigned spins = 0;
    while (static_cast<unsigned>(t.lo >> 32) != tag || static_cast<unsigned>(t.hi >> 32) != tag) {
        if (++spins > (1u << 26)) {   // about a minute
            *reinterpret_cast<volatile unsigned int*>(timeout_flag) = 1u;
            return __longlong_as_double(0x7ff8000000000000ll);
        }
        if (spins > 16) __nanosleep(spins > 4096 ? 512 : 32);
        t = ld_tagged(p);
    }
    return __longlong_as_double(static_cast<long long>((t.hi << 32) | (t.lo & 0xffffffffull)));
}

__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// ---------------------------------------------------------------------------------------
// The kernel.  G > 0: learner count known at compile time (all gradient loads of a tile are
// issued before any is consumed).  G == 0: runtime learner count.
// Persistent grid: gridDim.x = (#SMs x resident blocks/SM); block b walks global tiles b,
// b+grid, ... of the item-major (work item, tile) space ("pair-major": for large P the whole
// chip streams the same 2G+4 read streams and 4 write streams at any moment, so few 2 MB pages
// and DRAM rows are live at once -- giving each block one contiguous range instead measured
// 2-10 % slower at 2^20..2^26 parameters; for small P the items spread over the blocks instead
// of serialising).  A tile is
// THREADS x U units; thread t owns units t, t+THREADS, ... of the tile, so each warp request
// covers 1 KB contiguous of one stream.
// ---------------------------------------------------------------------------------------
template <int G, bool BF16, bool EXACT, bool DIAG, int MODE, bool EMIT, int WMODE, int U, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) step_kernel(const __grid_constant__ StepArgs a) {
    constexpr int UNIT = BF16 ? 16 : 8;
    constexpr int GA = G > 0 ? G : 1;
    constexpr bool PAIRED = (MODE != kSingle);
    constexpr bool PEER = (WMODE == kPeer);
    // weights addressed through the item's buffer indices: shared pairs, peer mode, and every
    // unmixed item (after an un-sharing copy the buffer of an unmixed member need not be its own)
    constexpr bool SLOTS = WMODE != kOwn || MODE == kSingle;
    static_assert(WMODE != kChain || MODE == kPair, "the CHAIN walk is for shared pair slots");
    constexpr bool ONE_STORE = (WMODE == kSlots || WMODE == kChain);   // pair members share ONE output buffer
    constexpr int NP = PAIRED ? U : 1;   // array extent of the partner's registers
    constexpr int WARPS = THREADS / 32;
    constexpr int NQ = PEER ? kNQPeer : kNQ;
    extern __shared__ double s_acc[];    // DIAG: [WARPS][n_work][NQ], each warp owns its rows

    const int tid = threadIdx.x;
    const long long n_units = a.unit_end - a.unit_begin;
    const float lr = a.lr, mu = a.mu, invG = a.invG;
    const long long P = a.P;
    const char* gbytes = static_cast<const char*>(a.g);
    constexpr long long TILE = static_cast<long long>(THREADS) * U;

    if constexpr (DIAG) {
        for (int idx = tid; idx < WARPS * a.n_work * NQ; idx += THREADS) s_acc[idx] = 0.;
        __syncthreads();
    }
    // Programmatic dependent launch: the host launches every step with "programmatic stream
    // serialization", so this grid may become resident while the launch before it on the stream is
    // still draining.  Nothing above touches global memory; everything below waits here until that
    // launch has completed and its writes are visible.  Then the NEXT launch is allowed in at once: its
    // blocks park at this same line (one more resident block per SM fits beside a working one), so
    // that back-to-back steps pay no launch latency between them.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    // Flattened (work item, tile) space; block b takes global tiles b, b+grid, ...
    //  item-major: tiles of item 0, then item 1, ...: for large P the whole chip streams one pair
    //              at a time (few 2 MB pages and DRAM rows live at once).
    //  tile-major (pairs share weight slots): all items of tile 0, then tile 1, ...: the slot two
    //              neighbouring pairs both read is fetched from HBM once and hits in L2 the second time.
    //  CHAIN (ditto): block b takes TILES b, b+grid, ... and walks every item of a tile itself -- see below.
    const long long n_tiles = (n_units + TILE - 1) / TILE;
    const long long total_tiles = n_tiles * a.n_work;
    // a5: per-thread sums of the item being worked on; when the block moves to another item they
    // go through a warp shuffle tree into the warp's own accumulator row of the old item (no
    // block barrier).  (Placing the hand-over after the next tile's loads, to hide its latency,
    // keeps all loads live across the shuffles and costs registers -- measured slower.)
    double d_gs = 0., d_gp = 0., d_ws = 0., d_wp = 0., d_gap = 0.;
    double d_pws = 0., d_pwp = 0., d_pgs = 0., d_pgp = 0.;   // PEER: owed by the resolved pending mixes
    int cur = -1;
    unsigned touched = 0;    // bit j: this block worked on item j (n_work <= 32)
    Item it = {0, 0, 0, 0, 0, 0, 0, 0};
    // element offsets of the current item's buffers, recomputed only when the item changes
    long long o_vs = 0, o_vp = 0, o_gs = 0, o_gp = 0;   // momentum / gradients: the member's own buffers
    long long o_ws = 0, o_wp = 0, o_wos = 0, o_wop = 0; // SLOTS: weight read buffers and write buffers
    const float* pb_s = nullptr;                        // PEER: pending-mix partner buffers (or null)
    const float* pb_p = nullptr;
    auto hand_over = [&](int item) {
        if constexpr (MODE == kPair) d_wp = d_ws;
        double q[NQ];
        q[0] = d_gs; q[1] = d_gp; q[2] = d_ws; q[3] = d_wp; q[4] = d_gap;
        if constexpr (PEER) { q[5] = d_pws; q[6] = d_pwp; q[7] = d_pgs; q[8] = d_pgp; }
#pragma unroll
        for (int k = 0; k < NQ; ++k) q[k] = warp_sum(q[k]);
        if ((tid & 31) == 0) {
            double* row = s_acc + (static_cast<size_t>(tid >> 5) * a.n_work + item) * NQ;
#pragma unroll
            for (int k = 0; k < NQ; ++k) row[k] += q[k];
        }
        d_gs = d_gp = d_ws = d_wp = d_gap = 0.;
        d_pws = d_pwp = d_pgs = d_pgp = 0.;
    };
    // CHAIN (shared slots): the block owns whole tiles and walks ALL items of a tile in order, so the
    // weight vector item j read for its second member -- which, in the ring schedule, is the very
    // slot item j+1 reads for its first member -- is handed on in registers, and the slot the last
    // item shares with the first is kept from the first: every shared slot is fetched ONCE.
    // (Measured on the 16 x 4 fp32 configs: 1.5 % faster and DRAM reads at the mode's own byte model; on
    // the 8 x 8 configs, where weights are a small share of the reads and the carry costs 16-32 more
    // registers, the plain tile-major walk -- all items of tile 0 across neighbouring blocks, then tile
    // 1, ..., the shared slot hitting in L2 -- stays 1-1.5 % faster, so both exist.)
    constexpr bool CHAIN = (WMODE == kChain);
    constexpr bool TILE_MAJOR = (WMODE == kSlots);
    Vec<UNIT> carry[CHAIN ? U : 1], first_w[CHAIN ? U : 1];
    int prev_ap = -1, first_as = -1;
    long long seq = 0;                                   // CHAIN: position in this block's (tile, item) walk
    for (long long gt = blockIdx.x; ; gt += gridDim.x, ++seq) {
        int j;
        long long tile;
        bool keep;        // this tile lies in the last part of the walk: its stores stay in L2 (st_stream32)
        // a.reverse: the same walk from its far end (the host alternates the direction from step to step,
        // so a step begins with what the step before it touched last and may still find it in L2)
        if constexpr (CHAIN) {
            const long long round = seq / a.n_work;
            j = static_cast<int>(seq - round * a.n_work);
            tile = blockIdx.x + round * gridDim.x;
            if (tile >= n_tiles) break;
            keep = tile >= a.keep_from;
            if (a.reverse) tile = n_tiles - 1 - tile;
        } else {
            if (gt >= total_tiles) break;
            keep = gt >= a.keep_from;
            const long long g2 = a.reverse ? total_tiles - 1 - gt : gt;
            if constexpr (TILE_MAJOR) { tile = g2 / a.n_work; j = static_cast<int>(g2 - tile * a.n_work); }
            else { j = static_cast<int>(g2 / n_tiles); tile = g2 - static_cast<long long>(j) * n_tiles; }
        }
        const long long base = tile * TILE;
        bool take_carry = false, take_first = false;     // CHAIN: w_s / w_p already sit in registers
        if (j != cur || CHAIN) {                         // block-uniform
            if constexpr (DIAG) { if (cur >= 0) hand_over(cur); }
            cur = j;
            touched |= 1u << j;
            it = a.items[j];
            o_vs = it.s * P; o_vp = it.p * P;
            o_gs = o_vs * a.G; o_gp = o_vp * a.G;               // learner 0 of each member
            if constexpr (SLOTS) { o_ws = it.a_s * P; o_wp = it.a_p * P; o_wos = it.o_s * P; o_wop = it.o_p * P; }
            if constexpr (PEER) {
                pb_s = it.b_s ? a.peer[it.b_s - 1] : nullptr;
                pb_p = (PAIRED && it.b_p) ? a.peer[it.b_p - 1] : nullptr;
            }
            if constexpr (CHAIN) {
                take_carry = j > 0 && it.a_s == prev_ap;
                take_first = j > 0 && j == a.n_work - 1 && it.a_p == first_as;
                if (j == 0) first_as = it.a_s;
                prev_ap = it.a_p;
            }
        }
        {
            Vec<UNIT> ws[U], vs[U], gbs[U], wp[NP], vp[NP], gbp[NP];
            Vec<UNIT> bs[PEER ? U : 1], bp[PEER ? NP : 1];
            bool live[U];
            long long elem[U];
#pragma unroll
            for (int q = 0; q < U; ++q) {
                const long long t = base + q * THREADS + tid;
                live[q] = t < n_units;
                elem[q] = (a.unit_begin + t) * UNIT;
            }

            if constexpr (G > 0) {
                // issue every load of the tile first: U x (2G + 4 x UNIT/8) x 32 B in flight per thread
                Raw8 grs[U][GA], grp[NP][GA];
#pragma unroll
                for (int q = 0; q < U; ++q) {
                    if (live[q]) {
                        load_grads<GA, BF16>(gbytes, P, o_gs + elem[q], grs[q]);
                        if constexpr (PAIRED) load_grads<GA, BF16>(gbytes, P, o_gp + elem[q], grp[q]);
                        if (CHAIN && take_carry) ws[q] = carry[q];
                        else load_state<UNIT>(a.w, (SLOTS ? o_ws : o_vs) + elem[q], ws[q]);
                        load_state<UNIT>(a.v, o_vs + elem[q], vs[q]);
                        if constexpr (PAIRED) {
                            if (CHAIN && take_first) wp[q] = first_w[q];
                            else load_state<UNIT>(a.w, (SLOTS ? o_wp : o_vp) + elem[q], wp[q]);
                            load_state<UNIT>(a.v, o_vp + elem[q], vp[q]);
                        }
                        if constexpr (PEER) {
                            if (pb_s) load_state<UNIT>(pb_s, elem[q], bs[q]);
                            if constexpr (PAIRED) { if (pb_p) load_state<UNIT>(pb_p, elem[q], bp[q]); }
                        }
                    }
                }
#pragma unroll
                for (int q = 0; q < U; ++q) {
                    if (live[q]) {
                        sum_grads<GA, BF16, EXACT, UNIT>(grs[q], gbs[q]);
                        if constexpr (PAIRED) sum_grads<GA, BF16, EXACT, UNIT>(grp[q], gbp[q]);
                    }
                }
            } else {
#pragma unroll
                for (int q = 0; q < U; ++q) {
                    if (live[q]) {
                        if (CHAIN && take_carry) ws[q] = carry[q];
                        else load_state<UNIT>(a.w, (SLOTS ? o_ws : o_vs) + elem[q], ws[q]);
                        load_state<UNIT>(a.v, o_vs + elem[q], vs[q]);
                        if constexpr (PAIRED) {
                            if (CHAIN && take_first) wp[q] = first_w[q];
                            else load_state<UNIT>(a.w, (SLOTS ? o_wp : o_vp) + elem[q], wp[q]);
                            load_state<UNIT>(a.v, o_vp + elem[q], vp[q]);
                        }
                        if constexpr (PEER) {
                            if (pb_s) load_state<UNIT>(pb_s, elem[q], bs[q]);
                            if constexpr (PAIRED) { if (pb_p) load_state<UNIT>(pb_p, elem[q], bp[q]); }
                        }
                        sum_grads_runtime<BF16, EXACT, UNIT>(gbytes, P, a.G, o_gs + elem[q], gbs[q]);
                        if constexpr (PAIRED) sum_grads_runtime<BF16, EXACT, UNIT>(gbytes, P, a.G, o_gp + elem[q], gbp[q]);
                    }
                }
            }

            if constexpr (CHAIN) {       // the OLD weights, as read, travel on (dead lanes carry junk they never use)
#pragma unroll
                for (int q = 0; q < U; ++q) {
                    if (j == 0) first_w[q] = ws[q];
                    carry[q] = wp[q];
                }
            }
#pragma unroll
            for (int q = 0; q < U; ++q) {
                const long long os = o_vs + elem[q];
                const long long op = o_vp + elem[q];
                const long long wos = SLOTS ? o_wos + elem[q] : os;
                const long long wop = SLOTS ? o_wop + elem[q] : op;
                Vec<UNIT> us, up, outs, outp, dif;
                if (live[q]) {
                    if constexpr (PEER) {   // finish the previous step's mix across arenas first
                        if (pb_s) resolve_pending<EXACT, DIAG, UNIT>(ws[q], bs[q], d_pws, d_pgs);
                        if constexpr (PAIRED) { if (pb_p) resolve_pending<EXACT, DIAG, UNIT>(wp[q], bp[q], d_pwp, d_pgp); }
                    }
                    apply_update<EXACT, UNIT>(gbs[q], invG, mu, lr, ws[q], vs[q], us);
                    if constexpr (PAIRED) apply_update<EXACT, UNIT>(gbp[q], invG, mu, lr, wp[q], vp[q], up);

                    // a4: pairwise average.  Default (R3): both members get 1/2 (u_s + u_p).
                    // kPairEq7: eq. (7) as printed, w'_s = 1/2 (w_s + w_p) - lr v'_s.
                    if constexpr (MODE == kPair) {
#pragma unroll
                        for (int e = 0; e < UNIT; ++e) {
                            float m = mul_<EXACT>(0.5f, add_<EXACT>(us.x[e], up.x[e]));
                            outs.x[e] = m;
                            if constexpr (DIAG) dif.x[e] = us.x[e] - up.x[e];
                        }
                    } else if constexpr (MODE == kPairEq7) {
#pragma unroll
                        for (int e = 0; e < UNIT; ++e) {
                            float m = mul_<EXACT>(0.5f, add_<EXACT>(ws[q].x[e], wp[q].x[e]));
                            // recover lr v' the same way the oracle does (one fp32 multiply)
                            float ts = mul_<EXACT>(lr, vs[q].x[e]), tp = mul_<EXACT>(lr, vp[q].x[e]);
                            outs.x[e] = EXACT ? __fsub_rn(m, ts) : m - ts;
                            outp.x[e] = EXACT ? __fsub_rn(m, tp) : m - tp;
                            if constexpr (DIAG) dif.x[e] = ws[q].x[e] - wp[q].x[e];
                        }
                    } else {
                        outs = us;
                    }

                    store_state<UNIT>(a.v, os, vs[q], keep);
                    store_state<UNIT>(a.w, wos, outs, keep);
                    if constexpr (PAIRED) {
                        store_state<UNIT>(a.v, op, vp[q], keep);
                        if constexpr (!ONE_STORE)       // pair members keep separate copies
                            store_state<UNIT>(a.w, wop, MODE == kPair ? outs : outp, keep);
                    }

                    if constexpr (DIAG) {
                        d_gs += static_cast<double>(sumsq<UNIT>(gbs[q]));
                        d_ws += static_cast<double>(sumsq<UNIT>(outs));
                        if constexpr (PAIRED) {
                            d_gp += static_cast<double>(sumsq<UNIT>(gbp[q]));
                            d_gap += static_cast<double>(sumsq<UNIT>(dif));
                            if constexpr (MODE == kPairEq7) d_wp += static_cast<double>(sumsq<UNIT>(outp));
                        }
                    }
                }
                if constexpr (EMIT) {     // outside `live`: the lanes of a warp shuffle together
                    store_bf16<UNIT>(a.wb, wos, outs, live[q], keep);
                    if constexpr (PAIRED && !ONE_STORE)
                        store_bf16<UNIT>(a.wb, wop, MODE == kPair ? outs : outp, live[q], keep);
                }
            }
        }

    }

    if constexpr (DIAG) {
        if (cur >= 0) hand_over(cur);
        __syncthreads();
        const int R = a.n_work * NQ;     // rows: (item, quantity)
        // row -> its place in the result.  k: 0 gsq_s, 1 gsq_p, 2 wsq_s, 3 wsq_p, 4 gap (reported for
        // both members), 5-8 (peer) the wsq / gap a resolved pending mix owes to the step before
        auto publish = [&](int row, double sum) {
            const int j = row / NQ, k = row - j * NQ;
            const Item w = a.items[j];
            const int s = w.s, p = w.p, S = a.S;
            double* gsq = a.diag; double* wsq = a.diag + S; double* gap = a.diag + 2 * S;
            auto put = [&](double* dst, double val) { *dst = a.accumulate_diag ? *dst + val : val; };
            if (k == 0) put(gsq + s, sum);
            if (k == 2) put(wsq + s, sum);
            if (PAIRED) {
                if (k == 1) put(gsq + p, sum);
                if (k == 3) put(wsq + p, sum);
                if (k == 4) { put(gap + s, sum); put(gap + p, sum); }
            } else if (k == 4) {
                put(gap + s, 0.0);
            }
            if constexpr (!PEER) {
                // a member that resolves no pending mix owes nothing from the step before: its pend_wsq /
                // pend_gap read 0 (every member is in exactly one item of a step, so a step rewrites all S)
                double* pws = a.diag + 3 * S; double* pgp = a.diag + 4 * S;
                if (k == 2) { put(pws + s, 0.0); put(pgp + s, 0.0); }
                if (PAIRED && k == 3) { put(pws + p, 0.0); put(pgp + p, 0.0); }
            }
            if constexpr (PEER) {
                double* pws = a.diag + 3 * S; double* pgp = a.diag + 4 * S;
                if (k == 5) put(pws + s, sum);
                if (k == 7) put(pgp + s, sum);
                if (PAIRED) {
                    if (k == 6) put(pws + p, sum);
                    if (k == 8) put(pgp + p, sum);
                }
            }
        };
        if (gridDim.x == 1) {            // the only block: its warp rows ARE the result
            for (int row = tid; row < R; row += THREADS) {
                double tot = 0.;
                for (int wi = 0; wi < WARPS; ++wi) tot += s_acc[static_cast<size_t>(wi) * R + row];   // fixed order
                publish(row, tot);
            }
            return;
        }
        // Block partial of the rows of every item this block worked on -> partials[block][row], TAGGED:
        // the two halves of the double travel in two 64-bit words whose upper halves carry this launch's
        // tag, so a reader that sees both tags has the value -- no fence, no ticket, no atomics, and no
        // block waits for its data stores to drain.
        for (int row = tid; row < R; row += THREADS) {
            if (!((touched >> (row / NQ)) & 1u)) continue;
            double tot = 0.;
            for (int wi = 0; wi < WARPS; ++wi) tot += s_acc[static_cast<size_t>(wi) * R + row];       // fixed order
            st_tagged(a.partials + static_cast<size_t>(blockIdx.x) * R + row, tot, a.tag);
        }
        // Item j is COLLECTED by block grid-1 - (j mod grid): the blocks with the highest ids, which are
        // dispatched last and have the fewest tiles.  Every other block is done here.  Forward progress:
        // a collector only waits for blocks with LOWER ids than its own (or itself), and blocks are handed
        // to SMs in block-id order, so by the time a collector runs every block it waits for is running or
        // done.  When the device is otherwise idle the whole grid is resident at once (the host sizes it
        // to this kernel's occupancy) and the order does not even matter; when the SMs are shared (other
        // handles on other streams, another process, a foreign persistent kernel) in-order dispatch is
        // what is relied on -- see wait_tagged for what happens if it failed.  Item j was worked on by exactly touch_count blocks: the i-th of them (in tile
        // order) is block (j * n_tiles + i) mod grid in the item-major walk, (j + i * n_work) mod grid in the
        // tile-major walk, block i in the CHAIN walk.  One warp per quantity: lane l polls contributors l,
        // l+32, ... (eight independent loads at a time), adds them in that order, the lanes combine in a
        // fixed shuffle tree, and each consumed slot is zeroed again for the launches that follow.  The
        // result depends on the launch shape only: run-to-run deterministic.
        const unsigned nb = gridDim.x;
        const int lane = tid & 31, warp = tid >> 5;
        for (int j = static_cast<int>(nb - 1u - blockIdx.x); j < a.n_work; j += static_cast<int>(nb)) {
            const int jw = a.reverse ? a.n_work - 1 - j : j;   // position of item j in the walk
            const unsigned long long first = CHAIN ? 0ull : TILE_MAJOR ? static_cast<unsigned long long>(jw)
                                                   : static_cast<unsigned long long>(jw) * static_cast<unsigned long long>(n_tiles);
            const unsigned long long step1 = TILE_MAJOR ? static_cast<unsigned long long>(a.n_work) : 1ull;
            for (int k = warp; k < NQ; k += WARPS) {
                const int row = j * NQ + k;
                double sum = 0.;
                for (int i0 = lane; i0 < a.touch_count; i0 += 32 * 8) {
                    TaggedDouble* src[8];
                    TaggedDouble t[8];
#pragma unroll
                    for (int m = 0; m < 8; ++m) {
                        const int i = i0 + 32 * m;
                        if (i < a.touch_count) {
                            const unsigned b = static_cast<unsigned>((first + step1 * static_cast<unsigned long long>(i)) % nb);
                            src[m] = a.partials + static_cast<size_t>(b) * R + row;
                            t[m] = ld_tagged(src[m]);
                        }
                    }
#pragma unroll
                    for (int m = 0; m < 8; ++m) {
                        if (i0 + 32 * m < a.touch_count) {
                            sum += wait_tagged(src[m], t[m], a.tag, a.timeout_flag);
                            clear_tagged(src[m]);
                        }
                    }
                }
                sum = warp_sum(sum);
                if (lane == 0) publish(row, sum);
            }
        }
    }
}

}  // namespace hadpsgd
