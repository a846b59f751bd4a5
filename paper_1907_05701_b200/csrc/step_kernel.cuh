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
// Diagnostics: per tile, per-thread sums -> warp shuffle tree -> the warp's own accumulator of
// that work item in shared memory (no atomics, no block barrier per tile) -> at the end one block
// partial per item in a fixed slot of global scratch -> the last block to finish (ticket) reduces
// the partials in a fixed order.  Results are therefore run-to-run deterministic.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace hadpsgd {

constexpr int kMaxWork = 480;   // work items per launch: 480 x 8 B keeps StepArgs under 4 KB
constexpr int kNQ = 5;  // gsq_a, gsq_b, wsq_a, wsq_b, gap

enum Mode : int { kPair = 0, kSingle = 1, kPairEq7 = 2 };

struct StepArgs {
    float* w;             // S buffers of P floats
    float* v;             // S buffers of P floats
    const void* g;        // S*G buffers of P grad elements
    void* wb;             // EMIT only: S buffers of P bf16, the working copy of the new weights
    long long P;          // padded elements per buffer
    long long unit_begin; // first vector unit of this launch
    long long unit_end;   // one past the last vector unit
    int G;
    int n_work;
    float lr, mu, invG;
    int accumulate_diag;  // 0: diag = result ; 1: diag += result (chunked host path)
    int S;
    double* partials;     // [n_work][kNQ][gridDim.x]
    double* diag;         // gsq[S] | wsq[S] | gap[S]
    unsigned int* ticket;
    unsigned long long work[kMaxWork];   // six 10-bit fields per item, see pack_item()
};

// Work item = (s, p, ws, wp, wo_s, wo_p): super-learner indices of the pair (gradients and
// momentum are always indexed by s / p), the weight slots w_s / w_p are READ from, and the slots
// the new weights are WRITTEN to (wo_s == wo_p when the pair shares one copy).  S <= 512.
__host__ __device__ inline unsigned long long pack_item(int s, int p, int ws, int wp, int wo_s, int wo_p) {
    return static_cast<unsigned long long>(s) | static_cast<unsigned long long>(p) << 10 |
           static_cast<unsigned long long>(ws) << 20 | static_cast<unsigned long long>(wp) << 30 |
           static_cast<unsigned long long>(wo_s) << 40 | static_cast<unsigned long long>(wo_p) << 50;
}
struct Item { int s, p, ws, wp, wo_s, wo_p; };
__device__ __forceinline__ Item unpack_item(unsigned long long w) {
    return {static_cast<int>(w & 1023u), static_cast<int>((w >> 10) & 1023u), static_cast<int>((w >> 20) & 1023u),
            static_cast<int>((w >> 30) & 1023u), static_cast<int>((w >> 40) & 1023u), static_cast<int>((w >> 50) & 1023u)};
}

// ---- memory access helpers -------------------------------------------------------------
// Every byte is touched once per step, so all traffic is issued as 32-byte vector accesses
// (ld/st.global.v8.b32, new on sm_100) carrying L2::evict_first: a warp covers 1 KB of each
// stream per request, which measured ~6 % faster than 16-byte accesses on this path
// because fewer, longer DRAM bursts are in flight per stream.
struct Raw8 { unsigned u[8]; };
__device__ __forceinline__ Raw8 ld_stream32(const void* p) {
    Raw8 r;
    asm volatile("ld.global.L1::no_allocate.L2::evict_first.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r.u[0]), "=r"(r.u[1]), "=r"(r.u[2]), "=r"(r.u[3]), "=r"(r.u[4]), "=r"(r.u[5]), "=r"(r.u[6]), "=r"(r.u[7])
                 : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream32(void* p, const Raw8& r) {
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
__device__ __forceinline__ void store_state(float* base, long long off, const Vec<UNIT>& in) {
#pragma unroll
    for (int q = 0; q < UNIT / 8; ++q) {
        Raw8 t;
#pragma unroll
        for (int e = 0; e < 8; ++e) t.u[e] = __float_as_uint(in.x[8 * q + e]);
        st_stream32(base + off + 8 * q, t);
    }
}

// EMIT: bf16 (round-to-nearest-even) copy of the new weights for mixed-precision learners
// (SURVEY.md 8(f) row f2).  8 floats -> one 16 B store, 16 floats -> one 32 B store.
template <int UNIT>
__device__ __forceinline__ void store_bf16(void* base, long long off, const Vec<UNIT>& in) {
    unsigned pk[UNIT / 2];
#pragma unroll
    for (int q = 0; q < UNIT / 2; ++q) {
        __nv_bfloat162 h = __floats2bfloat162_rn(in.x[2 * q], in.x[2 * q + 1]);   // .x = low half
        pk[q] = *reinterpret_cast<unsigned*>(&h);
    }
    __nv_bfloat16* dst = static_cast<__nv_bfloat16*>(base) + off;
    if constexpr (UNIT == 16) {
        Raw8 r;
#pragma unroll
        for (int q = 0; q < 8; ++q) r.u[q] = pk[q];
        st_stream32(dst, r);
    } else {
        // 16 B streaming store (an L2 evict-first cache-hint policy measured the same)
        __stcs(reinterpret_cast<uint4*>(dst), make_uint4(pk[0], pk[1], pk[2], pk[3]));
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
// SHARED (kPair only): pair members share weight slots (HADPSGD_SHARE_PAIR_WEIGHTS): weights are
// read from the item's read slots, the mixed weights are stored ONCE, and the walk is tile-major.
template <int G, bool BF16, bool EXACT, bool DIAG, int MODE, bool EMIT, bool SHARED, int U, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) step_kernel(const __grid_constant__ StepArgs a) {
    constexpr int UNIT = BF16 ? 16 : 8;
    constexpr int GA = G > 0 ? G : 1;
    constexpr bool PAIRED = (MODE != kSingle);
    // weights addressed through the item's slots: shared pairs, and every unmixed item (after an
    // un-sharing copy the slot of an unmixed member need not be its own index)
    constexpr bool SLOTS = SHARED || MODE == kSingle;
    constexpr int NP = PAIRED ? U : 1;   // array extent of the partner's registers
    constexpr int WARPS = THREADS / 32;
    extern __shared__ double s_acc[];    // DIAG: [WARPS][n_work][kNQ], each warp owns its rows
    __shared__ unsigned int s_last;

    const int tid = threadIdx.x;
    const long long n_units = a.unit_end - a.unit_begin;
    const float lr = a.lr, mu = a.mu, invG = a.invG;
    const long long P = a.P;
    const char* gbytes = static_cast<const char*>(a.g);
    constexpr long long TILE = static_cast<long long>(THREADS) * U;

    if constexpr (DIAG) {
        for (int idx = tid; idx < WARPS * a.n_work * kNQ; idx += THREADS) s_acc[idx] = 0.;
        __syncthreads();
    }

    // Flattened (work item, tile) space; block b takes global tiles b, b+grid, ...
    //  item-major: tiles of item 0, then item 1, ...: for large P the whole chip streams one pair
    //              at a time (few 2 MB pages and DRAM rows live at once).
    //  tile-major: all items of tile 0, then tile 1, ...: used when pairs share weight slots --
    //              the slot two neighbouring pairs both read is then fetched from HBM once and
    //              hits in L2 the second time.
    const long long n_tiles = (n_units + TILE - 1) / TILE;
    const long long total_tiles = n_tiles * a.n_work;
    // a5: per-thread sums of the item being worked on; when the block moves to another item they
    // go through a warp shuffle tree into the warp's own accumulator row of the old item (no
    // block barrier).  (Placing the hand-over after the next tile's loads, to hide its latency,
    // keeps all loads live across the shuffles and costs registers -- measured slower.)
    double d_gs = 0., d_gp = 0., d_ws = 0., d_wp = 0., d_gap = 0.;
    int cur = -1;
    Item it = {0, 0, 0, 0, 0, 0};
    // element offsets of the current item's buffers, recomputed only when the item changes
    long long o_vs = 0, o_vp = 0, o_gs = 0, o_gp = 0;   // momentum / gradients: the member's own buffers
    long long o_ws = 0, o_wp = 0, o_wo = 0;             // SHARED: weight read slots and the one write slot
    auto hand_over = [&](int item) {
        if constexpr (MODE == kPair) d_wp = d_ws;
        double q[kNQ] = {d_gs, d_gp, d_ws, d_wp, d_gap};
#pragma unroll
        for (int k = 0; k < kNQ; ++k) q[k] = warp_sum(q[k]);
        if ((tid & 31) == 0) {
            double* row = s_acc + (static_cast<size_t>(tid >> 5) * a.n_work + item) * kNQ;
#pragma unroll
            for (int k = 0; k < kNQ; ++k) row[k] += q[k];
        }
        d_gs = d_gp = d_ws = d_wp = d_gap = 0.;
    };
    for (long long gt = blockIdx.x; gt < total_tiles; gt += gridDim.x) {
        int j;
        long long tile;
        if constexpr (SHARED) { tile = gt / a.n_work; j = static_cast<int>(gt - tile * a.n_work); }
        else { j = static_cast<int>(gt / n_tiles); tile = gt - static_cast<long long>(j) * n_tiles; }
        const long long base = tile * TILE;
        if (j != cur) {                                  // block-uniform
            if constexpr (DIAG) { if (cur >= 0) hand_over(cur); }
            cur = j;
            it = unpack_item(a.work[j]);
            o_vs = it.s * P; o_vp = it.p * P;
            o_gs = o_vs * a.G; o_gp = o_vp * a.G;               // learner 0 of each member
            if constexpr (SLOTS) { o_ws = it.ws * P; o_wp = it.wp * P; o_wo = it.wo_s * P; }
        }
        {
            Vec<UNIT> ws[U], vs[U], gbs[U], wp[NP], vp[NP], gbp[NP];
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
                        load_state<UNIT>(a.w, (SLOTS ? o_ws : o_vs) + elem[q], ws[q]);
                        load_state<UNIT>(a.v, o_vs + elem[q], vs[q]);
                        if constexpr (PAIRED) {
                            load_state<UNIT>(a.w, (SLOTS ? o_wp : o_vp) + elem[q], wp[q]);
                            load_state<UNIT>(a.v, o_vp + elem[q], vp[q]);
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
                        load_state<UNIT>(a.w, (SLOTS ? o_ws : o_vs) + elem[q], ws[q]);
                        load_state<UNIT>(a.v, o_vs + elem[q], vs[q]);
                        if constexpr (PAIRED) {
                            load_state<UNIT>(a.w, (SLOTS ? o_wp : o_vp) + elem[q], wp[q]);
                            load_state<UNIT>(a.v, o_vp + elem[q], vp[q]);
                        }
                        sum_grads_runtime<BF16, EXACT, UNIT>(gbytes, P, a.G, o_gs + elem[q], gbs[q]);
                        if constexpr (PAIRED) sum_grads_runtime<BF16, EXACT, UNIT>(gbytes, P, a.G, o_gp + elem[q], gbp[q]);
                    }
                }
            }

#pragma unroll
            for (int q = 0; q < U; ++q) {
                if (!live[q]) continue;
                const long long os = o_vs + elem[q];
                const long long op = o_vp + elem[q];
                Vec<UNIT> us, up, outs, outp, dif;
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

                const long long wos = SLOTS ? o_wo + elem[q] : os;
                store_state<UNIT>(a.v, os, vs[q]);
                store_state<UNIT>(a.w, wos, outs);
                if constexpr (EMIT) store_bf16<UNIT>(a.wb, wos, outs);
                if constexpr (PAIRED) {
                    store_state<UNIT>(a.v, op, vp[q]);
                    if constexpr (!SHARED) {       // pair members keep separate copies
                        store_state<UNIT>(a.w, op, MODE == kPair ? outs : outp);
                        if constexpr (EMIT) store_bf16<UNIT>(a.wb, op, MODE == kPair ? outs : outp);
                    }
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
        }

    }

    if constexpr (DIAG) {
        if (cur >= 0) hand_over(cur);
        // block partial of every item (zero for items this block never touched) -> partials[j][q][block]
        __syncthreads();
        for (int idx = tid; idx < a.n_work * kNQ; idx += THREADS) {
            double tot = 0.;
            for (int wi = 0; wi < WARPS; ++wi) tot += s_acc[static_cast<size_t>(wi) * a.n_work * kNQ + idx];  // fixed order
            a.partials[static_cast<size_t>(idx) * gridDim.x + blockIdx.x] = tot;
        }
    }

    if constexpr (DIAG) {
        // last block to arrive reduces all block partials in a fixed order.  Order matters: every
        // thread's partial stores, then its fence, then a block barrier, and only then the ticket --
        // otherwise warp 0 could publish the ticket before another warp's partials are out.
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            unsigned int t = atomicAdd(a.ticket, 1u);
            s_last = (t == gridDim.x - 1) ? 1u : 0u;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            const int lane = tid & 31, wid = tid >> 5;
            for (int item = wid; item < a.n_work * kNQ; item += THREADS / 32) {
                const double* src = a.partials + static_cast<size_t>(item) * gridDim.x;
                double sum = 0.;
                for (unsigned b = lane; b < gridDim.x; b += 32) sum += __ldcg(src + b);
                sum = warp_sum(sum);
                if (lane == 0) {
                    const int j = item / kNQ, k = item % kNQ;
                    const Item it = unpack_item(a.work[j]);
                    const int s = it.s, p = it.p;
                    // k: 0 gsq_s, 1 gsq_p, 2 wsq_s, 3 wsq_p, 4 gap (reported for both members)
                    double* gsq = a.diag; double* wsq = a.diag + a.S; double* gap = a.diag + 2 * a.S;
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
                }
            }
            if (tid == 0) *a.ticket = 0u;  // re-arm for the next launch on this stream
        }
    }
}

}  // namespace hadpsgd
