// step_kernel.cuh -- B0: the fused H-ADPSGD step kernel for sm_100a.
//
// One launch per step, one pass over HBM.  For each work item
// (a pair (s,p) of super-learners, or a single s when unmixed) and each 16-byte vector of
// parameters, a thread
//   * streams the G gradient vectors of s and of p (read once -> evict-first loads),
//     w_s, v_s, w_p, v_p                                   [2G+4 independent 16 B loads in flight]
//   * reduces the G gradients left to right in fp32 registers (eq. (6))
//   * v <- mu v + gbar ; u = w - lr v                       (eq. (3), + momentum)
//   * w_s = w_p = 1/2 (u_s + u_p)                           (eq. (7))
//   * writes v_s, v_p, w_s, w_p (streaming stores), and accumulates the a5 diagnostics.
// The path is HBM-bound (0.3 flop/B): no tensor cores, no shared-memory staging of data --
// each byte is touched exactly once, so the design goal is only "enough coalesced 16 B
// requests in flight per SM" and full-sector writes.
//
// Diagnostics: per-thread double accumulators -> warp shuffle tree -> block partial in a
// fixed slot of global scratch (no atomics on data) -> the last block to finish (ticket)
// reduces the partials in a fixed order.  Results are therefore run-to-run deterministic.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace hadpsgd {

constexpr int kMaxWork = 512;
constexpr int kNQ = 5;  // gsq_a, gsq_b, wsq_a, wsq_b, gap

enum Mode : int { kPair = 0, kSingle = 1, kPairEq7 = 2 };

struct StepArgs {
    float* w;             // S buffers of P floats
    float* v;             // S buffers of P floats
    const void* g;        // S*G buffers of P grad elements
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
    short2 work[kMaxWork];
};

// ---- memory access helpers -------------------------------------------------------------
// Gradients are touched once per step and never again before they are overwritten:
// ld.global.cs (evict-first).  w and v are read then rewritten in place; they are also
// loaded .cs because nothing re-reads them before the whole 55 GB working set has streamed
// through the 126 MB L2.
__device__ __forceinline__ float4 ld_stream(const float4* p) { return __ldcs(p); }
__device__ __forceinline__ uint4 ld_stream(const uint4* p) { return __ldcs(p); }
__device__ __forceinline__ void st_stream(float4* p, float4 x) { __stcs(p, x); }

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

// One super-learner's vector unit: UNIT consecutive parameters.
template <int UNIT> struct Vec { float x[UNIT]; };

// Load + reduce the G learner gradients of super-learner s for one unit (a2).
// fp32: UNIT = 4, one 16 B load per learner.  bf16: UNIT = 8, one 16 B load per learner,
// widened exactly (bf16 is the top half of an fp32).
template <int G, bool BF16, bool EXACT, int UNIT>
__device__ __forceinline__ void load_grads(const void* gbase, long long P, int Grt, int s,
                                           long long elem, Vec<UNIT> (&gr)[G > 0 ? G : 1]) {
    static_assert(G > 0, "templated G only");
#pragma unroll
    for (int k = 0; k < G; ++k) {
        long long off = (static_cast<long long>(s) * Grt + k) * P + elem;
        if constexpr (BF16) {
            uint4 raw = ld_stream(reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(gbase) + off));
            unsigned r[4] = {raw.x, raw.y, raw.z, raw.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                gr[k].x[2 * q] = __uint_as_float(r[q] << 16);
                gr[k].x[2 * q + 1] = __uint_as_float(r[q] & 0xFFFF0000u);
            }
        } else {
            float4 raw = ld_stream(reinterpret_cast<const float4*>(static_cast<const float*>(gbase) + off));
            gr[k].x[0] = raw.x; gr[k].x[1] = raw.y; gr[k].x[2] = raw.z; gr[k].x[3] = raw.w;
        }
    }
}

template <int UNIT>
__device__ __forceinline__ void load_state(const float* base, long long off, Vec<UNIT>& out) {
#pragma unroll
    for (int q = 0; q < UNIT / 4; ++q) {
        float4 t = ld_stream(reinterpret_cast<const float4*>(base + off) + q);
        out.x[4 * q] = t.x; out.x[4 * q + 1] = t.y; out.x[4 * q + 2] = t.z; out.x[4 * q + 3] = t.w;
    }
}
template <int UNIT>
__device__ __forceinline__ void store_state(float* base, long long off, const Vec<UNIT>& in) {
#pragma unroll
    for (int q = 0; q < UNIT / 4; ++q)
        st_stream(reinterpret_cast<float4*>(base + off) + q,
                  make_float4(in.x[4 * q], in.x[4 * q + 1], in.x[4 * q + 2], in.x[4 * q + 3]));
}

// gbar (a2) then v', u (a3) for one super-learner; gradients already in registers.
template <int G, bool EXACT, int UNIT>
__device__ __forceinline__ void reduce_update(const Vec<UNIT> (&gr)[G], float invG, float mu, float lr,
                                              const Vec<UNIT>& w, Vec<UNIT>& v, Vec<UNIT>& u, Vec<UNIT>& gbar) {
#pragma unroll
    for (int e = 0; e < UNIT; ++e) {
        float acc = gr[0].x[e];
#pragma unroll
        for (int k = 1; k < G; ++k) acc = add_<EXACT>(acc, gr[k].x[e]);  // fixed learner order g = 0..G-1
        float gb = mul_<EXACT>(acc, invG);
        float vn = vupd_<EXACT>(mu, v.x[e], gb);
        gbar.x[e] = gb;
        v.x[e] = vn;
        u.x[e] = wupd_<EXACT>(lr, vn, w.x[e]);
    }
}

// Runtime-G variant (any G >= 1): learners are streamed in batches of 4 loads.
template <bool BF16, bool EXACT, int UNIT>
__device__ __forceinline__ void reduce_runtime_G(const void* gbase, long long P, int G, int s, long long elem,
                                                 Vec<UNIT>& acc) {
    Vec<UNIT> one[1];
    load_grads<1, BF16, EXACT, UNIT>(gbase, P, G, s, elem, one);
    acc = one[0];
    int k = 1;
    for (; k + 4 <= G; k += 4) {
        Vec<UNIT> b[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            Vec<UNIT> t[1];
            load_grads<1, BF16, EXACT, UNIT>(static_cast<const char*>(gbase) +
                                                 static_cast<size_t>(k + j) * P * (BF16 ? 2 : 4),
                                             P, G, s, elem, t);
            b[j] = t[0];
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int e = 0; e < UNIT; ++e) acc.x[e] = add_<EXACT>(acc.x[e], b[j].x[e]);
    }
    for (; k < G; ++k) {
        Vec<UNIT> t[1];
        load_grads<1, BF16, EXACT, UNIT>(static_cast<const char*>(gbase) + static_cast<size_t>(k) * P * (BF16 ? 2 : 4),
                                         P, G, s, elem, t);
#pragma unroll
        for (int e = 0; e < UNIT; ++e) acc.x[e] = add_<EXACT>(acc.x[e], t[0].x[e]);
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
// The kernel.  G > 0: learner count known at compile time (all gradient loads of a unit are
// issued before any is consumed).  G == 0: runtime learner count.
// Persistent grid: gridDim.x = (#SMs x resident blocks/SM); block b walks tiles b, b+grid, ...
// of every work item in turn ("pair-major": at any moment the whole chip streams the same
// 2G+4 read streams and 4 write streams, which keeps DRAM pages open).
// ---------------------------------------------------------------------------------------
template <int G, bool BF16, bool EXACT, bool DIAG, int MODE, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) step_kernel(const __grid_constant__ StepArgs a) {
    constexpr int UNIT = BF16 ? 8 : 4;
    constexpr int GA = G > 0 ? G : 1;
    constexpr bool PAIRED = (MODE != kSingle);
    __shared__ double s_red[THREADS / 32][kNQ];
    __shared__ unsigned int s_last;

    const int tid = threadIdx.x;
    const long long n_units = a.unit_end - a.unit_begin;
    const float lr = a.lr, mu = a.mu, invG = a.invG;
    const long long P = a.P;
    const char* gbytes = static_cast<const char*>(a.g);

    for (int j = 0; j < a.n_work; ++j) {
        const int s = a.work[j].x, p = a.work[j].y;
        double d_gs = 0., d_gp = 0., d_ws = 0., d_wp = 0., d_gap = 0.;

        for (long long t = static_cast<long long>(blockIdx.x) * THREADS + tid; t < n_units;
             t += static_cast<long long>(gridDim.x) * THREADS) {
            const long long elem = (a.unit_begin + t) * UNIT;
            const long long os = static_cast<long long>(s) * P + elem;
            const long long op = static_cast<long long>(p) * P + elem;

            Vec<UNIT> ws, vs, us, gbs, wp, vp, up, gbp;
            if constexpr (G > 0) {
                // issue every load of the unit first: 2G+4 (fp32) or 2G+8 (bf16) x 16 B in flight
                Vec<UNIT> grs[GA], grp[GA];
                load_grads<GA, BF16, EXACT, UNIT>(a.g, P, G, s, elem, grs);
                if constexpr (PAIRED) load_grads<GA, BF16, EXACT, UNIT>(a.g, P, G, p, elem, grp);
                load_state<UNIT>(a.w, os, ws);
                load_state<UNIT>(a.v, os, vs);
                if constexpr (PAIRED) { load_state<UNIT>(a.w, op, wp); load_state<UNIT>(a.v, op, vp); }
                reduce_update<GA, EXACT, UNIT>(grs, invG, mu, lr, ws, vs, us, gbs);
                if constexpr (PAIRED) reduce_update<GA, EXACT, UNIT>(grp, invG, mu, lr, wp, vp, up, gbp);
            } else {
                load_state<UNIT>(a.w, os, ws);
                load_state<UNIT>(a.v, os, vs);
                if constexpr (PAIRED) { load_state<UNIT>(a.w, op, wp); load_state<UNIT>(a.v, op, vp); }
                Vec<UNIT> acc[1];
                reduce_runtime_G<BF16, EXACT, UNIT>(gbytes, P, a.G, s, elem, acc[0]);
                reduce_update<1, EXACT, UNIT>(acc, invG, mu, lr, ws, vs, us, gbs);
                if constexpr (PAIRED) {
                    reduce_runtime_G<BF16, EXACT, UNIT>(gbytes, P, a.G, p, elem, acc[0]);
                    reduce_update<1, EXACT, UNIT>(acc, invG, mu, lr, wp, vp, up, gbp);
                }
            }

            // a4: pairwise average.  Default (R3): both members get 1/2 (u_s + u_p).
            // kPairEq7: eq. (7) as printed, w'_s = 1/2 (w_s + w_p) - lr v'_s.
            Vec<UNIT> outs, outp, dif;
            if constexpr (MODE == kPair) {
#pragma unroll
                for (int e = 0; e < UNIT; ++e) {
                    float m = mul_<EXACT>(0.5f, add_<EXACT>(us.x[e], up.x[e]));
                    outs.x[e] = m; outp.x[e] = m;
                    if constexpr (DIAG) dif.x[e] = us.x[e] - up.x[e];
                }
            } else if constexpr (MODE == kPairEq7) {
#pragma unroll
                for (int e = 0; e < UNIT; ++e) {
                    float m = mul_<EXACT>(0.5f, add_<EXACT>(ws.x[e], wp.x[e]));
                    // u = w - lr v' was formed above; recover lr v' the same way the oracle does
                    float ts = mul_<EXACT>(lr, vs.x[e]), tp = mul_<EXACT>(lr, vp.x[e]);
                    outs.x[e] = EXACT ? __fsub_rn(m, ts) : m - ts;
                    outp.x[e] = EXACT ? __fsub_rn(m, tp) : m - tp;
                    if constexpr (DIAG) dif.x[e] = ws.x[e] - wp.x[e];
                }
            } else {
                outs = us;
            }

            store_state<UNIT>(a.v, os, vs);
            store_state<UNIT>(a.w, os, outs);
            if constexpr (PAIRED) { store_state<UNIT>(a.v, op, vp); store_state<UNIT>(a.w, op, outp); }

            if constexpr (DIAG) {
                d_gs += static_cast<double>(sumsq<UNIT>(gbs));
                d_ws += static_cast<double>(sumsq<UNIT>(outs));
                if constexpr (PAIRED) {
                    d_gp += static_cast<double>(sumsq<UNIT>(gbp));
                    d_gap += static_cast<double>(sumsq<UNIT>(dif));
                    if constexpr (MODE == kPairEq7) d_wp += static_cast<double>(sumsq<UNIT>(outp));
                }
            }
        }

        if constexpr (DIAG) {
            if constexpr (MODE == kPair) d_wp = d_ws;
            // block partial for work item j -> partials[j][q][blockIdx.x]
            double q[kNQ] = {d_gs, d_gp, d_ws, d_wp, d_gap};
#pragma unroll
            for (int k = 0; k < kNQ; ++k) q[k] = warp_sum(q[k]);
            if ((tid & 31) == 0)
#pragma unroll
                for (int k = 0; k < kNQ; ++k) s_red[tid >> 5][k] = q[k];
            __syncthreads();
            if (tid < kNQ) {
                double tot = 0.;
                for (int wi = 0; wi < THREADS / 32; ++wi) tot += s_red[wi][tid];  // fixed order
                a.partials[(static_cast<size_t>(j) * kNQ + tid) * gridDim.x + blockIdx.x] = tot;
            }
            __syncthreads();
        }
    }

    if constexpr (DIAG) {
        // last block to arrive reduces all block partials in a fixed order
        __threadfence();
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
                    const int s = a.work[j].x, p = a.work[j].y;
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
