// peer_flush.cu -- hadpsgd_peer_flush (row f4): materialise the pending mixes of a peer-mode handle.
//
// A member whose partner lives in another arena ends a step with u_s in its own stage buffer and its
// mix pending; the next step resolves it on the fly.  This kernel does the same resolution WITHOUT a
// step, so that the weights can be read:  w_s = 0.5f * (u_s + u_p)  -- phase 2 of the oracle's step
// (eq. (7)) -- with u_p read through the peer pointer table (NVLink when the partner's
// arena is on another GPU).  Not on the timed path.  Also delivers the two diagnostics the pending
// step still owed (R14): pend_wsq[s] = sum w_s^2, pend_gap[s] = sum (u_s - u_p)^2, reduced
// in a fixed order (block partials, then one block) so they are run-to-run deterministic.
#include <cuda_runtime.h>

#include "internal.h"

namespace hadpsgd {

namespace {

constexpr int kThreads = 256;
constexpr int kMaxFlush = 32;   // members per launch

struct FlushArgs {
    float* w_main;             // main weight buffers [S][P]
    const float* a_stage;      // this handle's stage buffers of the parity being resolved [S][P]
    const float* const* peer;  // device pointer table
    long long P;
    int n;
    int S;
    double* partials;          // [grid][n][2] or null
    double* diag;              // device result arrays (pend_wsq at 3S, pend_gap at 4S) or null
    int member[kMaxFlush];
    int entry[kMaxFlush];
};

__global__ void __launch_bounds__(kThreads) flush_kernel(const __grid_constant__ FlushArgs a) {
    __shared__ double s_red[kThreads / 32][2];
    const long long n4 = a.P / 4;   // P_padded is a multiple of 64
    for (int j = 0; j < a.n; ++j) {
        const float4* us = reinterpret_cast<const float4*>(a.a_stage + static_cast<size_t>(a.member[j]) * a.P);
        const float4* up = reinterpret_cast<const float4*>(a.peer[a.entry[j]]);
        float4* out = reinterpret_cast<float4*>(a.w_main + static_cast<size_t>(a.member[j]) * a.P);
        double wsq = 0., gap = 0.;
        for (long long t = static_cast<long long>(blockIdx.x) * kThreads + threadIdx.x; t < n4;
             t += static_cast<long long>(gridDim.x) * kThreads) {
            const float4 x = us[t], y = up[t];
            float4 m;
            m.x = __fmul_rn(0.5f, __fadd_rn(x.x, y.x)); m.y = __fmul_rn(0.5f, __fadd_rn(x.y, y.y));
            m.z = __fmul_rn(0.5f, __fadd_rn(x.z, y.z)); m.w = __fmul_rn(0.5f, __fadd_rn(x.w, y.w));
            out[t] = m;
            const float d0 = x.x - y.x, d1 = x.y - y.y, d2 = x.z - y.z, d3 = x.w - y.w;
            gap += static_cast<double>(fmaf(d0, d0, fmaf(d1, d1, fmaf(d2, d2, d3 * d3))));
            wsq += static_cast<double>(fmaf(m.x, m.x, fmaf(m.y, m.y, fmaf(m.z, m.z, m.w * m.w))));
        }
        if (a.partials) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                wsq += __shfl_xor_sync(0xffffffffu, wsq, o);
                gap += __shfl_xor_sync(0xffffffffu, gap, o);
            }
            if ((threadIdx.x & 31) == 0) { s_red[threadIdx.x >> 5][0] = wsq; s_red[threadIdx.x >> 5][1] = gap; }
            __syncthreads();
            if (threadIdx.x < 2) {
                double tot = 0.;
                for (int i = 0; i < kThreads / 32; ++i) tot += s_red[i][threadIdx.x];   // fixed order
                a.partials[(static_cast<size_t>(blockIdx.x) * a.n + j) * 2 + threadIdx.x] = tot;
            }
            __syncthreads();
        }
    }
}

// one block: sums the block partials of every (member, quantity) in block order
__global__ void flush_reduce_kernel(const __grid_constant__ FlushArgs a, int grid) {
    for (int row = threadIdx.x; row < a.n * 2; row += blockDim.x) {
        double tot = 0.;
        for (int b = 0; b < grid; ++b) tot += a.partials[static_cast<size_t>(b) * a.n * 2 + row];
        const int j = row / 2, q = row - 2 * j;
        a.diag[(q == 0 ? 3 : 4) * a.S + a.member[j]] = tot;
    }
}

}  // namespace

// members: n pairs (local member, peer-table entry).  Enqueues on `stream`.
int launch_peer_flush(float* w_main, const float* a_stage, const float* const* peer, const int32_t* members,
                      int n_members, long long P_padded, int S, int num_sms, double* partials, double* diag,
                      cudaStream_t stream, cudaError_t* err) {
    *err = cudaSuccess;
    for (int first = 0; first < n_members && *err == cudaSuccess; first += kMaxFlush) {
        FlushArgs a;
        a.w_main = w_main; a.a_stage = a_stage; a.peer = peer; a.P = P_padded; a.S = S;
        a.n = n_members - first < kMaxFlush ? n_members - first : kMaxFlush;
        a.partials = partials; a.diag = diag;
        for (int j = 0; j < a.n; ++j) { a.member[j] = members[2 * (first + j)]; a.entry[j] = members[2 * (first + j) + 1]; }
        long long want = (P_padded / 4 + kThreads - 1) / kThreads;
        long long grid = static_cast<long long>(num_sms) * 4;
        if (grid > want) grid = want;
        if (grid > kMaxGridBlocks) grid = kMaxGridBlocks;
        if (grid < 1) grid = 1;
        flush_kernel<<<static_cast<unsigned>(grid), kThreads, 0, stream>>>(a);
        *err = cudaGetLastError();
        if (*err == cudaSuccess && partials) {
            flush_reduce_kernel<<<1, 64, 0, stream>>>(a, static_cast<int>(grid));
            *err = cudaGetLastError();
        }
    }
    return 0;
}

}  // namespace hadpsgd
