// consensus.cu -- optional diagnostic, NOT part of the timed step: the consensus distance
//   D = sum_i sum_s (w_s[i] - wbar[i])^2 ,  wbar[i] = (1/S) sum_s w_s[i]
// i.e. how far the S super-learners are from the point (1/n) sum theta^i that repeated mixing
// drives them to.  It needs all S columns of an element at once, so it cannot ride
// in the pair-local step kernel (R14); one extra read of the S weight buffers.
#include <cuda_runtime.h>

#include "internal.h"

namespace hadpsgd {

namespace {

constexpr int kThreads = 256;

struct SlotTable { short slot[HADPSGD_MAX_S]; };   // slot[s] = weight buffer that holds w_s

__global__ void __launch_bounds__(kThreads) consensus_kernel(const float* __restrict__ w, long long P, int S,
                                                             const __grid_constant__ SlotTable tab,
                                                             double* __restrict__ block_out) {
    __shared__ double s_red[kThreads / 32];
    const long long n_units = P / 4;   // P_padded is a multiple of 64
    double acc = 0.;
    for (long long t = static_cast<long long>(blockIdx.x) * kThreads + threadIdx.x; t < n_units;
         t += static_cast<long long>(gridDim.x) * kThreads) {
        const float4* col = reinterpret_cast<const float4*>(w) + t;
        const long long stride = P / 4;
        double m0 = 0., m1 = 0., m2 = 0., m3 = 0.;
        for (int s = 0; s < S; ++s) {   // pass 1: the mean, in double, s = 0..S-1
            const float4 x = col[tab.slot[s] * stride];
            m0 += x.x; m1 += x.y; m2 += x.z; m3 += x.w;
        }
        const double inv = 1.0 / static_cast<double>(S);
        m0 *= inv; m1 *= inv; m2 *= inv; m3 *= inv;
        for (int s = 0; s < S; ++s) {   // pass 2: squared deviations (the re-read hits L1/L2)
            const float4 x = col[tab.slot[s] * stride];
            const double d0 = x.x - m0, d1 = x.y - m1, d2 = x.z - m2, d3 = x.w - m3;
            acc += d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.;
        for (int i = 0; i < kThreads / 32; ++i) tot += s_red[i];   // fixed order
        block_out[blockIdx.x] = tot;
    }
}

}  // namespace

// Enqueues the kernel on `stream`; block_out (device, >= grid doubles) receives one partial per
// block.  Returns the grid size used (the caller sums block_out[0..grid) in order on the host).
int launch_consensus(const float* w, long long P_padded, int S, const int32_t* w_slot, int num_sms,
                     double* block_out, cudaStream_t stream, cudaError_t* err) {
    SlotTable tab;
    for (int s = 0; s < S; ++s) tab.slot[s] = static_cast<short>(w_slot[s]);
    long long want = (P_padded / 4 + kThreads - 1) / kThreads;
    long long grid = static_cast<long long>(num_sms) * 8;
    if (grid > want) grid = want;
    if (grid > kMaxGridBlocks) grid = kMaxGridBlocks;
    if (grid < 1) grid = 1;
    consensus_kernel<<<static_cast<unsigned>(grid), kThreads, 0, stream>>>(w, P_padded, S, tab, block_out);
    *err = cudaGetLastError();
    return static_cast<int>(grid);
}

}  // namespace hadpsgd
