// consensus_noalloc.cu -- hadpsgd_consensus_noalloc(): the consensus distance
//   D = sum_i sum_s (w_s[i] - wbar[i])^2 ,  wbar[i] = (1/S) sum_s w_s[i]
// for callers that must not allocate device memory.
//
// Who that is.  hadpsgd_consensus() works on a handle, and a handle needs an arena: either the
// library cudaMallocs it, or the caller carves hadpsgd_required_bytes() out of its own memory.  Some
// users of this library can do neither at the moment they want D:
//   * a training process whose framework allocator (torch's caching allocator and the like) has
//     already reserved nearly all of the GPU's memory -- a raw cudaMalloc from inside a library then
//     fails although "free" memory exists inside the framework's pool;
//   * a monitor that runs between two training steps of a latency-bound loop: cudaMalloc and cudaFree
//     synchronise the whole device, so every stream of the process would stall on a diagnostic;
//   * a hook that only BORROWS the S weight buffers (say S parameter tensors of a framework) and owns
//     no arena in which the block partials of the reduction could live.
// For them the block partials live in a fixed array that is part of the loaded library image
// (g_scratch below): HADPSGD_NOALLOC_SCRATCH_BYTES per GPU that runs this entry point, held until the
// process exits.  The caller passes only inputs (the S weight pointers) and the output (one double).
//
// The kernel is a variant of consensus_kernel (consensus.cu): same per-thread arithmetic, same
// grid-stride partition, same fixed-order sums -- but the S buffers come as S pointers instead of
// base + slot table, a ragged tail (n not a multiple of 4) is handled, and the final sum over the
// block partials is formed on the device by the last block to finish (ticket counter) instead of on
// the host, so the result lands in device memory without a copy or a synchronisation.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/hadpsgd.h"

namespace {

constexpr int kThreads = 256;
constexpr int kMaxBlocks = HADPSGD_NOALLOC_MAX_BLOCKS;
constexpr int kTicketSlot = kMaxBlocks;      // the ticket counter sits behind the partials, on a 256 B line of its own
constexpr int kScratchDoubles = kMaxBlocks + 32;
static_assert(kScratchDoubles * sizeof(double) == HADPSGD_NOALLOC_SCRATCH_BYTES, "header and scratch array disagree");

// The scratch.  In HOST code this name is only a stand-in symbol of the host image -- never a device
// address; the launch below gets the real address from cudaGetSymbolAddress (scratch_of_device()).
// Zero at module load.  Contents between calls: partial[0..grid) of the last call (overwritten before
// they are read), and the ticket counter, which the last block of every call puts back to zero.
static __device__ __align__(256) double g_scratch[kScratchDoubles];

struct PtrTable { const float* w[HADPSGD_NOALLOC_MAX_S]; };

__global__ void __launch_bounds__(kThreads) consensus_noalloc_kernel(const __grid_constant__ PtrTable tab, long long n,
                                                                     int S, double* __restrict__ scratch,
                                                                     double* __restrict__ D_out) {
    __shared__ double s_red[kThreads / 32];
    __shared__ double s_part[kMaxBlocks];
    __shared__ bool s_last;
    const long long n_units = n / 4;
    const double inv = 1.0 / static_cast<double>(S);
    double acc = 0.;
    for (long long t = static_cast<long long>(blockIdx.x) * kThreads + threadIdx.x; t < n_units;
         t += static_cast<long long>(gridDim.x) * kThreads) {
        double m0 = 0., m1 = 0., m2 = 0., m3 = 0.;
        for (int s = 0; s < S; ++s) {   // pass 1: the mean, in double, s = 0..S-1
            const float4 x = reinterpret_cast<const float4*>(tab.w[s])[t];
            m0 += x.x; m1 += x.y; m2 += x.z; m3 += x.w;
        }
        m0 *= inv; m1 *= inv; m2 *= inv; m3 *= inv;
        for (int s = 0; s < S; ++s) {   // pass 2: squared deviations (the re-read hits L1/L2)
            const float4 x = reinterpret_cast<const float4*>(tab.w[s])[t];
            const double d0 = x.x - m0, d1 = x.y - m1, d2 = x.z - m2, d3 = x.w - m3;
            acc += d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x < static_cast<unsigned>(n & 3)) {   // ragged tail: up to 3 single elements
        const long long i = n_units * 4 + threadIdx.x;
        double m = 0.;
        for (int s = 0; s < S; ++s) m += tab.w[s][i];
        m *= inv;
        for (int s = 0; s < S; ++s) { const double d = tab.w[s][i] - m; acc += d * d; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = acc;
    __syncthreads();
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + kTicketSlot);
    if (threadIdx.x == 0) {
        double tot = 0.;
        for (int i = 0; i < kThreads / 32; ++i) tot += s_red[i];   // fixed order
        scratch[blockIdx.x] = tot;
        __threadfence();                                           // the partial is visible before the ticket is taken
        s_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    // Last block to finish: every partial of this launch is in scratch[0..grid).  Entries beyond the
    // grid belong to an earlier, larger call and are not touched.
    __threadfence();
    for (int i = threadIdx.x; i < static_cast<int>(gridDim.x); i += kThreads) s_part[i] = __ldcg(scratch + i);
    __syncthreads();
    if (threadIdx.x == 0) {
        double D = 0.;
        for (int i = 0; i < static_cast<int>(gridDim.x); ++i) D += s_part[i];   // b = 0..grid-1: run-to-run deterministic
        *D_out = D;
        *ticket = 0u;   // the next call (after this one in stream order) starts from zero again
    }
}

// ---- host side -----------------------------------------------------------------------------

thread_local char g_error[256] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    std::vsnprintf(g_error, sizeof g_error, fmt, ap);
    va_end(ap);
    return code;
}

constexpr int kMaxDevices = 64;
struct DeviceState { double* scratch = nullptr; int num_sms = 0; bool ready = false; };
std::mutex g_mutex;
DeviceState g_device[kMaxDevices];

// Set-up, once per device, with that device current: the DEVICE address of g_scratch on this GPU
// (every device that loads the library has its own instance of the array).
int scratch_of_device(int dev, cudaStream_t stream, DeviceState* out) {
    std::lock_guard<std::mutex> lock(g_mutex);
    DeviceState& st = g_device[dev];
    if (!st.ready) {
        int major = 0, sms = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return fail(HADPSGD_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        if (major != 10) return fail(HADPSGD_UNSUPPORTED_DEVICE, "libhadpsgd is built for sm_100a only; device %d is sm_%dx", dev, major);
        double* ptr = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_scratch);
        if (e != cudaSuccess || !ptr) return fail(HADPSGD_CUDA, "cudaGetSymbolAddress(g_scratch): %s", cudaGetErrorString(e));
        // the ticket counter must start at zero: it does at module load, and it is cleared once more here
        // so that this does not rest on the loader; ordered before the first launch on the caller's stream
        e = cudaMemsetAsync(ptr + kTicketSlot, 0, 256, stream);
        if (e != cudaSuccess) return fail(HADPSGD_CUDA, "cudaMemsetAsync(ticket): %s", cudaGetErrorString(e));
        st.scratch = ptr; st.num_sms = sms; st.ready = true;
    }
    *out = st;
    return HADPSGD_OK;
}

}  // namespace

extern "C" const char* hadpsgd_consensus_noalloc_error(void) { return g_error; }

extern "C" int hadpsgd_consensus_noalloc(const float* const* w, int S, int64_t n, double* D_out, void* stream_) {
    g_error[0] = 0;
    // argument checks first: they need no GPU
    if (!w || !D_out) return fail(HADPSGD_INVALID_ARG, "w and D_out must not be NULL");
    if (S < 1) return fail(HADPSGD_INVALID_ARG, "S = %d: need at least one weight buffer", S);
    if (S > HADPSGD_NOALLOC_MAX_S)
        return fail(HADPSGD_INVALID_ARG, "S = %d exceeds HADPSGD_NOALLOC_MAX_S = %d (the pointer table of the no-allocation "
                    "entry point is fixed-size; use hadpsgd_consensus on a handle for more)", S, HADPSGD_NOALLOC_MAX_S);
    if (n < 0 || n > HADPSGD_NOALLOC_MAX_ELEMS)
        return fail(HADPSGD_INVALID_ARG, "n = %lld elements per buffer is outside [0, HADPSGD_NOALLOC_MAX_ELEMS = %lld]",
                    static_cast<long long>(n), static_cast<long long>(HADPSGD_NOALLOC_MAX_ELEMS));
    PtrTable tab;
    for (int s = 0; s < S; ++s) {
        if (!w[s]) return fail(HADPSGD_INVALID_ARG, "w[%d] is NULL", s);
        if (reinterpret_cast<uintptr_t>(w[s]) % 16 != 0) return fail(HADPSGD_INVALID_ARG, "w[%d] is not 16-byte aligned", s);
        tab.w[s] = w[s];
    }
    for (int s = S; s < HADPSGD_NOALLOC_MAX_S; ++s) tab.w[s] = nullptr;
    if (reinterpret_cast<uintptr_t>(D_out) % 8 != 0) return fail(HADPSGD_INVALID_ARG, "D_out is not 8-byte aligned");

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(HADPSGD_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(HADPSGD_INVALID_ARG, "device ordinal %d is beyond the %d this entry point tracks", dev, kMaxDevices);
    // a plain host pointer would fault inside the kernel: refuse it here (no allocation, no stream work)
    for (int s = 0; s <= S; ++s) {
        const void* p = s < S ? static_cast<const void*>(w[s]) : static_cast<const void*>(D_out);
        cudaPointerAttributes attr;
        e = cudaPointerGetAttributes(&attr, p);
        if (e != cudaSuccess) return fail(HADPSGD_CUDA, "cudaPointerGetAttributes: %s", cudaGetErrorString(e));
        if (attr.type == cudaMemoryTypeUnregistered) {
            char name[24];
            if (s < S) std::snprintf(name, sizeof name, "w[%d]", s); else std::snprintf(name, sizeof name, "D_out");
            return fail(HADPSGD_INVALID_ARG, "%s is a plain host pointer: this entry point takes DEVICE pointers", name);
        }
    }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    DeviceState st;
    const int rc = scratch_of_device(dev, stream, &st);
    if (rc != HADPSGD_OK) return rc;

    const long long want = (n / 4 + kThreads - 1) / kThreads;
    long long grid = static_cast<long long>(st.num_sms) * 8;   // as launch_consensus (consensus.cu)
    if (grid > want) grid = want;
    if (grid > kMaxBlocks) grid = kMaxBlocks;                  // one partial slot per block: the scratch bounds the grid, not n
    if (grid < 1) grid = 1;
    consensus_noalloc_kernel<<<static_cast<unsigned>(grid), kThreads, 0, stream>>>(tab, n, S, st.scratch, D_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(HADPSGD_CUDA, "consensus_noalloc_kernel launch: %s", cudaGetErrorString(e));
    return HADPSGD_OK;
}
