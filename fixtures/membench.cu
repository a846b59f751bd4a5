// membench.cu -- FIXTURE: this device's streaming ceilings, measured with the access shape of the
// step kernel (persistent grid of one 256-thread block per SM, 32-byte vector accesses carrying L2
// evict_first, `n_streams` buffers walked in lock step).  bench.py uses the pure-read and pure-write
// rates to state a ceiling for a kernel's own byte mix:  t >= bytes_read / BW_read + bytes_written /
// BW_write  (reads and writes share one DRAM bus).  Holds none of the method's arithmetic and is
// linked into neither libhadpsgd.so nor the oracle.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

struct Raw8 { unsigned u[8]; };
__device__ __forceinline__ Raw8 ld32(const void* p) {
    Raw8 r;
    asm volatile("ld.global.L1::no_allocate.L2::evict_first.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r.u[0]), "=r"(r.u[1]), "=r"(r.u[2]), "=r"(r.u[3]), "=r"(r.u[4]), "=r"(r.u[5]), "=r"(r.u[6]), "=r"(r.u[7])
                 : "l"(p));
    return r;
}
__device__ __forceinline__ void st32(void* p, const Raw8& r) {
    asm volatile("st.global.L1::no_allocate.L2::evict_first.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "l"(p), "r"(r.u[0]), "r"(r.u[1]), "r"(r.u[2]), "r"(r.u[3]), "r"(r.u[4]), "r"(r.u[5]), "r"(r.u[6]), "r"(r.u[7])
                 : "memory");
}

constexpr int kThreads = 256;
constexpr int kMaxStreams = 12;

// buf holds n_streams streams of stream_bytes each, back to back.  Tile t covers bytes
// [t * 8 KB, (t+1) * 8 KB) of EVERY stream; block b walks tiles b, b+grid, ...
template <int NS, bool WRITE>
__global__ void __launch_bounds__(kThreads, 1) stream_kernel(char* buf, long long stream_bytes, unsigned* sink) {
    const long long tiles = stream_bytes / (kThreads * 32);
    unsigned acc = 0;
    for (long long t = blockIdx.x; t < tiles; t += gridDim.x) {
        const long long off = t * (kThreads * 32) + threadIdx.x * 32;
        if constexpr (WRITE) {
            Raw8 r;
#pragma unroll
            for (int q = 0; q < 8; ++q) r.u[q] = static_cast<unsigned>(t) + q;
#pragma unroll
            for (int s = 0; s < NS; ++s) st32(buf + s * stream_bytes + off, r);
        } else {
            Raw8 r[NS];
#pragma unroll
            for (int s = 0; s < NS; ++s) r[s] = ld32(buf + s * stream_bytes + off);
#pragma unroll
            for (int s = 0; s < NS; ++s)
#pragma unroll
                for (int q = 0; q < 8; ++q) acc ^= r[s].u[q];
        }
    }
    if (!WRITE && acc == 0x9e3779b9u) *sink = acc;   // keeps the loads alive
}

template <bool WRITE>
int launch(int n_streams, char* buf, long long stream_bytes, unsigned* sink, int grid, cudaStream_t st) {
    switch (n_streams) {
        case 1: stream_kernel<1, WRITE><<<grid, kThreads, 0, st>>>(buf, stream_bytes, sink); break;
        case 2: stream_kernel<2, WRITE><<<grid, kThreads, 0, st>>>(buf, stream_bytes, sink); break;
        case 4: stream_kernel<4, WRITE><<<grid, kThreads, 0, st>>>(buf, stream_bytes, sink); break;
        case 6: stream_kernel<6, WRITE><<<grid, kThreads, 0, st>>>(buf, stream_bytes, sink); break;
        case 8: stream_kernel<8, WRITE><<<grid, kThreads, 0, st>>>(buf, stream_bytes, sink); break;
        case 12: stream_kernel<12, WRITE><<<grid, kThreads, 0, st>>>(buf, stream_bytes, sink); break;
        default: return static_cast<int>(cudaErrorInvalidValue);
    }
    return static_cast<int>(cudaGetLastError());
}

}  // namespace

// dev_buf: DEVICE buffer of at least n_streams * stream_bytes bytes (stream_bytes a multiple of 8 KB)
// plus 4 bytes the kernel may write a dummy word to at dev_sink.  write: 0 = read every byte once,
// 1 = write every byte once.  Asynchronous on `stream`; the caller times it with events.  n_streams in
// {1, 2, 4, 6, 8, 12}.  Returns the cudaError_t of the launch.
extern "C" int hadpsgd_fixture_membench(void* dev_buf, long long stream_bytes, int n_streams, int write,
                                        void* dev_sink, void* stream) {
    if (!dev_buf || stream_bytes <= 0 || stream_bytes % (kThreads * 32) != 0 || n_streams > kMaxStreams)
        return static_cast<int>(cudaErrorInvalidValue);
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    char* buf = static_cast<char*>(dev_buf);
    unsigned* sink = static_cast<unsigned*>(dev_sink);
    return write ? launch<true>(n_streams, buf, stream_bytes, sink, sms, st)
                 : launch<false>(n_streams, buf, stream_bytes, sink, sms, st);
}
