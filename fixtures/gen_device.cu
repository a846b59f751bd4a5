// gen_device.cu -- FIXTURE: device-side twin of fixtures/generator.py.
//
// Fills device buffers with the same counter-hash values as the numpy generator, bit for
// bit (integer shaping + one fp32 multiply, no libm), so the 55 GB working sets of the
// full-size configs never have to cross PCIe.  Holds none of the method's arithmetic and
// is linked into neither libhadpsgd.so nor the oracle.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ uint64_t mix64(uint64_t x) {
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
__device__ __forceinline__ uint64_t raw_bits(uint64_t key, long long i) {
    return mix64(key + 0x9E3779B97F4A7C15ull * static_cast<uint64_t>(i + 1));
}
__device__ __forceinline__ float shape_uniform(uint64_t x, float scale) {
    int k = static_cast<int>(x >> 40) - (1 << 23);
    return __fmul_rn(static_cast<float>(k), scale);
}
__device__ __forceinline__ float shape_normal(uint64_t x, float scale) {
    int t = static_cast<int>(x & 0xFFFF) + static_cast<int>((x >> 16) & 0xFFFF) +
            static_cast<int>((x >> 32) & 0xFFFF) + static_cast<int>(x >> 48);
    return __fmul_rn(static_cast<float>(t - 131070), scale);
}
__device__ __forceinline__ uint16_t bf16_rne(float f) {
    uint32_t b = __float_as_uint(f);
    return static_cast<uint16_t>((b + 0x7FFFu + ((b >> 16) & 1u)) >> 16);
}

// dist: 0 uniform, 1 normal (Irwin-Hall n=4).  out_bf16: 0 -> float, 1 -> bf16 bits.
__global__ void fill_kernel(void* out, long long n, long long elem_offset, uint64_t key, float scale,
                            int dist, int out_bf16) {
    long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
    for (long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; i < n; i += stride) {
        uint64_t x = raw_bits(key, elem_offset + i);
        float f = dist == 0 ? shape_uniform(x, scale) : shape_normal(x, scale);
        if (out_bf16) static_cast<uint16_t*>(out)[i] = bf16_rne(f);
        else static_cast<float*>(out)[i] = f;
    }
}

}  // namespace

// dev_out: DEVICE pointer to n elements (float or bf16).  Writes value(elem_offset + i) to
// dev_out[i].  Asynchronous on `stream`.  Returns the cudaError_t of the launch.
extern "C" int hadpsgd_fixture_fill(void* dev_out, long long n, long long elem_offset, uint64_t key,
                                    float scale, int dist, int out_bf16, void* stream) {
    if (n <= 0) return 0;
    long long blocks = (n + 255) / 256;
    static int cap = 0;                      // 16 blocks per SM of the current device
    if (cap == 0) {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
            sms = 128;
        cap = sms * 16;
    }
    if (blocks > cap) blocks = cap;
    fill_kernel<<<static_cast<unsigned>(blocks), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        dev_out, n, elem_offset, key, scale, dist, out_bf16);
    return static_cast<int>(cudaGetLastError());
}
