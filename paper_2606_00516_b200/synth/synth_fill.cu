// Device-side twin of synth/gen.py: fills a bf16 buffer with the seeded N(0,1) stream
// value(seed, tensor_id, index).  Input generation only — none of the method's arithmetic.
// Built as its own library (libpa_synth.so); cross-checked bit-for-bit against gen.py in tests.
#include <cuda_runtime.h>
#include <cstdint>

namespace {

__host__ __device__ inline uint64_t splitmix64(uint64_t x) {
    uint64_t z = x + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__device__ inline uint16_t value_bits(uint64_t key, uint64_t idx) {
    const uint64_t h0 = splitmix64(key + 2 * idx), h1 = splitmix64(key + 2 * idx + 1);
    int s = 0;
#pragma unroll
    for (int f = 0; f < 6; ++f) {
        s += (int)((h0 >> (10 * f)) & 0x3FF);
        s += (int)((h1 >> (10 * f)) & 0x3FF);
    }
    const float x = (float)(2 * s - 12276) * 4.8828125e-4f;  // * 2^-11, exact
    uint32_t u = __float_as_uint(x);
    u += 0x7FFFu + ((u >> 16) & 1u);                          // RNE to bf16
    return (uint16_t)(u >> 16);
}

__global__ void fill_kernel(uint16_t* dst, int64_t n, uint64_t key, int64_t start) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x * 8;
    for (int64_t base = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 8; base < n; base += stride) {
        if (base + 8 <= n && ((reinterpret_cast<uintptr_t>(dst + base) & 15) == 0)) {
            uint32_t w[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint32_t lo = value_bits(key, (uint64_t)(start + base + 2 * i));
                const uint32_t hi = value_bits(key, (uint64_t)(start + base + 2 * i + 1));
                w[i] = lo | (hi << 16);
            }
            *reinterpret_cast<uint4*>(dst + base) = make_uint4(w[0], w[1], w[2], w[3]);
        } else {
            for (int64_t i = base; i < n && i < base + 8; ++i) dst[i] = value_bits(key, (uint64_t)(start + i));
        }
    }
}

}  // namespace

extern "C" int32_t synth_fill_bf16(void* dst, int64_t n, uint64_t seed, uint32_t tensor_id, int64_t start, void* stream) {
    if (n <= 0) return 0;
    const uint64_t key = splitmix64(seed * 0x100000001B3ull + (uint64_t)tensor_id);
    const int block = 256;
    int64_t want = (n / 8 + block - 1) / block + 1;
    const int grid = (int)(want < 148 * 16 ? want : 148 * 16);
    fill_kernel<<<grid, block, 0, static_cast<cudaStream_t>(stream)>>>(static_cast<uint16_t*>(dst), n, key, start);
    return (int32_t)cudaGetLastError();
}
