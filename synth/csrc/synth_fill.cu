// CUDA twin of synth/gen.py: fills a device buffer with the seeded synthetic values (harness, not method).
// Holds none of the method's arithmetic.  See synth/gen.py for the recipe.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {
__device__ __forceinline__ uint64_t mix(uint64_t z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__device__ __forceinline__ int sum16(uint64_t h) {
    return (int)(h & 0xFFFF) + (int)((h >> 16) & 0xFFFF) + (int)((h >> 32) & 0xFFFF) + (int)(h >> 48);
}
__device__ __forceinline__ float value(uint64_t base, uint64_t x, float c) {
    const uint64_t G = 0x9E3779B97F4A7C15ull;
    const int S = sum16(mix(base + (2 * x) * G)) + sum16(mix(base + (2 * x + 1) * G));
    return __fmul_rn((float)(S - 262140), c);
}
__global__ void fill_kernel(void* out, uint64_t base, uint64_t start, uint64_t count, float c, int bf16) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (uint64_t)gridDim.x * blockDim.x) {
        const float w = value(base, start + i, c);
        if (bf16) {
            uint32_t b = __float_as_uint(w);
            b += 0x7FFFu + ((b >> 16) & 1u);
            static_cast<uint16_t*>(out)[i] = (uint16_t)(b >> 16);
        } else {
            static_cast<float*>(out)[i] = w;
        }
    }
}
}  // namespace

// kind: 0 weight (sigma 0.02), 1 N(0,1).  bf16: 1 -> uint16 bf16 bits, 0 -> float.  Returns cudaError_t.
extern "C" int synth_fill(void* d_out, uint64_t seed, uint64_t tensor, uint64_t start, uint64_t count, int kind,
                          int bf16, void* stream) {
    if (count == 0) return 0;
    const uint64_t G = 0x9E3779B97F4A7C15ull;
    auto hmix = [](uint64_t z) {
        z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
        z ^= z >> 27; z *= 0x94D049BB133111EBull;
        return z ^ (z >> 31);
    };
    const uint64_t base = hmix(hmix(seed + G) ^ (tensor * 0xD1B54A32D192ED03ull + 0x8CB92BA72F3D8DD7ull));
    union { uint32_t u; float f; } c;
    c.u = kind == 0 ? 0x34C8A986u : 0x379CC471u;
    uint64_t blocks = (count + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    fill_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(d_out, base, start, count, c.f, bf16);
    return (int)cudaGetLastError();
}
