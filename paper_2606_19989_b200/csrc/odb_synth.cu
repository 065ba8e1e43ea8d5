// Synthetic input utility: fills a device token buffer with the counter-based ids of DESIGN.md
// "Input recipe" (SplitMix64 finaliser of the global token index), so benchmarks need no multi-GB
// upload.  Input generation only: none of the method's arithmetic lives here.  The CPU side has its
// own implementation of the same specification (odb_inputs/gen.py); the two share no code.
#include <cuda_runtime.h>
#include <stdint.h>

#include "odb.h"

namespace {

__device__ __forceinline__ uint64_t mix64(uint64_t z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}

__global__ void k_synth_tokens(int32_t *__restrict__ out, uint64_t base, int64_t start, int64_t count, uint32_t vocab) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < count; j += stride) {
        const uint64_t hi = mix64(base + (uint64_t)(start + j)) >> 32;
        out[j] = (int32_t)((hi * (uint64_t)vocab) >> 32);
    }
}

}  // namespace

extern "C" int odb_synth_tokens(int32_t *d_tokens, int64_t start, int64_t count, uint64_t seed, int32_t vocab, void *stream) {
    if (count < 0 || vocab < 1 || (count > 0 && !d_tokens)) return ODB_ERR_INVALID_ARG;
    if (count == 0) return ODB_OK;
    int64_t blocks = (count + 1023) / 1024;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_synth_tokens<<<(int)blocks, 256, 0, (cudaStream_t)stream>>>(d_tokens, seed * 0x9E3779B97F4A7C15ull, start, count,
                                                                  (uint32_t)vocab);
    return cudaGetLastError() == cudaSuccess ? ODB_OK : ODB_ERR_CUDA;
}
