// Bandwidth probes (measurement utility, not part of the method): what the collate kernel's byte MIX --
// 4 bytes read per element, 13 bytes written (3 x int32 + 1 x uint8) -- can reach on this device with trivial
// indexing, in the two store forms the collate kernel can use, next to a pure-store stream and a plain copy.
// bench.py reports them as roofline.mix_ceiling, so that the collate kernel's fraction is read against a
// ceiling with its own read/write ratio and not only against a 50/50 copy.  sm_100a only.
#include "odb_internal.cuh"

namespace odb {

constexpr int kPbThreads = 256;
constexpr int kPbChunk = 512;  // elements per warp iteration: one 16-element unit per lane, as in k_collate
constexpr int kPbStage = 3 * kPbChunk * 4 + kPbChunk;  // bytes of one warp's staging buffer (bulk-store forms)

__device__ __forceinline__ void pb_st256(int32_t *p, const int32_t (&v)[16], int o) {
    asm volatile("st.global.cs.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(v[o]), "r"(v[o + 1]), "r"(v[o + 2]),
                 "r"(v[o + 3]), "r"(v[o + 4]), "r"(v[o + 5]), "r"(v[o + 6]), "r"(v[o + 7])
                 : "memory");
}
__device__ __forceinline__ void pb_bulk_store(void *gdst, const void *ssrc, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst),
                 "r"((uint32_t)__cvta_generic_to_shared(ssrc)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void pb_bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void pb_bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void pb_bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void pb_fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// KIND 0: mix, 256-bit streaming stores   1: mix, bulk (TMA) stores from shared memory
//      2: stores only, 256-bit            3: stores only, bulk          4: copy (4 B read, 4 B written, 256-bit stores)
template <int KIND>
__global__ void __launch_bounds__(kPbThreads, 3)
k_probe(const int32_t *__restrict__ in, int32_t *__restrict__ o0, int32_t *__restrict__ o1, int32_t *__restrict__ o2,
        uint8_t *__restrict__ o3, int64_t n_chunks, unsigned long long *counter) {
    extern __shared__ __align__(128) unsigned char pb_smem[];
    constexpr bool kBulk = (KIND == 1 || KIND == 3);
    constexpr bool kRead = (KIND == 0 || KIND == 1 || KIND == 4);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char *stage = pb_smem + (size_t)warp * kPbStage;
    // the work distribution of k_collate: persistent CTAs take runs of 16 tiles (8 chunks each) from a counter
    __shared__ long long s_grab;
    constexpr int kWarps = kPbThreads / 32, kGrab = 16;
    const int64_t n_tiles = (n_chunks + kWarps - 1) / kWarps;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_grab = (long long)atomicAdd(counter, (unsigned long long)kGrab);
        __syncthreads();
        const int64_t t0 = s_grab;
        if (t0 >= n_tiles) break;
        const int64_t t1 = min(t0 + kGrab, n_tiles);
#pragma unroll 1
    for (int64_t tile = t0; tile < t1; ++tile) {
        const int64_t c = tile * kWarps + warp;
        if (c >= n_chunks) break;
        const int64_t a = c * kPbChunk + 16 * lane;
        int32_t x[16];
        if (kRead) {
            const int4 *p = reinterpret_cast<const int4 *>(in + a);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int4 v = __ldg(p + i);
                x[4 * i] = v.x;
                x[4 * i + 1] = v.y;
                x[4 * i + 2] = v.z;
                x[4 * i + 3] = v.w;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) x[i] = (int32_t)a + i;
        }
        if (KIND == 4) {
            pb_st256(o0 + a, x, 0);
            pb_st256(o0 + a + 8, x, 8);
        } else {
        int32_t y[16], z[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            y[i] = x[i] ^ 0x55;
            z[i] = (int32_t)(a & 0xffff) + i;
        }
        const int4 m = make_int4(0x01010101, 0x01010101, 0x01010101, x[0] & 0x01010101);
        if (!kBulk) {
            pb_st256(o0 + a, x, 0);
            pb_st256(o0 + a + 8, x, 8);
            pb_st256(o1 + a, y, 0);
            pb_st256(o1 + a + 8, y, 8);
            pb_st256(o2 + a, z, 0);
            pb_st256(o2 + a + 8, z, 8);
            __stcs(reinterpret_cast<int4 *>(o3 + a), m);
        } else {
            if (lane == 0) pb_bulk_wait_read();  // the previous chunk's bulk stores have read the staging buffer
            __syncwarp();
            int4 *s0 = reinterpret_cast<int4 *>(stage) + 4 * lane;
            int4 *s1 = reinterpret_cast<int4 *>(stage + kPbChunk * 4) + 4 * lane;
            int4 *s2 = reinterpret_cast<int4 *>(stage + 2 * kPbChunk * 4) + 4 * lane;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                s0[i] = make_int4(x[4 * i], x[4 * i + 1], x[4 * i + 2], x[4 * i + 3]);
                s1[i] = make_int4(y[4 * i], y[4 * i + 1], y[4 * i + 2], y[4 * i + 3]);
                s2[i] = make_int4(z[4 * i], z[4 * i + 1], z[4 * i + 2], z[4 * i + 3]);
            }
            reinterpret_cast<int4 *>(stage + 3 * kPbChunk * 4)[lane] = m;
            pb_fence_async();
            __syncwarp();
            if (lane == 0) {
                const int64_t a0 = c * kPbChunk;
                pb_bulk_store(o0 + a0, stage, kPbChunk * 4);
                pb_bulk_store(o1 + a0, stage + kPbChunk * 4, kPbChunk * 4);
                pb_bulk_store(o2 + a0, stage + 2 * kPbChunk * 4, kPbChunk * 4);
                pb_bulk_store(o3 + a0, stage + 3 * kPbChunk * 4, kPbChunk);
                pb_bulk_commit();
            }
        }
        }
    }
    }
    if (kBulk) {
        if (lane == 0) pb_bulk_wait_all();
        __syncwarp();
    }
}

template <int KIND>
static cudaError_t run_probe(const int32_t *in, int32_t *o0, int32_t *o1, int32_t *o2, uint8_t *o3, int64_t n_chunks,
                             int blocks, unsigned long long *counter, cudaStream_t st) {
    constexpr bool kBulk = (KIND == 1 || KIND == 3);
    const size_t smem = kBulk ? (size_t)(kPbThreads / 32) * kPbStage : 0;
    if (kBulk) {
        cudaError_t e = cudaFuncSetAttribute(k_probe<KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    cudaError_t e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    k_probe<KIND><<<blocks, kPbThreads, smem, st>>>(in, o0, o1, o2, o3, n_chunks, counter);
    return cudaGetLastError();
}

}  // namespace odb

using namespace odb;

extern "C" int odb_probe_bandwidth(int kind, const int32_t *d_in, int32_t *d_out0, int32_t *d_out1, int32_t *d_out2,
                                   uint8_t *d_out3, int64_t n_elems, int reps, void *stream, float *h_ms) {
    if (kind < 0 || kind > 4 || !h_ms || n_elems < kPbChunk || reps < 1 || !d_out0) return ODB_ERR_INVALID_ARG;
    if ((kind == 0 || kind == 1 || kind == 4) && !d_in) return ODB_ERR_INVALID_ARG;
    if (kind != 4 && (!d_out1 || !d_out2 || !d_out3)) return ODB_ERR_INVALID_ARG;
    if (((uintptr_t)d_in | (uintptr_t)d_out0 | (uintptr_t)d_out1 | (uintptr_t)d_out2 | (uintptr_t)d_out3) & 15u)
        return ODB_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) != cudaSuccess) return ODB_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int64_t n_chunks = n_elems / kPbChunk;
    const int blocks = (int)std::min<int64_t>((n_chunks + 127) / 128, (int64_t)sms * 3);
    cudaEvent_t e0, e1;
    unsigned long long *counter = nullptr;
    if (cudaMalloc((void **)&counter, sizeof(unsigned long long)) != cudaSuccess) return ODB_ERR_CUDA;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return ODB_ERR_CUDA;
    cudaError_t e = cudaSuccess;
    for (int i = 0; i <= reps && e == cudaSuccess; ++i) {  // rep 0 is a warm-up
        if (i == 1) cudaEventRecord(e0, st);
        switch (kind) {
        case 0: e = run_probe<0>(d_in, d_out0, d_out1, d_out2, d_out3, n_chunks, blocks, counter, st); break;
        case 1: e = run_probe<1>(d_in, d_out0, d_out1, d_out2, d_out3, n_chunks, blocks, counter, st); break;
        case 2: e = run_probe<2>(d_in, d_out0, d_out1, d_out2, d_out3, n_chunks, blocks, counter, st); break;
        case 3: e = run_probe<3>(d_in, d_out0, d_out1, d_out2, d_out3, n_chunks, blocks, counter, st); break;
        default: e = run_probe<4>(d_in, d_out0, d_out1, d_out2, d_out3, n_chunks, blocks, counter, st); break;
        }
    }
    cudaEventRecord(e1, st);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(counter);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return ODB_ERR_CUDA;
    }
    *h_ms = ms / (float)reps;
    return ODB_OK;
}
