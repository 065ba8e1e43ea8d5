// odb_static.cu -- odb_slot_offsets_static: the output-offset scan (A9; the padded block of a
// group is count x width, padded to the group maximum) for callers that must not
// allocate device memory.
//
// Who that is: a data-loading plugin that runs inside a trainer whose framework has already taken the
// whole HBM for its own caching allocator (a cudaMalloc from a second party then fails, or succeeds by
// pushing the trainer into an out-of-memory error later), and any caller sitting in the middle of a
// training step, where cudaMalloc / cudaFree stall every stream of the device while they run.  Such a
// caller cannot use odb_create either (the context allocates ~70 bytes per sample), so this entry
// point takes no context: inputs and outputs are the caller's, and the only other global memory the
// kernels touch -- the tile records of the single-pass scan -- is the fixed array below, which is part
// of the library image.
//
// The kernel is a variant of k_fin_scan (odb_plan.cu): the same ticketed decoupled look-back, reduced
// to the one quantity the caller asked for.  k_fin_scan itself and every other path are unchanged.
#include <cuda_runtime.h>

#include <mutex>

#include "odb.h"
#include "odb_device.cuh"

namespace {

constexpr int kThreads = 256;                  // threads per CTA
constexpr int kItems = 4;                      // consecutive slots per thread
constexpr int kTile = kThreads * kItems;       // slots per tile (1024)
constexpr int64_t kMaxSlots = ODB_STATIC_MAX_SLOTS;
constexpr int kMaxTiles = (int)(kMaxSlots / kTile);
static_assert(kMaxSlots % kTile == 0, "the maximum is a whole number of tiles");

// Layout of the scratch, in 8-byte words.  Word 0: the tile ticket.  From word kHead on, four words per
// tile: [0] the tile's own sum, [1] the inclusive prefix up to and including the tile, [2] the state
// (0 nothing yet, 1 own sum published, 2 inclusive prefix published), [3] unused.
constexpr int kHead = 32;
constexpr int kWordsPerTile = 4;
constexpr size_t kWords = (size_t)kHead + (size_t)kMaxTiles * kWordsPerTile;

// THE scratch: 128.25 KiB of every GPU that loads libodb.so, held until the process exits.  Every call
// on a device shares it and finds in it what the previous call left.
static __device__ __align__(256) unsigned long long g_static_scratch[kWords];

// Device code of this file may name the array; the clearing pass does.  What has to start at zero is the
// ticket and the state word of every tile the coming scan will use.
__global__ void k_static_clear(int n_tiles) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) g_static_scratch[0] = 0ull;
    if (i < n_tiles) g_static_scratch[kHead + (size_t)i * kWordsPerTile + 2] = 0ull;
}

// offset[s] = sum over s' < s of round_up(count[s'] * width[s'], 16); offset[n_slots] = the total.
// `scratch` is the DEVICE address of g_static_scratch (the host passes what cudaGetSymbolAddress gave it).
__global__ void __launch_bounds__(kThreads)
k_slot_offsets_static(const int32_t *__restrict__ grp_count, const int32_t *__restrict__ grp_width, int64_t n_slots,
                      int64_t *__restrict__ grp_offset, unsigned long long *scratch) {
    __shared__ long long s_scan[34];
    __shared__ long long s_base;
    __shared__ int s_tile;
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch);
    const int n_tiles = n_slots > 0 ? (int)((n_slots + kTile - 1) / kTile) : 1;  // an empty table still writes offset[0]
    for (;;) {
        __syncthreads();  // everyone is done with s_tile / s_base of the previous tile
        if (threadIdx.x == 0) s_tile = (int)atomicAdd(ticket, 1u);  // a ticket: every earlier tile is running or done
        __syncthreads();
        const int tile = s_tile;
        if (tile >= n_tiles) break;
        const int64_t s0 = (int64_t)tile * kTile + (int64_t)threadIdx.x * kItems;
        long long v[kItems];
        long long sum = 0;
#pragma unroll
        for (int i = 0; i < kItems; ++i) {
            const int64_t s = s0 + i;
            long long area = 0;
            if (s < n_slots) area = (long long)grp_count[s] * (long long)grp_width[s];
            v[i] = (area + 15) / 16 * 16;
            sum += v[i];
        }
        long long total;
        const long long ex = odb::block_excl_scan<long long>(sum, s_scan, total);
        unsigned long long *me = scratch + kHead + (size_t)tile * kWordsPerTile;
        int *my_state = reinterpret_cast<int *>(me + 2);
        if (threadIdx.x == 0) {
            me[0] = (unsigned long long)total;
            if (tile == 0) {
                me[1] = (unsigned long long)total;
                s_base = 0;
            }
            odb::st_flag(my_state, tile == 0 ? 2 : 1);
        }
        if (tile > 0 && threadIdx.x < 32) {  // warp 0 looks back, 32 predecessors at a time
            const int lane = threadIdx.x;
            long long acc = 0;
            int t = tile - 1;
            for (;;) {
                const int tt = t - lane;
                int f = 2;  // in front of tile 0: an inclusive prefix of 0
                long long x = 0;
                if (tt >= 0) {
                    const unsigned long long *rec = scratch + kHead + (size_t)tt * kWordsPerTile;
                    do {
                        f = odb::ld_flag(reinterpret_cast<const int *>(rec + 2));
                    } while (f == 0);
                    x = (long long)__ldcg(rec + (f == 2 ? 1 : 0));
                }
                const uint32_t done = __ballot_sync(ODB_FULL_MASK, f == 2);
                const int first = __ffs(done) - 1;  // the nearest predecessor that already knows its prefix
                long long y = (done == 0 || lane <= first) ? x : 0;
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) y += __shfl_xor_sync(ODB_FULL_MASK, y, d);
                acc += y;
                if (done) break;
                t -= 32;
            }
            if (lane == 0) {
                s_base = acc;
                me[1] = (unsigned long long)(acc + total);
                odb::st_flag(my_state, 2);
            }
        }
        __syncthreads();
        long long run = s_base + ex;
#pragma unroll
        for (int i = 0; i < kItems; ++i) {
            const int64_t s = s0 + i;
            if (s < n_slots) grp_offset[s] = run;
            run += v[i];
        }
        if (threadIdx.x == 0 && tile == n_tiles - 1) grp_offset[n_slots] = s_base + total;
    }
}

// ---- host side --------------------------------------------------------------------------------------
// In host code `g_static_scratch` is only a handle for the runtime, not memory a kernel can use.  Its
// device address differs from GPU to GPU and is asked for once per device, with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned long long *g_scratch_addr[kMaxDevices] = {};
thread_local int t_last_cuda = 0;

int cuda_failed(cudaError_t e) {
    t_last_cuda = (int)e;
    return ODB_ERR_CUDA;
}

}  // namespace

extern "C" {

ODB_API int64_t odb_static_max_slots(void) { return kMaxSlots; }

ODB_API int odb_static_last_cuda_error(void) { return t_last_cuda; }

ODB_API int odb_slot_offsets_static(const int32_t *d_grp_count, const int32_t *d_grp_width, int64_t n_slots,
                                    int64_t *d_grp_offset, void *stream) {
    // argument checks first: they need no GPU
    if (n_slots < 0 || !d_grp_offset || (n_slots > 0 && (!d_grp_count || !d_grp_width))) return ODB_ERR_INVALID_ARG;
    if (n_slots > kMaxSlots) return ODB_ERR_CAPACITY;  // more slots than the fixed scratch has tile records for
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_failed(e);
    if (dev < 0 || dev >= kMaxDevices) return ODB_ERR_INVALID_ARG;
    unsigned long long *scratch;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_scratch_addr[dev]) {  // first call on this device: it is the current one
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e != cudaSuccess) return cuda_failed(e);
            g_scratch_addr[dev] = static_cast<unsigned long long *>(p);
        }
        scratch = g_scratch_addr[dev];
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int n_tiles = n_slots > 0 ? (int)((n_slots + kTile - 1) / kTile) : 1;
    k_static_clear<<<(n_tiles + 255) / 256, 256, 0, st>>>(n_tiles);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_failed(e);
    const int grid = n_tiles < 592 ? n_tiles : 592;  // 148 SMs x 4; the tickets hand out the remaining tiles
    k_slot_offsets_static<<<grid, kThreads, 0, st>>>(d_grp_count, d_grp_width, n_slots, d_grp_offset, scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_failed(e);
    return ODB_OK;
}

}  // extern "C"
