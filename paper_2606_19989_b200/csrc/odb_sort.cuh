// Device-side pieces of the window sort (A0 + A1), shared by the cluster sort kernel (odb_sort.cu) and the
// persistent round-loop kernel (odb_rounds.cu): a CTA merge-sorts 4096 64-bit keys in shared memory.
#pragma once

#include "odb_device.cuh"
#include "odb_internal.cuh"

namespace odb {

constexpr int kMsThreads = 256;
constexpr int kMsItems = 16;
constexpr int kMsChunk = kMsThreads * kMsItems;  // 4096 keys per CTA
static_assert(kMsChunk == kSortChunk, "one CTA sorts one chunk");
constexpr int kMsPadded = kMsChunk + kMsChunk / 16;  // one spare key per 16: conflict-free 16-key runs

__device__ __forceinline__ int ms_pad(int i) { return i + (i >> 4); }

// ---- cluster / DSMEM primitives (PTX; no cooperative-groups dependency) --------------------------
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cluster_map(uint32_t addr, uint32_t cta) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(cta));
    return r;
}
__device__ __forceinline__ uint64_t ld_dsmem_u64(uint32_t addr) {
    uint64_t v;
    asm volatile("ld.shared::cluster.u64 %0, [%1];" : "=l"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

__device__ __forceinline__ void ms_cmp_xchg(uint64_t &lo, uint64_t &hi, bool asc) {
    const bool sw = (lo > hi) == asc;
    const uint64_t a = sw ? hi : lo, b = sw ? lo : hi;
    lo = a;
    hi = b;
}

// ascending sort of 16 keys in registers: the bitonic network (10 stages, 80 compare-exchanges)
__device__ __forceinline__ void ms_sort16(uint64_t (&k)[16]) {
#pragma unroll
    for (int kk = 2; kk <= 16; kk <<= 1) {
#pragma unroll
        for (int j = kk >> 1; j > 0; j >>= 1) {
#pragma unroll
            for (int r = 0; r < 16; ++r)
                if ((r & j) == 0) ms_cmp_xchg(k[r], k[r | j], kk == 16 || (r & kk) == 0);
        }
    }
}

// keys taken from run a (na keys) among the first d outputs of merge(a, b); runs are in PADDED local shared memory
__device__ __forceinline__ int ms_path_local(const uint64_t *X, int a0, int na, int b0, int nb, int d) {
    int lo = max(0, d - nb), hi = min(d, na);
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (X[ms_pad(a0 + mid)] < X[ms_pad(b0 + d - 1 - mid)]) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

// 16 outputs of merge(X[a.. a_end), X[b.. b_end)) starting at the split (ai, bi), into registers
__device__ __forceinline__ void ms_merge16(const uint64_t *X, int ai, int a_end, int bi, int b_end, uint64_t (&out)[16]) {
    uint64_t ka = ai < a_end ? X[ms_pad(ai)] : ~0ull;
    uint64_t kb = bi < b_end ? X[ms_pad(bi)] : ~0ull;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        // keys are unique (the id is part of the key), padding keys (~0) sort last: ties are irrelevant
        const bool take_a = (bi >= b_end) || (ai < a_end && ka < kb);
        out[q] = take_a ? ka : kb;
        if (take_a) {
            ++ai;
            ka = ai < a_end ? X[ms_pad(ai)] : ~0ull;
        } else {
            ++bi;
            kb = bi < b_end ? X[ms_pad(bi)] : ~0ull;
        }
    }
}

// The CTA-local part: 16 keys per thread (any assignment) -> X holds the 4096 keys ascending (padded layout).
// All kMsThreads threads must call it.
__device__ __forceinline__ void ms_sort_cta(uint64_t (&k)[16], uint64_t *X) {
    const int t = threadIdx.x;
    ms_sort16(k);
#pragma unroll
    for (int q = 0; q < 16; ++q) X[ms_pad(16 * t + q)] = k[q];
    __syncthreads();
#pragma unroll 1
    for (int w = 16; w < kMsChunk; w <<= 1) {  // runs of w keys are merged pairwise; thread t owns outputs [16 t, 16 t + 16)
        const int o = 16 * t;
        const int ps = o & ~(2 * w - 1);  // first key of the pair of runs
        const int d = o - ps;
        const int ai = ms_path_local(X, ps, w, ps + w, w, d);
        ms_merge16(X, ps + ai, ps + w, ps + w + (d - ai), ps + 2 * w, k);
        __syncthreads();  // every read of this level is done
#pragma unroll
        for (int q = 0; q < 16; ++q) X[ms_pad(o + q)] = k[q];
        __syncthreads();
    }
}

// key i of a run that starts at CTA `cta0` of the cluster (4096 keys per CTA, padded layout), through DSMEM
__device__ __forceinline__ uint64_t ms_run_key(uint32_t x_addr, int cta0, int i) {
    return ld_dsmem_u64(cluster_map(x_addr + 8u * (uint32_t)ms_pad(i & (kMsChunk - 1)), (uint32_t)(cta0 + (i >> 12))));
}

__device__ __forceinline__ int ms_path_remote(uint32_t x_addr, int ctaA, int na, int ctaB, int nb, int d) {
    int lo = max(0, d - nb), hi = min(d, na);
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (ms_run_key(x_addr, ctaA, mid) < ms_run_key(x_addr, ctaB, d - 1 - mid)) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

// window size of rank r this round: leftovers + un-fetched samples, capped by buffer_size (A0)
__device__ __forceinline__ int ms_window_size(int n_left, int fetch_pos, int n_arrived, int buffer_size) {
    long long avail = (long long)n_left + (long long)max(n_arrived - fetch_pos, 0);
    if (buffer_size > 0 && avail > buffer_size) avail = buffer_size;
    return (int)avail;
}

struct SortArgs {
    const int32_t *len;
    const int64_t *rank_ptr;
    int32_t *n_left, *fetch_pos, *emit_cur;
    const int32_t *left_ids;
    const int32_t *arrived;
    int buffer_size;
    uint64_t *keys_out;
    int32_t *S_out;
    RoundRec *rec;
    // first round of a run: the per-run state is cleared here instead of by a launch of its own
    int first;
    int64_t n_total;
    int32_t *emit_pos;
    int32_t *step_samples;
    int64_t step_cap;
};


// first round of a run: every sample un-emitted, step totals zero, lengths validated (len >= 1); the
// whole grid sweeps (me = this thread's index among nthreads)
__device__ __forceinline__ void ms_first_round_init(const SortArgs &A, int64_t me, int64_t nthreads) {
    int bad = 0;
    const int64_t bound = max(A.n_total, A.step_cap);
    for (int64_t i = me; i < bound; i += nthreads) {
        if (i < A.n_total) {
            A.emit_pos[i] = -1;
            if (A.len[i] < 1) bad = 1;
        }
        if (i < A.step_cap) A.step_samples[i] = 0;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) A.rec->bad_length = 1;
}

// this thread's 16 keys of the chunk [c0, c0 + cnt) of rank r's window (any assignment will do: coalesced)
__device__ __forceinline__ void ms_load_keys(const SortArgs &A, int64_t base, int nl, int fp, int c0, int cnt,
                                             uint64_t (&k)[16]) {
    const int t = threadIdx.x;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int e = q * kMsThreads + t;
        uint64_t key = ~0ull;  // padding sorts to the end
        if (e < cnt) {
            const int w = c0 + e;
            const int id = w < nl ? A.left_ids[base + w] : fp + (w - nl);
            const int l = A.len[base + id];
            key = ((uint64_t)(uint32_t)max(l, 0) << 32) | (uint32_t)id;
        }
        k[q] = key;
    }
}

}  // namespace odb
