// Device-side pieces of the window sort (A0 + A1), shared by the cluster sort kernel (odb_sort.cu) and the
// persistent round-loop kernel (odb_rounds.cu): a CTA merge-sorts 4096 64-bit keys in shared memory.
#pragma once

#include "odb_device.cuh"
#include "odb_internal.cuh"

namespace odb {

constexpr int kMsThreads = 1024;
constexpr int kMsItems = 4;                      // keys per thread: short serial merges, many threads to hide latency
constexpr int kMsChunk = kMsThreads * kMsItems;  // 4096 keys per CTA
static_assert(kMsChunk == kSortChunk, "one CTA sorts one chunk");
constexpr int kMsPadded = kMsChunk + kMsChunk / kMsItems;  // one spare key per thread run: conflict-free stores

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

// The sort's device functions are templates over ITEMS = keys per thread (a power of two): the persistent round loop
// and the round-parallel planner sort small windows with 4 keys per thread (short serial merges, many threads to hide
// latency: 6 us per 1024-key window against 18 us with 16), the cluster kernel sorts 4096-key chunks with fewer,
// longer thread runs (fewer merge-path searches and barriers per key; measured in profiles/r02_planning.md).
template <int ITEMS>
struct MsSort {
    static constexpr int kChunk = kMsChunk;                  // keys per CTA
    static constexpr int kThreads = kMsChunk / ITEMS;        // threads that hold a full chunk
    static constexpr int kPadded = kMsChunk + kMsChunk / ITEMS;  // one spare key per thread run: conflict-free stores

    static __device__ __forceinline__ int pad(int i) { return i + i / ITEMS; }

    // ascending sort of this thread's keys in registers: the bitonic network
    static __device__ __forceinline__ void sort_items(uint64_t (&k)[ITEMS]) {
#pragma unroll
        for (int kk = 2; kk <= ITEMS; kk <<= 1) {
#pragma unroll
            for (int j = kk >> 1; j > 0; j >>= 1) {
#pragma unroll
                for (int r = 0; r < ITEMS; ++r)
                    if ((r & j) == 0) ms_cmp_xchg(k[r], k[r | j], kk == ITEMS || (r & kk) == 0);
            }
        }
    }

    // keys taken from run a (na keys) among the first d outputs of merge(a, b); runs are in PADDED local shared memory
    static __device__ __forceinline__ int path_local(const uint64_t *X, int a0, int na, int b0, int nb, int d) {
        int lo = max(0, d - nb), hi = min(d, na);
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (X[pad(a0 + mid)] < X[pad(b0 + d - 1 - mid)]) lo = mid + 1;
            else hi = mid;
        }
        return lo;
    }

    // ITEMS outputs of merge(X[a.. a_end), X[b.. b_end)) starting at the split (ai, bi), into registers
    static __device__ __forceinline__ void merge_items(const uint64_t *X, int ai, int a_end, int bi, int b_end,
                                                       uint64_t (&out)[ITEMS]) {
        uint64_t ka = ai < a_end ? X[pad(ai)] : ~0ull;
        uint64_t kb = bi < b_end ? X[pad(bi)] : ~0ull;
#pragma unroll
        for (int q = 0; q < ITEMS; ++q) {
            // keys are unique (the id is part of the key), padding keys (~0) sort last: ties are irrelevant
            const bool take_a = (bi >= b_end) || (ai < a_end && ka < kb);
            out[q] = take_a ? ka : kb;
            if (q + 1 < ITEMS) {
                if (take_a) {
                    ++ai;
                    ka = ai < a_end ? X[pad(ai)] : ~0ull;
                } else {
                    ++bi;
                    kb = bi < b_end ? X[pad(bi)] : ~0ull;
                }
            }
        }
    }

    // Keys in play for a window of S keys: a power of two, at least one warp's worth, at most the chunk.
    static __device__ __forceinline__ int active_keys(int S) {
        int n = 32 * ITEMS;
        while (n < S) n <<= 1;
        return min(n, kMsChunk);
    }

    // The CTA-local part: the first n_keys / ITEMS threads hold ITEMS keys each (any assignment) -> X holds
    // the n_keys keys ascending (padded layout).  n_keys = active_keys(.).  All threads of the CTA must call it.
    static __device__ __forceinline__ void sort_cta(uint64_t (&k)[ITEMS], uint64_t *X, int n_keys) {
        const int o = ITEMS * (int)threadIdx.x;
        const bool active = o < n_keys;
        if (active) {
            sort_items(k);
#pragma unroll
            for (int q = 0; q < ITEMS; ++q) X[pad(o + q)] = k[q];
        }
        __syncthreads();
#pragma unroll 1
        for (int w = ITEMS; w < n_keys; w <<= 1) {  // runs of w keys are merged pairwise; a thread owns ITEMS outputs
            if (active) {
                const int ps = o & ~(2 * w - 1);  // first key of the pair of runs
                const int d = o - ps;
                const int ai = path_local(X, ps, w, ps + w, w, d);
                merge_items(X, ps + ai, ps + w, ps + w + (d - ai), ps + 2 * w, k);
            }
            // (while a pair of runs lies inside one warp's 32 * ITEMS keys, the warp's own barrier is enough)
            const bool in_warp = 2 * w <= 32 * ITEMS;
            if (in_warp) __syncwarp();
            else __syncthreads();  // every read of this level is done
            if (active) {
#pragma unroll
                for (int q = 0; q < ITEMS; ++q) X[pad(o + q)] = k[q];
            }
            if (in_warp && 4 * w <= 32 * ITEMS) __syncwarp();
            else __syncthreads();
        }
    }

    // key i of a run that starts at CTA `cta0` of the cluster (4096 keys per CTA, padded layout), through DSMEM
    static __device__ __forceinline__ uint64_t run_key(uint32_t x_addr, int cta0, int i) {
        return ld_dsmem_u64(cluster_map(x_addr + 8u * (uint32_t)pad(i & (kMsChunk - 1)), (uint32_t)(cta0 + (i >> 12))));
    }

    // Merge-path cut over DSMEM by ONE WARP: 32 probes per round split [lo, hi) into 33 parts (the predicate
    // "a[mid] < b[d - 1 - mid]" is true below the answer and false from it on), so runs of 32768 keys need three
    // rounds of two remote loads instead of fifteen dependent ones.  All 32 lanes must call it; all return the cut.
    static __device__ __forceinline__ int path_remote(uint32_t x_addr, int ctaA, int na, int ctaB, int nb, int d) {
        const int lane = threadIdx.x & 31;
        int lo = max(0, d - nb), hi = min(d, na);
        while (lo < hi) {  // warp-uniform
            const int mid = lo + (int)(((long long)(hi - lo) * (lane + 1)) / 33);  // in [lo, hi), non-decreasing in lane
            const bool below = run_key(x_addr, ctaA, mid) < run_key(x_addr, ctaB, d - 1 - mid);
            const int p = __popc(__ballot_sync(ODB_FULL_MASK, below));  // the probes below the answer are the first p lanes
            const int lo_n = __shfl_sync(ODB_FULL_MASK, mid, max(p - 1, 0)) + 1;
            const int hi_n = __shfl_sync(ODB_FULL_MASK, mid, min(p, 31));
            if (p > 0) lo = lo_n;
            if (p < 32) hi = hi_n;
        }
        return lo;
    }
};

// the 4-keys-per-thread instance under its round-1 names (k_rounds, k_spec_form)
__device__ __forceinline__ int ms_pad(int i) { return MsSort<kMsItems>::pad(i); }
__device__ __forceinline__ int ms_active_keys(int S) { return MsSort<kMsItems>::active_keys(S); }
__device__ __forceinline__ void ms_sort_cta(uint64_t (&k)[kMsItems], uint64_t *X, int n_keys) {
    MsSort<kMsItems>::sort_cta(k, X, n_keys);
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

// the keys of the chunk [c0, c0 + cnt) of rank r's window, ITEMS per thread on the first n_keys / ITEMS
// threads (any assignment will do: coalesced); positions beyond cnt are padding that sorts to the end
template <int ITEMS>
__device__ __forceinline__ void ms_load_keys_t(const SortArgs &A, int64_t base, int nl, int fp, int c0, int cnt, int n_keys,
                                               uint64_t (&k)[ITEMS]) {
    const int t = threadIdx.x, na = n_keys / ITEMS;
#pragma unroll
    for (int q = 0; q < ITEMS; ++q) {
        const int e = q * na + t;
        uint64_t key = ~0ull;
        if (t < na && e < cnt) {
            const int w = c0 + e;
            const int id = w < nl ? A.left_ids[base + w] : fp + (w - nl);
            const int l = A.len[base + id];
            key = ((uint64_t)(uint32_t)max(l, 0) << 32) | (uint32_t)id;
        }
        k[q] = key;
    }
}
__device__ __forceinline__ void ms_load_keys(const SortArgs &A, int64_t base, int nl, int fp, int c0, int cnt, int n_keys,
                                             uint64_t (&k)[kMsItems]) {
    ms_load_keys_t<kMsItems>(A, base, nl, fp, c0, cnt, n_keys, k);
}

}  // namespace odb
