// Planning kernels of the ODB hot path (rows A0..A9 of DESIGN.md): window fill + segmented sort,
// greedy successor, pointer-jumping list ranking, cross-rank reduction, split / overflow, step
// totals + quota cut, round commit, the whole round loop on the device (k_rounds: sequential, one CTA per rank;
// k_spec_form / k_spec_commit: every round that starts without leftovers at once; k_spec_T_world: the same over
// several processes), and the rank-major plan tables (whole plan or a step range).  sm_100a only.
//
// Paper: /root/reference/PAPER.md (P:<line>).  Section 2.2 P:32-36 and Eq. 1 (grouping), Eq. 3
// (target), Alg. 1 P:258-279 (split / overflow), P:28 (IDLE slots), Thm 2 P:48 + P:347 (quota).
#include <cstring>

#include "odb_internal.cuh"
#include "odb_device.cuh"
#include "odb_sort.cuh"

namespace odb {

// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t key_len(uint64_t k) { return (uint32_t)(k >> 32); }
__device__ __forceinline__ int32_t key_id(uint64_t k) { return (int32_t)(uint32_t)(k & 0xffffffffull); }

__device__ __forceinline__ int next_pow2(int n) {
    int p = 1;
    while (p < n) p <<= 1;
    return p;
}

// Bitonic sort of n2 (power of two) uint64 keys, ascending, by the whole CTA.  Works on shared or
// global memory (the CTA's own writes are visible to it after __syncthreads).
__device__ __forceinline__ void block_bitonic(uint64_t *k, int n2) {
    for (int kk = 2; kk <= n2; kk <<= 1) {
        for (int j = kk >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < (n2 >> 1); t += blockDim.x) {
                int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                int l = i | j;
                bool asc = (i & kk) == 0;
                uint64_t a = k[i], b = k[l];
                if ((a > b) == asc) {
                    k[i] = b;
                    k[l] = a;
                }
            }
            __syncthreads();
        }
    }
}

// window size of rank r this round: leftovers + un-fetched samples, capped by buffer_size (A0)
__device__ __forceinline__ int window_size(int n_left, int fetch_pos, int n_arrived, int buffer_size) {
    long long avail = (long long)n_left + (long long)max(n_arrived - fetch_pos, 0);
    if (buffer_size > 0 && avail > buffer_size) avail = buffer_size;
    return (int)avail;
}

// ---------------------------------------------------------------------------------------------
// start of a run: clear the per-rank state, mark every sample un-emitted, zero the step totals and
// validate the lengths (len >= 1) -- one launch.  rec was zeroed by the caller.
// ---------------------------------------------------------------------------------------------
__global__ void k_begin(const int32_t *__restrict__ len, int64_t n, int R, int32_t *__restrict__ n_left,
                        int32_t *__restrict__ fetch_pos, int32_t *__restrict__ emit_cur, int32_t *__restrict__ G,
                        int32_t *__restrict__ S, int32_t *__restrict__ emit_pos,
                        int32_t *__restrict__ step_samples, int64_t step_cap, RoundRec *rec) {
    int bad = 0;
    const int64_t bound = max(n, max((int64_t)R, step_cap));
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < bound; i += (int64_t)gridDim.x * blockDim.x) {
        if (i < R) {
            n_left[i] = 0;
            fetch_pos[i] = 0;
            emit_cur[i] = 0;
            G[i] = 0;
            S[i] = 0;
        }
        if (i < n) {
            emit_pos[i] = -1;
            if (len[i] < 1) bad = 1;
        }
        if (i < step_cap) step_samples[i] = 0;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) rec->bad_length = 1;
}

// ---------------------------------------------------------------------------------------------
// A0 + A1a: fill the window and sort chunks of kSortChunk keys in shared memory.
// key = (len << 32) | local id, so ascending key order is the composite order (len, id) (U1).
// grid = (chunks of the largest possible window, R)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kSortThreads)
k_chunk_sort(const int32_t *__restrict__ len, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ n_left,
             const int32_t *__restrict__ fetch_pos, const int32_t *__restrict__ left_ids,
             const int32_t *__restrict__ arrived, int buffer_size, uint64_t *__restrict__ keys_out,
             int32_t *__restrict__ S_out, RoundRec *rec) {
    __shared__ uint64_t sk[kSortChunk];
    const int r = blockIdx.y;
    const int64_t base = rank_ptr[r];
    const int n_r = (int)(rank_ptr[r + 1] - base);
    const int nl = n_left[r], fp = fetch_pos[r];
    // only the views the workers have delivered so far can be drained (App. C.1; odb_set_available)
    const int S = window_size(nl, fp, min(n_r, arrived[r]), buffer_size);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        S_out[r] = S;
        if (r == 0) rec->n_finished = 0;  // counted again by this round's commit
    }
    const int c0 = blockIdx.x * kSortChunk;
    if (c0 >= S) return;
    const int cnt = min(kSortChunk, S - c0);
    const int n2 = next_pow2(cnt);
    for (int i = threadIdx.x; i < n2; i += blockDim.x) {
        uint64_t key = ~0ull;
        if (i < cnt) {
            int w = c0 + i;
            int id = w < nl ? left_ids[base + w] : fp + (w - nl);
            int l = len[base + id];
            key = ((uint64_t)(uint32_t)max(l, 0) << 32) | (uint32_t)id;
        }
        sk[i] = key;
    }
    __syncthreads();
    block_bitonic(sk, n2);
    for (int i = threadIdx.x; i < cnt; i += blockDim.x) keys_out[base + c0 + i] = sk[i];
}

// A0 + A1a, register-blocked version for full-size chunks: the same bitonic network over 4096 keys,
// but 256 threads hold 16 keys each in registers.  Position i of the network lives
//   layout A: i = (warp << 9) | (lane << 4) | r   -- strides 1..8 are compare-exchanges inside a thread,
//             strides 16..256 are lane exchanges (shuffles);
//   layout B: i = (r << 8) | t                    -- strides 512..2048 are inside a thread;
// the two layouts are swapped through shared memory (padded by one key per 16: conflict-free on both
// sides) three times in the whole sort, instead of one shared-memory pass per network stage.
constexpr int kSortRegThreads = 256;
constexpr int kSortRegKeys = kSortChunk / kSortRegThreads;  // 16
static_assert(kSortChunk == 4096 && kSortRegKeys == 16, "layouts A / B below are written for 4096 keys, 16 per thread");

__device__ __forceinline__ void cmp_xchg(uint64_t &lo, uint64_t &hi, bool asc) {
    const bool sw = (lo > hi) == asc;
    const uint64_t a = sw ? hi : lo, b = sw ? lo : hi;
    lo = a;
    hi = b;
}
__device__ __forceinline__ int sort_pad(int i) { return i + (i >> 4); }

template <int J>  // layout A, stride J < 16
__device__ __forceinline__ void sort_reg_stage(uint64_t (&k)[16], int kk, int ibase) {
#pragma unroll
    for (int r = 0; r < 16; ++r)
        if ((r & J) == 0) cmp_xchg(k[r], k[r | J], ((ibase | r) & kk) == 0);
}
// layout A, stride j = 16 .. 256: the partner lives in lane ^ (j >> 4)
__device__ __forceinline__ void sort_shfl_stage(uint64_t (&k)[16], int j, int kk, int ibase, int lane) {
    const int m = j >> 4;
    const bool lower = (lane & m) == 0;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const uint64_t o = __shfl_xor_sync(ODB_FULL_MASK, k[r], m);
        const bool asc = ((ibase | r) & kk) == 0;
        const uint64_t mn = k[r] < o ? k[r] : o, mx = k[r] < o ? o : k[r];
        k[r] = (lower == asc) ? mn : mx;
    }
}
template <int JR>  // layout B, stride JR << 8
__device__ __forceinline__ void sort_regB_stage(uint64_t (&k)[16], int kk) {
#pragma unroll
    for (int r = 0; r < 16; ++r)
        if ((r & JR) == 0) cmp_xchg(k[r], k[r | JR], ((r << 8) & kk) == 0);
}

__global__ void __launch_bounds__(kSortRegThreads)
k_chunk_sort_reg(const int32_t *__restrict__ len, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ n_left,
                 const int32_t *__restrict__ fetch_pos, const int32_t *__restrict__ left_ids,
                 const int32_t *__restrict__ arrived, int buffer_size, uint64_t *__restrict__ keys_out,
                 int32_t *__restrict__ S_out, RoundRec *rec) {
    __shared__ uint64_t sk[kSortChunk + kSortChunk / 16];
    const int r_ = blockIdx.y;
    const int64_t base = rank_ptr[r_];
    const int n_r = (int)(rank_ptr[r_ + 1] - base);
    const int nl = n_left[r_], fp = fetch_pos[r_];
    const int S = window_size(nl, fp, min(n_r, arrived[r_]), buffer_size);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        S_out[r_] = S;
        if (r_ == 0) rec->n_finished = 0;
    }
    const int c0 = blockIdx.x * kSortChunk;
    if (c0 >= S) return;
    const int cnt = min(kSortChunk, S - c0);
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    uint64_t k[16];
    // any assignment of window elements to network positions will do: read them coalesced
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int e = r * kSortRegThreads + t;
        uint64_t key = ~0ull;  // padding sorts to the end
        if (e < cnt) {
            const int w = c0 + e;
            const int id = w < nl ? left_ids[base + w] : fp + (w - nl);
            const int l = len[base + id];
            key = ((uint64_t)(uint32_t)max(l, 0) << 32) | (uint32_t)id;
        }
        k[r] = key;
    }
    const int ibase = (warp << 9) | (lane << 4);
#pragma unroll 1
    for (int kk = 2; kk <= kSortChunk; kk <<= 1) {
        if (kk >= 1024) {  // strides 512 .. kk/2 in layout B
#pragma unroll
            for (int r = 0; r < 16; ++r) sk[sort_pad(ibase | r)] = k[r];
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 16; ++r) k[r] = sk[sort_pad((r << 8) | t)];
            if (kk >= 4096) sort_regB_stage<8>(k, kk);
            if (kk >= 2048) sort_regB_stage<4>(k, kk);
            sort_regB_stage<2>(k, kk);
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 16; ++r) sk[sort_pad((r << 8) | t)] = k[r];
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 16; ++r) k[r] = sk[sort_pad(ibase | r)];
            __syncthreads();
        }
#pragma unroll 1
        for (int j = min(kk >> 1, 256); j >= 16; j >>= 1) sort_shfl_stage(k, j, kk, ibase, lane);
        if (kk >= 16) sort_reg_stage<8>(k, kk, ibase);
        if (kk >= 8) sort_reg_stage<4>(k, kk, ibase);
        if (kk >= 4) sort_reg_stage<2>(k, kk, ibase);
        sort_reg_stage<1>(k, kk, ibase);
    }
    // sorted in layout A; go through shared memory once more for coalesced stores
#pragma unroll
    for (int r = 0; r < 16; ++r) sk[sort_pad(ibase | r)] = k[r];
    __syncthreads();
    for (int i = t; i < cnt; i += kSortRegThreads) keys_out[base + c0 + i] = sk[sort_pad(i)];
}

// A1b: one merge pass; sorted runs of width w are merged pairwise (merge path).  A CTA produces
// kMergeTile consecutive output keys of one pair of runs: two threads find where the tile's first and
// last diagonal cut the runs (binary search in global memory, ~log2 w dependent loads, once per CTA),
// the two input pieces are staged in shared memory with coalesced loads, every thread finds its own
// diagonal there and merges kMergeItems keys sequentially, and the tile leaves through shared memory
// with coalesced stores.  Keys are unique, so ties never arise.  (The earlier version let every key
// binary-search its position in the sibling run: 13+ dependent L2 loads per key, 18.3 us per pass on
// the default workload, bound by the number of L2 requests.)
constexpr int kMergeItems = 8;
constexpr int kMergeTile = kMergeThreads * kMergeItems;  // 2048 outputs per CTA; divides 2 * kSortChunk
static_assert((2 * kSortChunk) % kMergeTile == 0, "a tile must not straddle two pairs of runs");

// number of keys taken from a[0, na) among the first d outputs of merge(a, b)
__device__ __forceinline__ int merge_path(const uint64_t *a, int na, const uint64_t *b, int nb, int d) {
    int lo = max(0, d - nb), hi = min(d, na);
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (a[mid] < b[d - 1 - mid]) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(kMergeThreads)
k_merge_pass(const uint64_t *__restrict__ src, uint64_t *__restrict__ dst, const int64_t *__restrict__ rank_ptr,
             const int32_t *__restrict__ S_arr, int w) {
    __shared__ uint64_t s_in[kMergeTile];
    __shared__ uint64_t s_out[kMergeTile];
    __shared__ int s_cut[2];
    const int r = blockIdx.y;
    const int S = S_arr[r];
    const long long o0 = (long long)blockIdx.x * kMergeTile;  // first output position of the tile
    if (o0 >= S) return;
    const uint64_t *s = src + rank_ptr[r];
    const long long ps = (o0 / (2ll * w)) * (2ll * w);         // first position of the pair of runs
    const int na = (int)(min((long long)S, ps + w) - ps);
    const int nb = (int)(min((long long)S, ps + 2ll * w) - (ps + na));
    const uint64_t *A = s + ps, *B = s + ps + na;
    const int d0 = (int)(o0 - ps), d1 = min(d0 + kMergeTile, na + nb);
    if (threadIdx.x < 2) s_cut[threadIdx.x] = merge_path(A, na, B, nb, threadIdx.x ? d1 : d0);
    __syncthreads();
    const int a0 = s_cut[0], a1 = s_cut[1];
    const int b0 = d0 - a0, b1 = d1 - a1;
    const int la = a1 - a0, lb = b1 - b0, total = la + lb;
    for (int i = threadIdx.x; i < total; i += blockDim.x) s_in[i] = i < la ? A[a0 + i] : B[b0 + (i - la)];
    __syncthreads();
    const uint64_t *sa = s_in, *sb = s_in + la;
    const int ld = threadIdx.x * kMergeItems;
    if (ld < total) {
        int ai = merge_path(sa, la, sb, lb, ld);
        int bi = ld - ai;
#pragma unroll
        for (int k = 0; k < kMergeItems; ++k) {
            if (ld + k < total) {
                const bool take_a = bi >= lb || (ai < la && sa[ai] < sb[bi]);
                s_out[ld + k] = take_a ? sa[ai] : sb[bi];
                ai += take_a ? 1 : 0;
                bi += take_a ? 0 : 1;
            }
        }
    }
    __syncthreads();
    uint64_t *out = dst + rank_ptr[r] + o0;
    for (int i = threadIdx.x; i < total; i += blockDim.x) out[i] = s_out[i];
}

// ---------------------------------------------------------------------------------------------
// A2 + A3: successor array, pointer-jumping reachability from the head, candidate group starts.
// One CTA per rank.  Chase coordinate x in [0, S]:
//   THRESHOLD: x = position in the longest->shortest visit order; J[0] = 1 (t starts at 1),
//              J[x] = min(S, x + B(len(v[x-1]))), B from Eq. 1 (the group that starts at x closes
//              after B(l) samples, l = the last sample of the previous group).
//   MAXFIT:    x = ascending position; J[x] = largest e <= S with (e - x) * slen[e-1] <= L, >= x+1.
// Round p marks next^(k + 2^p)(0) for every marked next^k(0) and squares the jump array, so after
// ceil(log2 G) + 1 rounds exactly the orbit of 0 is marked.  Output: ascending start positions
// gpos[0..G] (gpos[G] = S) and G_r.  A THRESHOLD mark at chase x > 0 is the ascending start S - x.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int successor(const uint64_t *k, int x, int S, uint32_t budget, int rule) {
    if (x == S) return S;
    if (rule == ODB_RULE_THRESHOLD) {
        if (x == 0) return 1;
        const uint32_t l = key_len(k[S - x]);  // v[x-1] = ascending position S-1-(x-1)
        uint32_t q = budget / (l > 0u ? l : 1u);  // Eq. 1 floor; budget < 2^31
        if (q < 1u) q = 1u;
        const uint32_t jj = (uint32_t)x + q;  // < 2^32
        return (int)(jj < (uint32_t)S ? jj : (uint32_t)S);
    }
    int lo = x + 1, hi = S;  // the singleton [x, x+1) is always accepted (U10)
    while (lo < hi) {
        const int m = (lo + hi + 1) >> 1;
        if ((long long)(m - x) * (long long)key_len(k[m - 1]) <= (long long)budget) lo = m;
        else hi = m - 1;
    }
    return lo;
}

// Shared-memory version (windows of up to kFormSmemMaxS samples): the jump arrays are uint16 pairs
// of buffers and the marks a bit set, all in the CTA's shared memory, so a round costs shared-memory
// latency instead of L2 round trips.
__global__ void __launch_bounds__(kRankThreads)
k_form_groups_smem(const uint64_t *__restrict__ keys, const int64_t *__restrict__ rank_ptr,
                   const int32_t *__restrict__ S_arr, uint32_t budget, int rule, int32_t *__restrict__ gpos,
                   int32_t *__restrict__ G_out) {
    extern __shared__ __align__(16) unsigned char fg_smem[];
    __shared__ int s_scan[34];
    const int r = blockIdx.x;
    const int S = S_arr[r];
    if (S == 0) {
        if (threadIdx.x == 0) G_out[r] = 0;
        return;
    }
    const int64_t base = rank_ptr[r];
    const uint64_t *k = keys + base;
    const int n1 = S + 1;
    const int n1p = (n1 + 7) & ~7;
    const int words = (n1 + 31) >> 5;
    uint16_t *cur = reinterpret_cast<uint16_t *>(fg_smem);
    uint16_t *nxt = cur + n1p;
    uint32_t *mk = reinterpret_cast<uint32_t *>(nxt + n1p);
    for (int w = threadIdx.x; w < words; w += blockDim.x) mk[w] = (w == 0) ? 1u : 0u;  // x = 0 is a start
    // entries (S, n1p) are padding: they jump to S like S itself, so pairs can be processed blindly
    for (int x = threadIdx.x; x < n1p; x += blockDim.x)
        cur[x] = (uint16_t)(x <= S ? successor(k, x, S, budget, rule) : S);
    __syncthreads();
    while (true) {
        int changed = 0;
        // two positions per thread and iteration: one 32-bit load / store for the pair's jump entries
        const uint32_t *cur2 = reinterpret_cast<const uint32_t *>(cur);
        uint32_t *nxt2 = reinterpret_cast<uint32_t *>(nxt);
        for (int p = threadIdx.x; 2 * p <= S; p += blockDim.x) {
            const uint32_t v = cur2[p];
            const int j0 = (int)(v & 0xffffu), j1 = (int)(v >> 16);
            nxt2[p] = (uint32_t)cur[j0] | ((uint32_t)cur[j1] << 16);  // cur[S] == S
            const uint32_t mw = mk[p >> 4] >> ((2 * p) & 31);          // marks of x = 2p (bit 0) and 2p + 1 (bit 1)
            if ((mw & 1u) && j0 < S && !((mk[j0 >> 5] >> (j0 & 31)) & 1u)) {
                atomicOr(&mk[j0 >> 5], 1u << (j0 & 31));
                changed = 1;
            }
            if ((mw & 2u) && j1 < S && !((mk[j1 >> 5] >> (j1 & 31)) & 1u)) {
                atomicOr(&mk[j1 >> 5], 1u << (j1 & 31));
                changed = 1;
            }
        }
        if (!__syncthreads_or(changed)) break;
        uint16_t *t = cur;
        cur = nxt;
        nxt = t;
    }
    // marks live on x in [0, S); G = their number
    int part = 0;
    for (int w = threadIdx.x; w < words; w += blockDim.x) part += __popc(mk[w]);
    int G;
    (void)block_excl_scan<int>(part, s_scan, G);
    int32_t *gp = gpos + base + r;
    int carry = 0;
    for (int w0 = 0; w0 < words; w0 += blockDim.x) {
        const int w = w0 + threadIdx.x;
        uint32_t bits = w < words ? mk[w] : 0u;
        int tot;
        int i = block_excl_scan<int>(__popc(bits), s_scan, tot) + carry;
        while (bits) {
            const int x = (w << 5) + __ffs(bits) - 1;
            bits &= bits - 1;
            if (rule == ODB_RULE_THRESHOLD) gp[G - i] = S - x;  // i-th mark (ascending x) -> start S - x
            else gp[i] = x;
            ++i;
        }
        carry += tot;
    }
    if (threadIdx.x == 0) {
        if (rule == ODB_RULE_THRESHOLD) gp[0] = 0;
        else gp[G] = S;
        G_out[r] = G;
    }
}

// Hierarchical version (windows of up to 32768 samples; the default): the successor is strictly increasing
// (next[x] > x), so the orbit of 0 can be found with JUMP-OUT TABLES instead of pointer doubling over the
// whole window.  Positions are cut into blocks of 32 and superblocks of 1024:
//   out1[x] = the first element of x's chain that leaves x's block      (backward DP inside each block:
//             one thread per block, 32 dependent steps);
//   out2[x] = the first element of x's chain that leaves x's superblock (one warp per superblock walks its
//             32 blocks from the last to the first, a lane per position: out2[x] = out1[x] if that is
//             outside, else out2[out1[x]], already known);
// then the orbit is expanded top-down: thread 0 chases out2 from 0 (at most 32 steps) and records where
// the orbit enters each superblock; a thread per superblock chases out1 from there and records where it
// enters each block; a thread per block chases next and builds the block's 32-bit mark word in a register.
// About 5 x 32 dependent shared-memory steps in all, and O(S) work per phase whatever the group sizes --
// against ceil(log2 G) + 1 passes over the whole window for pointer doubling (51 us -> see profiles/).
// Arrays are uint16 (S <= 32768) with one spare entry per 32, so a thread per block walks without bank conflicts.
__device__ __forceinline__ int fg_pad(int i) { return i + (i >> 5); }

// (a device function: the persistent round-loop kernel calls it too, on keys it has just written itself)
__device__ __forceinline__ int
form_hier_body(const uint64_t *k, int S, uint32_t budget, int rule, int32_t *gp, unsigned char *fh_smem, int *s_scan,
               uint16_t *s_e2) {
    const int np = fg_pad(S) + 2;            // entries per array (even, so the arrays stay 4-byte aligned)
    const int npe = (np + 1) & ~1;
    const int nb1 = (S + 31) >> 5, nb2 = (S + 1023) >> 10;
    uint16_t *nxt = reinterpret_cast<uint16_t *>(fh_smem);
    uint16_t *out1 = nxt + npe;
    uint16_t *out2 = out1 + npe;
    uint16_t *e1 = out2 + npe;                                  // nb1 entries (padded to even)
    uint32_t *mk = reinterpret_cast<uint32_t *>(e1 + ((nb1 + 1) & ~1));  // nb1 words
    constexpr uint16_t kNone = 0xFFFFu;
    if (rule == ODB_RULE_THRESHOLD) {
        // J[x] = min(S, x + B(len(v[x-1]))), B from Eq. 1; eight independent (coalesced) key loads in flight per
        // thread: a load per iteration would serialise on the L2 latency
        for (int x0 = threadIdx.x; x0 < S; x0 += 8 * blockDim.x) {
            uint32_t l[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int x = x0 + u * blockDim.x;
                l[u] = (x > 0 && x < S) ? key_len(k[S - x]) : 1u;
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int x = x0 + u * blockDim.x;
                if (x < S) {
                    uint32_t q = budget / (l[u] > 0u ? l[u] : 1u);  // Eq. 1 floor; budget < 2^31
                    if (q < 1u) q = 1u;
                    const uint32_t jj = (uint32_t)x + q;
                    nxt[fg_pad(x)] = (uint16_t)(x == 0 ? 1u : (jj < (uint32_t)S ? jj : (uint32_t)S));
                }
            }
        }
    } else {
        for (int x = threadIdx.x; x < S; x += blockDim.x) nxt[fg_pad(x)] = (uint16_t)successor(k, x, S, budget, rule);
    }
    for (int b = threadIdx.x; b < nb1; b += blockDim.x) e1[b] = kNone;
    if (threadIdx.x < 32) s_e2[threadIdx.x] = kNone;
    __syncthreads();
    // out1: one thread per block, from the block's last position down
    for (int b = threadIdx.x; b < nb1; b += blockDim.x) {
        const int lo = b << 5, end = min(S, lo + 32);
        for (int i = end - 1; i >= lo; --i) {
            const int j = nxt[fg_pad(i)];
            out1[fg_pad(i)] = (uint16_t)(j >= end ? j : out1[fg_pad(j)]);
        }
    }
    __syncthreads();
    // out2: one warp per superblock, its blocks from the last to the first, a lane per position
    // (a window of one superblock needs none: the orbit enters it at 0)
    if (nb2 > 1) {
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
        for (int sb = w; sb < nb2; sb += nw) {
            const int slo = sb << 10, send = min(S, slo + 1024);
            for (int blk = ((send - 1) >> 5); blk >= (slo >> 5); --blk) {
                const int i = (blk << 5) + lane;
                if (i < send) {
                    const int j = out1[fg_pad(i)];
                    out2[fg_pad(i)] = (uint16_t)(j >= send ? j : out2[fg_pad(j)]);
                }
                __syncwarp();
            }
        }
    }
    __syncthreads();
    // top-down: where the orbit of 0 enters each superblock, each block, and its marks inside each block
    if (threadIdx.x == 0) {
        int x = 0;
        if (nb2 == 1) s_e2[0] = 0;
        else
            while (x < S) {
                s_e2[x >> 10] = (uint16_t)x;
                x = out2[fg_pad(x)];
            }
    }
    __syncthreads();
    if (threadIdx.x < nb2 && s_e2[threadIdx.x] != kNone) {
        const int send = min(S, ((int)threadIdx.x + 1) << 10);
        int x = s_e2[threadIdx.x];
        while (x < send) {
            e1[x >> 5] = (uint16_t)x;
            x = out1[fg_pad(x)];
        }
    }
    __syncthreads();
    int part = 0;
    for (int b = threadIdx.x; b < nb1; b += blockDim.x) {
        uint32_t word = 0u;
        if (e1[b] != kNone) {
            const int end = min(S, (b + 1) << 5);
            int x = e1[b];
            while (x < end) {
                word |= 1u << (x & 31);
                x = nxt[fg_pad(x)];
            }
        }
        mk[b] = word;
        part += __popc(word);
    }
    // marks live on chase coordinates x in [0, S); G = their number
    int G;
    (void)block_excl_scan<int>(part, s_scan, G);  // (its barriers also publish mk)
    int carry = 0;
    for (int w0 = 0; w0 < nb1; w0 += blockDim.x) {
        const int w = w0 + threadIdx.x;
        uint32_t bits = w < nb1 ? mk[w] : 0u;
        int tot;
        int i = block_excl_scan<int>(__popc(bits), s_scan, tot) + carry;
        while (bits) {
            const int x = (w << 5) + __ffs(bits) - 1;
            bits &= bits - 1;
            if (rule == ODB_RULE_THRESHOLD) gp[G - i] = S - x;  // i-th mark (ascending x) -> start S - x
            else gp[i] = x;
            ++i;
        }
        carry += tot;
    }
    if (threadIdx.x == 0) {
        if (rule == ODB_RULE_THRESHOLD) gp[0] = 0;
        else gp[G] = S;
    }
    return G;
}

__global__ void __launch_bounds__(kRankThreads)
k_form_groups_hier(const uint64_t *__restrict__ keys, const int64_t *__restrict__ rank_ptr,
                   const int32_t *__restrict__ S_arr, uint32_t budget, int rule, int32_t *__restrict__ gpos,
                   int32_t *__restrict__ G_out) {
    extern __shared__ __align__(16) unsigned char fh_smem[];
    __shared__ int s_scan[34];
    __shared__ uint16_t s_e2[32];
    const int r = blockIdx.x;
    const int S = S_arr[r];
    if (S == 0) {
        if (threadIdx.x == 0) G_out[r] = 0;
        return;
    }
    const int64_t base = rank_ptr[r];
    const int G = form_hier_body(keys + base, S, budget, rule, gpos + base + r, fh_smem, s_scan, s_e2);
    if (threadIdx.x == 0) G_out[r] = G;
}

// Global-memory version for windows that do not fit the shared-memory one.
__global__ void __launch_bounds__(kRankThreads)
k_form_groups(const uint64_t *__restrict__ keys, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ S_arr,
              uint32_t budget, int rule, int32_t *jA, int32_t *jB, uint8_t *mark, int32_t *__restrict__ gpos,
              int32_t *__restrict__ G_out) {
    __shared__ int s_scan[34];
    const int r = blockIdx.x;
    const int S = S_arr[r];
    if (S == 0) {
        if (threadIdx.x == 0) G_out[r] = 0;
        return;
    }
    const int64_t base = rank_ptr[r];
    const int64_t jb = base + r;  // regions of S+1 entries
    const uint64_t *k = keys + base;
    int32_t *cur = jA + jb, *nxt = jB + jb;
    uint8_t *mk = mark + jb;
    for (int x = threadIdx.x; x <= S; x += blockDim.x) {
        cur[x] = successor(k, x, S, budget, rule);
        mk[x] = (x == 0) ? 1 : 0;
    }
    __syncthreads();
    while (true) {
        int changed = 0;
        for (int x = threadIdx.x; x <= S; x += blockDim.x) {
            int j = cur[x];
            nxt[x] = cur[j];  // cur[S] == S
            if (x < S && mk[x] && j < S && !mk[j]) {
                mk[j] = 1;
                changed = 1;
            }
        }
        if (!__syncthreads_or(changed)) break;
        int32_t *t = cur;
        cur = nxt;
        nxt = t;
    }
    int32_t *gp = gpos + jb;
    int G = block_compact(
        S, s_scan, [&](int a) { return (rule == ODB_RULE_THRESHOLD) ? (a == 0 || mk[S - a] != 0) : (mk[a] != 0); },
        [&](int a, int kidx) { gp[kidx] = a; });
    if (threadIdx.x == 0) {
        gp[G] = S;
        G_out[r] = G;
    }
}

// ---------------------------------------------------------------------------------------------
// A4 + A5 + A6: T_grp (Eq. 3), split, overflow.  Output per rank: aligned groups in emit order as
// (agpos[k], agcnt[k]) over the sorted window, k < T.  Adds the counts into step_samples (A8a).
//
// Split closed form: Alg. 1's backward scan pops the last row of the rightmost
// multi-sample group until G_r = T, i.e. it turns the d = T - G_r rightmost NON-START positions of
// the sorted window into starts.  With ns(j) = (S - gpos[j]) - (G_r - j) = non-start positions in
// groups j.., group j gives up k_j = min(d, ns(j)) - min(d, ns(j+1)) rows, and its head moves to
// list index h_j = j + d - min(d, ns(j)); its k_j singletons follow it.  No scan needed.
//
// Overflow: sort groups by (count desc, index asc), keep the first T (shared memory when G_r fits).
// ---------------------------------------------------------------------------------------------
// One rank's alignment to T (A5 / A6): aligned groups in emit order as (ap[k], ac[k]) over the sorted window,
// ag[k] = list index of the head of the candidate group slot k was cut from; counts added into
// step_tot[k] (= step_samples + step_base; integer atomics).  A device function: k_align and the persistent
// round-loop kernel call it.  `ok` = scratch for the overflow sort (next_pow2(Gr) keys).
__device__ __forceinline__ void align_body(int S, int Gr, int T, const int32_t *gp, int32_t *ap, int32_t *ac, int32_t *ag,
                                           uint64_t *ok, int32_t *step_tot) {
    if (Gr <= T) {
        const int d = T - Gr;
        const int lane = threadIdx.x & 31;
        for (int j0 = (threadIdx.x >> 5) << 5; j0 < Gr; j0 += blockDim.x) {  // warp-uniform trip count
            const int j = j0 + lane;
            int p = 0, pn = 0, kj = 0, h = 0;
            if (j < Gr) {
                p = gp[j];
                pn = gp[j + 1];
                const int conv_from = min(d, (S - p) - (Gr - j));
                const int conv_after = min(d, (S - pn) - (Gr - 1 - j));
                kj = conv_from - conv_after;
                h = j + d - conv_from;
                const int c = pn - p - kj;
                ap[h] = p;
                ac[h] = c;
                ag[h] = h;
                atomicAdd(&step_tot[h], c);
            }
            uint32_t sp = __ballot_sync(ODB_FULL_MASK, kj > 0);
            while (sp) {  // expand the singletons of the (few) groups that split
                const int src = __ffs(sp) - 1;
                sp &= sp - 1;
                const int kk = __shfl_sync(ODB_FULL_MASK, kj, src);
                const int hh = __shfl_sync(ODB_FULL_MASK, h, src);
                const int pe = __shfl_sync(ODB_FULL_MASK, pn, src);
                for (int i = lane; i < kk; i += 32) {
                    ap[hh + 1 + i] = pe - kk + i;
                    ac[hh + 1 + i] = 1;
                    ag[hh + 1 + i] = hh;  // cut from the candidate group whose head sits at hh
                    atomicAdd(&step_tot[hh + 1 + i], 1);
                }
            }
        }
        if (threadIdx.x == 0) ap[T] = S;
    } else {
        const int n2 = next_pow2(Gr);
        for (int j = threadIdx.x; j < n2; j += blockDim.x) {
            uint64_t key = ~0ull;
            if (j < Gr) key = ((uint64_t)(uint32_t)(S - (gp[j + 1] - gp[j])) << 32) | (uint32_t)j;
            ok[j] = key;
        }
        __syncthreads();
        block_bitonic(ok, n2);
        for (int k = threadIdx.x; k < T; k += blockDim.x) {
            int j = key_id(ok[k]);
            int p = gp[j], c = gp[j + 1] - p;
            ap[k] = p;
            ac[k] = c;
            ag[k] = k;
            atomicAdd(&step_tot[k], c);
        }
    }
}

// Eq. 3 from the reduced status of all ranks: T = max(min(max_A G, C+min, S+min), 1); 0 when A is empty
__device__ __forceinline__ int target_groups(int maxG, int minS, int slot_capacity) {
    int T = maxG;
    if (slot_capacity > 0 && T > slot_capacity) T = slot_capacity;  // C+min (same C on every rank)
    if (T > minS) T = minS;                                         // S+min
    if (T < 1) T = 1;
    if (maxG == 0) T = 0;  // A is empty: a skip round, nothing is emitted (Lemma 2)
    return T;
}

__global__ void __launch_bounds__(kRankThreads)
k_align(const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ S_arr, const int32_t *__restrict__ G_arr, int R,
        const int32_t *__restrict__ gs_world, int world_ranks, int join_mode, int slot_capacity, const int32_t *__restrict__ gpos, int32_t *__restrict__ agpos, int32_t *__restrict__ agcnt,
        int32_t *__restrict__ agorg, uint64_t *ovf, int32_t *step_samples, int step_base,
        const int32_t *__restrict__ emit_cur, int32_t *__restrict__ emit_snap, RoundRec *rec) {
    extern __shared__ __align__(16) unsigned char al_smem[];
    __shared__ int s_maxG, s_minS, s_nfin;
    const int r = blockIdx.x;
    if (threadIdx.x == 0) {
        s_maxG = 0;
        s_minS = 0x7fffffff;
        s_nfin = 0;
    }
    __syncthreads();
    // the reduction runs over every rank of the job: the local tables, or -- distributed mode -- the
    // all_gathered (G, S) pairs of all world_ranks ranks (the paper's per-round all_gather)
    const int nq = gs_world ? world_ranks : R;
    for (int q = threadIdx.x; q < nq; q += blockDim.x) {
        const int g = gs_world ? gs_world[2 * q] : G_arr[q];
        const int sq = gs_world ? gs_world[2 * q + 1] : S_arr[q];
        if (g > 0) {  // active set A = {r : G_r > 0}
            atomicMax(&s_maxG, g);
            if (sq > 0) atomicMin(&s_minS, sq);
        }
        if (sq < 0) atomicAdd(&s_nfin, 1);  // status -1 "finished", encoded by k_pack_summary
    }
    __syncthreads();
    if (gs_world) {
        // termination predicates on the status every process holds identically (Thm 3 proof P:341)
        const bool done = join_mode ? (s_nfin == world_ranks) : (s_nfin > 0);
        if (done) {
            if (r == 0 && threadIdx.x == 0) {
                rec->T = 0;
                rec->done = 1;
            }
            return;
        }
    }
    const int T = target_groups(s_maxG, s_minS, slot_capacity);
    if (r == 0 && threadIdx.x == 0) rec->T = T;
    const int Gr = G_arr[r];
    if (Gr == 0) return;  // finished rank: IDLE slots are written by the commit kernel
    // k_commit runs several CTAs per rank and one of them advances emit_cur: they all read this snapshot
    if (threadIdx.x == 0) emit_snap[r] = emit_cur[r];
    const int S = S_arr[r];
    const int64_t base = rank_ptr[r];
    const int64_t jb = base + r;
    uint64_t *ok = (next_pow2(Gr) <= kAlignSmemKeys) ? reinterpret_cast<uint64_t *>(al_smem) : ovf + 2 * base;
    align_body(S, Gr, T, gpos + jb, agpos + jb, agcnt + jb, agorg + jb, ok, step_samples + step_base);
}

// ---------------------------------------------------------------------------------------------
// A7 + A8a: commit the round.  Finds the quota cut k* (non-join), writes the step-major staging
// tables, appends the emitted ids to the rank's emit region (recording every sample's emit
// position), compacts the leftovers, advances the rank state and counts the ranks that will be
// finished next round.
// ---------------------------------------------------------------------------------------------
// one rank's slices of the per-round scratch: global memory (per-round kernels) or shared memory (k_rounds)
struct RankView {
    const uint64_t *k;                 // the sorted window
    const int32_t *ap, *ac, *ag;       // aligned groups: start position, count, origin
    int32_t *ao;                       // their emit offsets (slow path)
    uint8_t *pf;                       // "emitted" flags over window positions (slow path)
    int S, Gr, cur, n_r;               // window size, candidate groups, emit cursor before this round, stream length
    int64_t base;                      // first global sample of the rank
    int32_t *n_left, *fetch_pos, *emit_cur;  // the rank's state words
};

__device__ __forceinline__ void
commit_body(const int r, const int R, const RankView V, const int32_t *step_samples, int step_base, int round, int join_mode,
            long long quota, long long emitted_before, int32_t *st_count, int32_t *st_width, int32_t *st_real,
            int32_t *st_round, int32_t *st_origin, int32_t *emit_ids, int32_t *emit_pos, int32_t *left_ids, RoundRec *rec,
            bool own_rec, int part, int nparts) {

    __shared__ int s_scan[34];
    __shared__ long long s_scan64[34];
    __shared__ int s_found;
    // nparts CTAs per rank share the fast path below; everything that needs a rank-wide scan, and all
    // state updates, is done by part 0 alone
    if (rec->done) {  // distributed mode: this round was the terminal check
        if (part != 0) return;
        if (r == 0 && threadIdx.x == 0) {
            rec->T_emit = 0;
            rec->quota_hit = 0;
            rec->emitted_round = 0;
        }
        return;
    }
    const int T = rec->T;
    int T_emit = T, quota_hit = 0;
    if (!join_mode && quota > 0) {
        if (threadIdx.x == 0) s_found = 0x7fffffff;
        __syncthreads();
        long long carry = 0;
        for (int b0 = 0; b0 < T; b0 += blockDim.x) {
            int k = b0 + threadIdx.x;
            long long v = (k < T) ? (long long)__ldcg(&step_samples[step_base + k]) : 0ll;
            long long tot;
            long long ex = block_excl_scan<long long>(v, s_scan64, tot);
            if (k < T && emitted_before + carry + ex + v >= quota) atomicMin(&s_found, k);
            __syncthreads();
            if (s_found != 0x7fffffff) break;
            carry += tot;
        }
        if (s_found != 0x7fffffff) {
            T_emit = s_found + 1;
            quota_hit = 1;
        }
        __syncthreads();
    }
    if ((r == 0 || own_rec) && part == 0) {  // round totals for the host (or for this CTA, in the persistent round loop)
        long long acc = 0;
        for (int k = threadIdx.x; k < T_emit; k += blockDim.x) acc += __ldcg(&step_samples[step_base + k]);
        long long tot;
        (void)block_excl_scan<long long>(acc, s_scan64, tot);
        if (threadIdx.x == 0) {
            rec->T_emit = T_emit;
            rec->quota_hit = quota_hit;
            rec->emitted_round = tot;
        }
    }
    const int Gr = V.Gr, S = V.S, n_r = V.n_r;
    const int64_t base = V.base;
    if (Gr == 0) {  // finished rank: IDLE slots (U14)
        if (part != 0) return;
        for (int k = threadIdx.x; k < T_emit; k += blockDim.x) {
            int64_t idx = (int64_t)(step_base + k) * R + r;
            st_count[idx] = 0;
            st_width[idx] = 0;
            st_real[idx] = 0;
            st_round[idx] = round;
            st_origin[idx] = step_base + k;
        }
        // finished (nothing buffered, nothing pending) or merely waiting for the workers (status 0)?
        if (threadIdx.x == 0 && *V.n_left == 0 && *V.fetch_pos >= n_r) atomicAdd(&rec->n_finished, 1);
        return;
    }
    const uint64_t *k_ = V.k;
    const int32_t *ap = V.ap, *ac = V.ac;
    int32_t *ao = V.ao;
    uint8_t *pf = V.pf;
    const int cur = V.cur;  // emit_cur[r] as k_align saw it (part 0 advances emit_cur below)
    // every sample of the window is emitted unless groups were dropped (overflow) or cut (quota)
    const bool all_emitted = (Gr <= T) && (T_emit == T);
    int emitted_r;
    if (all_emitted) {
        // Fast path (no overflow, no quota cut): the aligned groups are consecutive runs of the sorted
        // window in order, so the emit order IS the sorted order -- one coalesced pass over the samples,
        // then one thread per group for the tables (short groups sum their lengths there; long ones are
        // summed by a warp each).
        const int tid = part * blockDim.x + threadIdx.x, nth = nparts * blockDim.x;
#pragma unroll 4
        for (int a = tid; a < S; a += nth) {
            const int id = key_id(k_[a]);
            emit_ids[base + cur + a] = id;
            emit_pos[base + id] = cur + a;
        }
        for (int k = tid; k < T_emit; k += nth) {
            const int p = ap[k], c = ac[k];
            const int64_t idx = (int64_t)(step_base + k) * R + r;
            st_count[idx] = c;
            st_width[idx] = (int32_t)key_len(k_[p + c - 1]);  // rows ascending: the last row is the longest
            st_round[idx] = round;
            st_origin[idx] = step_base + V.ag[k];
            if (c <= 32) {
                uint32_t sum = 0;  // count * max_len <= budget < 2^31, or a singleton
                for (int j = 0; j < c; ++j) sum += key_len(k_[p + j]);
                st_real[idx] = (int32_t)sum;
            }
        }
        const int lane = threadIdx.x & 31, w = tid >> 5, nw = nth >> 5;
        for (int k = w; k < T_emit; k += nw) {
            const int c = ac[k];
            if (c <= 32) continue;
            const int p = ap[k];
            uint32_t sum = 0;
            for (int j = lane; j < c; j += 32) sum += key_len(k_[p + j]);
            sum = __reduce_add_sync(ODB_FULL_MASK, sum);
            if (lane == 0) st_real[(int64_t)(step_base + k) * R + r] = (int32_t)sum;
        }
        emitted_r = S;
        if (part != 0) return;
    } else {
        if (part != 0) return;
        for (int a = threadIdx.x; a < S; a += blockDim.x) pf[a] = 0;
        int carry = 0;
        for (int b0 = 0; b0 < T_emit; b0 += blockDim.x) {
            int k = b0 + threadIdx.x;
            int c = (k < T_emit) ? ac[k] : 0;
            int tot;
            int ex = block_excl_scan<int>(c, s_scan, tot) + carry;
            if (k < T_emit) {
                int64_t idx = (int64_t)(step_base + k) * R + r;
                int p = ap[k];
                st_count[idx] = c;
                st_width[idx] = (int32_t)key_len(k_[p + c - 1]);
                st_round[idx] = round;
                st_origin[idx] = step_base + V.ag[k];
                ao[k] = cur + ex;
            }
            carry += tot;
        }
        emitted_r = carry;
        __syncthreads();
        // copy ids and sum the lengths: one warp per group
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
        for (int k = w; k < T_emit; k += nw) {
            const int p = ap[k], c = ac[k], o = ao[k];
            uint32_t sum = 0;
            for (int j = lane; j < c; j += 32) {
                const uint64_t key = k_[p + j];
                const int id = key_id(key);
                sum += key_len(key);
                emit_ids[base + o + j] = id;
                emit_pos[base + id] = o + j;
                pf[p + j] = 1;
            }
            sum = __reduce_add_sync(ODB_FULL_MASK, sum);
            if (lane == 0) st_real[(int64_t)(step_base + k) * R + r] = (int32_t)sum;
        }
    }
    int n_left_new = 0;
    if (!all_emitted) {
        __syncthreads();
        int32_t *lf = left_ids + base;
        n_left_new = block_compact(
            S, s_scan, [&](int a) { return pf[a] == 0; }, [&](int a, int kidx) { lf[kidx] = key_id(k_[a]); });
    }
    if (threadIdx.x == 0) {
        int nl_old = *V.n_left, fp = *V.fetch_pos;
        int fp_new = fp + (S - nl_old);
        *V.emit_cur = cur + emitted_r;
        *V.n_left = n_left_new;
        *V.fetch_pos = fp_new;
        if (n_left_new + (n_r - fp_new) == 0) atomicAdd(&rec->n_finished, 1);
    }
}

// The kernel: the body above, then -- single-process mode -- the LAST CTA to finish closes the round on
// the device: it evaluates the termination predicates on the status every rank shares (Thm 3 proof
// P:341) exactly as the host state machine does, and writes the plan sizes into the device-resident
// PlanDims, so that the kernels after the round loop (slot scan, collate preparation, collate) can be
// enqueued behind this one without a host round trip: they read `complete` and skip if another round is due.
__global__ void __launch_bounds__(kRankThreads)
k_commit(const uint64_t *__restrict__ keys, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ S_arr,
         const int32_t *__restrict__ G_arr, int R, const int32_t *__restrict__ agpos, const int32_t *__restrict__ agcnt,
         const int32_t *__restrict__ agorg, int32_t *__restrict__ agoff, const int32_t *__restrict__ step_samples, int step_base, int round, int join_mode,
         long long quota, long long emitted_before, int32_t *__restrict__ st_count, int32_t *__restrict__ st_width,
         int32_t *__restrict__ st_real, int32_t *__restrict__ st_round, int32_t *__restrict__ st_origin,
         uint8_t *__restrict__ posflag,
         int32_t *__restrict__ emit_ids, int32_t *__restrict__ emit_pos, int32_t *__restrict__ left_ids, int32_t *n_left,
         int32_t *fetch_pos, int32_t *emit_cur, const int32_t *__restrict__ emit_snap, RoundRec *rec, PlanDims *dims,
         unsigned int *done_ctr, RoundRec *h_rec_out) {
    {
        const int r = blockIdx.x;
        RankView V;
        V.base = rank_ptr[r];
        const int64_t jb = V.base + r;
        V.k = keys + V.base;
        V.ap = agpos + jb;
        V.ac = agcnt + jb;
        V.ag = agorg + jb;
        V.ao = agoff + jb;
        V.pf = posflag + V.base;
        V.S = S_arr[r];
        V.Gr = G_arr[r];
        V.cur = emit_snap[r];
        V.n_r = (int)(rank_ptr[r + 1] - V.base);
        V.n_left = n_left + r;
        V.fetch_pos = fetch_pos + r;
        V.emit_cur = emit_cur + r;
        commit_body(r, R, V, step_samples, step_base, round, join_mode, quota, emitted_before, st_count, st_width, st_real,
                    st_round, st_origin, emit_ids, emit_pos, left_ids, rec, false, blockIdx.y, gridDim.y);
    }
    if (!dims) return;  // distributed mode: the host decides from the gathered status
    __shared__ int s_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(done_ctr, 1u);
        s_last = (t == gridDim.x * gridDim.y - 1u) ? 1 : 0;
    }
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        const volatile RoundRec *vr = rec;
        const int T_emit = vr->T_emit, quota_hit = vr->quota_hit, n_fin = vr->n_finished, bad = vr->bad_length;
        int complete = 0, stop = 0, n_rounds = 0;
        if (quota_hit) {  // Thm 2 / P:347: the trainer-side emitted-sample count reached the quota
            complete = 1;
            stop = ODB_STOP_QUOTA;
            n_rounds = round + 1;
        } else if (join_mode ? (n_fin == R) : (n_fin > 0)) {  // the next round is the terminal check
            complete = 1;
            stop = join_mode ? ODB_STOP_ALL_FINISHED : ODB_STOP_LOGICAL;
            n_rounds = round + 2;
        }
        dims->n_steps = step_base + T_emit;
        dims->n_rounds = n_rounds;
        dims->stop_reason = stop;
        dims->bad_length = bad;
        dims->err = 0;
        dims->complete = bad ? 0 : complete;
        *done_ctr = 0u;
        // the round's status goes straight to the host's pinned copy (odb_round_status waits for an event behind this
        // kernel): no copy operation between the commit and the slot scan
        if (h_rec_out) {
            RoundRec out;
            out.T = vr->T;
            out.T_emit = T_emit;
            out.quota_hit = quota_hit;
            out.n_finished = n_fin;
            out.bad_length = bad;
            out.done = vr->done;
            out.emitted_round = vr->emitted_round;
            *h_rec_out = out;
            __threadfence_system();
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The whole round loop in ONE launch (A0 .. A8, every protocol round): the paper's operating point is a
// grouping buffer of about a thousand samples per rank, i.e. tens of protocol rounds per rank stream,
// each of them a few microseconds of work -- far less than a kernel launch plus a host round trip.
// One persistent CTA per rank (cooperative launch: all R CTAs are resident) loops over the rounds:
//   window fill + merge sort in shared memory (A0, A1) -> successor + jump-out tables (A2, A3) ->
//   the rank's (G_r, S_r / "finished") goes into a double-buffered summary, GRID BARRIER -- the paper's one
//   unconditional exchange per round (deadlock-freedom Lemma 3) -- every CTA evaluates Eq. 3 and
//   the termination predicates on the same summary (Thm 3 proof P:341) -> split / overflow (A5, A6) ->
//   [non-join with a quota: a second grid barrier, the global step totals are needed for the cut] ->
//   commit (A7, A8a).
// The device functions are the ones the per-round kernels use; per-round scratch lives in the same global
// arrays (L2-resident).  Requirements (odb_api.cu checks them): windows of at most 4096 samples, R resident
// CTAs, every view has arrived (no odb_set_available), single-process mode.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int *p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// all CTAs of the (cooperatively launched) grid; `target` = arrivals expected so far, counter zeroed by the host
__device__ __forceinline__ void grid_barrier(unsigned int *ctr, unsigned int target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(ctr, 1u);
        while (ld_acquire_u32(ctr) < target) {
        }
        __threadfence();
    }
    __syncthreads();
}

struct RoundsArgs {
    SortArgs sort;  // window fill + sort inputs (first = 1: the per-run state is cleared in round 0)
    int R;
    uint32_t budget;
    int rule, join_mode, slot_capacity;
    long long quota, emitted_before;
    int32_t *G, *S, *gpos, *agpos, *agcnt, *agorg, *agoff, *emit_snap;
    int32_t *st_count, *st_width, *st_real, *st_round, *st_origin;
    uint8_t *posflag;
    int32_t *emit_ids, *left_ids_w;
    int32_t *gs;  // [2][2 R]: the per-round summary, double-buffered by round parity
    unsigned int *bar;
    PlanDims *dims;
    const SpecRec *spec;  // non-NULL: the rounds [0, spec->j_star) were committed by the round-parallel planner
};

// dynamic shared memory of k_rounds: the sort buffer (also scratch of the list ranking and of the overflow
// sort), the sorted window, and the round's group tables
constexpr size_t kRoundsSmem = (size_t)kMsPadded * 8 + (size_t)kMsChunk * 8 + 4 * (size_t)(kMsChunk + 4) * 4;

__global__ void __launch_bounds__(kMsThreads) k_rounds(const RoundsArgs A) {
    extern __shared__ __align__(16) unsigned char rd_smem[];
    __shared__ int s_scan[34];
    __shared__ uint16_t s_e2[32];
    __shared__ int s_red[3];
    __shared__ int s_state[3];  // n_left, fetch_pos, emit_cur of this rank
    __shared__ RoundRec s_rec;
    uint64_t *X = reinterpret_cast<uint64_t *>(rd_smem);  // kMsPadded keys
    uint64_t *K = X + kMsPadded;                          // the sorted window, kMsChunk keys
    int32_t *s_gp = reinterpret_cast<int32_t *>(K + kMsChunk);
    int32_t *s_ap = s_gp + (kMsChunk + 4), *s_ac = s_ap + (kMsChunk + 4), *s_ag = s_ac + (kMsChunk + 4);
    const int r = blockIdx.x, t = threadIdx.x, R = A.R;
    const SortArgs &SA = A.sort;
    if (SA.first) ms_first_round_init(SA, (int64_t)r * kMsThreads + t, (int64_t)gridDim.x * kMsThreads);
    const int64_t base = SA.rank_ptr[r];
    const int n_r = (int)(SA.rank_ptr[r + 1] - base);
    const int64_t jb = base + r;
    unsigned int n_bar = 0;
    int n_steps = 0, n_rounds = 0, stop = 0, bad = 0, round0 = 0;
    bool run_loop = true;
    if (t < 3) s_state[t] = 0;
    if (A.spec) {
        // resume behind the round-parallel planner: no leftovers so far, every rank has fetched round0 windows
        round0 = __ldcg(&A.spec->j_star);
        n_steps = __ldcg(&A.spec->n_steps);
        const int fp0 = (int)min((long long)round0 * SA.buffer_size, (long long)n_r);
        if (t == 1 || t == 2) s_state[t] = fp0;  // fetch_pos, emit_cur
        if (t == 0) bad = __ldcg(&SA.rec->bad_length);
        bad = __syncthreads_or(bad);
        if (bad) run_loop = false;
        else if (__ldcg(&A.spec->complete)) {  // round0 is the terminal check
            stop = A.join_mode ? ODB_STOP_ALL_FINISHED : ODB_STOP_LOGICAL;
            n_rounds = round0 + 1;
            run_loop = false;
        }
    }
    __syncthreads();
    long long emitted_before = A.emitted_before;
    const bool quota_mode = !A.join_mode && A.quota > 0;
    if (A.spec && quota_mode && round0 > 0) {
        // the committed rounds emitted their whole windows: the first round0 * B views of every stream (or all of it)
        __shared__ long long s_emit64[34];
        long long part = 0;
        for (int q = t; q < R; q += kMsThreads) {
            const long long nq = SA.rank_ptr[q + 1] - SA.rank_ptr[q];
            part += min((long long)round0 * SA.buffer_size, nq);
        }
        long long tot;
        (void)block_excl_scan<long long>(part, s_emit64, tot);
        emitted_before += tot;
    }
    for (int round = round0; run_loop; ++round) {
        // ---- A0 + A1: this rank's window, sorted ----
        const int nl = s_state[0], fp = s_state[1], cur = s_state[2];
        const int S = ms_window_size(nl, fp, n_r, SA.buffer_size);
        int G = 0;
        if (S > 0) {
            uint64_t k[kMsItems];
            const int n_keys = ms_active_keys(S);
            ms_load_keys(SA, base, nl, fp, 0, S, n_keys, k);
            ms_sort_cta(k, X, n_keys);
            for (int i = t; i < S; i += kMsThreads) K[i] = X[ms_pad(i)];
            __syncthreads();
            // ---- A2 + A3: candidate groups ----
            G = form_hier_body(K, S, A.budget, A.rule, s_gp, rd_smem, s_scan, s_e2);
        }
        // ---- the exchange: (G_r, S_r), S_r = -1 for "finished" (nothing buffered, nothing pending) ----
        int32_t *gs = A.gs + (size_t)(round & 1) * 2 * R;
        if (t == 0) {
            __stcg(&gs[2 * r], G);
            __stcg(&gs[2 * r + 1], S == 0 ? -1 : S);
            s_red[0] = 0;
            s_red[1] = 0x7fffffff;
            s_red[2] = 0;
        }
        grid_barrier(A.bar, (unsigned int)R * (++n_bar));
        for (int q = t; q < R; q += kMsThreads) {
            const int g = __ldcg(&gs[2 * q]), sq = __ldcg(&gs[2 * q + 1]);
            if (g > 0) {  // active set A = {r : G_r > 0}
                atomicMax(&s_red[0], g);
                if (sq > 0) atomicMin(&s_red[1], sq);
            }
            if (sq < 0) atomicAdd(&s_red[2], 1);
        }
        if (round == 0 && t == 0) bad = __ldcg(&SA.rec->bad_length);  // (a resumed run has checked it above)
        bad = __syncthreads_or(bad);
        if (bad) break;
        const int n_fin = s_red[2];
        // termination predicates, identical in every CTA (Thm 3 proof P:341)
        if (A.join_mode ? (n_fin == R) : (n_fin > 0)) {
            stop = A.join_mode ? ODB_STOP_ALL_FINISHED : ODB_STOP_LOGICAL;
            n_rounds = round + 1;  // this round was the terminal check
            break;
        }
        const int T = target_groups(s_red[0], s_red[1], A.slot_capacity);
        __syncthreads();  // s_red is rewritten next round
        if ((long long)n_steps + T > SA.step_cap) {  // cannot happen (n_steps <= the longest stream); never write past the tables
            bad = 2;
            break;
        }
        // ---- A4 .. A6: align to T ----
        if (G > 0) align_body(S, G, T, s_gp, s_ap, s_ac, s_ag, X, SA.step_samples + n_steps);
        if (quota_mode) grid_barrier(A.bar, (unsigned int)R * (++n_bar));  // the global step totals are complete
        if (t == 0) {
            s_rec.T = T;
            s_rec.done = 0;
            s_rec.n_finished = 0;
        }
        __syncthreads();
        // ---- A7 + A8a: commit ----
        RankView V;
        V.k = K;
        V.ap = s_ap;
        V.ac = s_ac;
        V.ag = s_ag;
        V.ao = A.agoff + jb;
        V.pf = A.posflag + base;
        V.S = S;
        V.Gr = G;
        V.cur = cur;
        V.n_r = n_r;
        V.base = base;
        V.n_left = &s_state[0];
        V.fetch_pos = &s_state[1];
        V.emit_cur = &s_state[2];
        commit_body(r, R, V, SA.step_samples, n_steps, round, A.join_mode, A.quota, emitted_before, A.st_count, A.st_width,
                    A.st_real, A.st_round, A.st_origin, A.emit_ids, SA.emit_pos, A.left_ids_w, &s_rec, true, 0, 1);
        __syncthreads();
        n_steps += s_rec.T_emit;
        if (quota_mode) {
            emitted_before += s_rec.emitted_round;
            if (s_rec.quota_hit) {  // Thm 2 / P:347
                stop = ODB_STOP_QUOTA;
                n_rounds = round + 1;
                break;
            }
        }
        __syncthreads();  // s_rec is rewritten next round
    }
    if (t == 0) {  // the rank's final state, for the kernels behind the round loop
        SA.n_left[r] = s_state[0];
        SA.fetch_pos[r] = s_state[1];
        SA.emit_cur[r] = s_state[2];
        if (r == 0) {
            A.dims->n_steps = n_steps;
            A.dims->n_rounds = n_rounds;
            A.dims->stop_reason = stop;
            A.dims->bad_length = bad == 1 ? 1 : 0;
            A.dims->err = bad == 2 ? ODB_ERR_STATE : 0;
            A.dims->complete = bad ? 0 : 1;
        }
        // the last CTA to leave rewinds the barrier counter for the next launch (every CTA has passed every barrier)
        if (atomicAdd(A.bar + 1, 1u) == (unsigned int)(R - 1)) {
            A.bar[0] = 0u;
            A.bar[1] = 0u;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The protocol rounds ROUND-PARALLEL (A0 .. A8 for every round at once).  The round loop above keeps one CTA per
// rank busy and leaves the other SMs idle; at the paper's operating point (a 1024-sample grouping buffer,
// P:28) a rank stream is tens of rounds.  But a round only depends on its predecessors through the leftovers
// ("returned to the buffer") -- and there are none as long as no round overflows: splitting (T >= G_r)
// emits every sample of the window (Lemma 1).  Under that assumption round j of rank r drains exactly the
// views [j B, (j + 1) B) of its stream, so ALL windows of ALL rounds can be sorted and grouped at once:
//   k_spec_form    one CTA per (rank, round): window fill + sort + candidate groups (the device functions of the
//                  round loop); the last CTA of a round to arrive evaluates Eq. 3 on the round's (G_r, S_r) and
//                  checks the assumption for the NEXT round (nobody overflows: max_A G_r <= min(C+min, S+min));
//                  the last CTA of the launch finds j* = the first round that breaks it and scans the step bases;
//   k_spec_commit  one CTA per (rank, round < j*): split + commit (align_body / commit_body as they are);
//   k_rounds       resumes at round j* with the state those rounds leave behind (or only records the plan sizes
//                  when j* is the terminal check).
// The rounds that are terminal checks are known on the host (join: the first round in which every stream is
// drained; non-join without a quota: the first in which one is), so the grid holds only non-terminal rounds.
// With a sample quota the grid ends before the round whose cumulative emission reaches it (the host knows that
// round: committed rounds emit whole windows) and that round, with its cut, is the loop's.  Not used with arrival
// schedules; distributed mode gathers the G tables first (k_spec_T_world).  Results are those of the sequential
// loop by construction; tests compare both with the oracle.
// ---------------------------------------------------------------------------------------------
struct SpecArgs {
    SortArgs sort;
    int R, n_rounds;
    uint32_t budget;
    int rule, join_mode, slot_capacity;
    int x_keys;  // padded sort keys the shared-memory layout reserves
    int eval_T;  // 1: the launch closes the rounds itself (all ranks are local); 0: only the G table (distributed mode)
    int terminal_after;  // 1: the round behind the grid is the terminal check; 0: it is an ordinary round (quota mode)
    int32_t *gpos, *agpos, *agcnt, *agorg;
    int32_t *st_count, *st_width, *st_real, *st_round, *st_origin;
    int32_t *emit_ids, *left_ids_w;
    SpecRec *rec;
    int32_t *T_tab, *sb_tab, *G_tab;
    unsigned int *ctr;  // [0, n_rounds): arrivals per round; [kSpecMaxRounds]: rounds closed (all self-resetting)
};

// first scratch entry of window (r, j): every non-empty window of S samples owns S + 1 entries
__device__ __forceinline__ int64_t spec_off(int64_t base, int B, int r, int j) {
    return base + (base + B - 1) / B + r + (int64_t)j * (B + 1);
}

template <int ITEMS>
__global__ void __launch_bounds__(kMsChunk / ITEMS) k_spec_form(const SpecArgs A) {
    using MS = MsSort<ITEMS>;
    extern __shared__ __align__(16) unsigned char sp_smem[];
    __shared__ int s_scan[34];
    __shared__ uint16_t s_e2[32];
    __shared__ int s_red[2];
    __shared__ int s_flag;
    const SortArgs &SA = A.sort;
    const int r = blockIdx.x, j = blockIdx.y, t = threadIdx.x, R = A.R, B = SA.buffer_size;
    ms_first_round_init(SA, ((int64_t)j * R + r) * blockDim.x + t, (int64_t)gridDim.x * gridDim.y * blockDim.x);
    const int64_t base = SA.rank_ptr[r];
    const int n_r = (int)(SA.rank_ptr[r + 1] - base);
    const int fp = (int)min((long long)j * B, (long long)n_r);
    const int S = min(B, n_r - fp);
    int G = 0;
    if (S > 0) {
        uint64_t *X = reinterpret_cast<uint64_t *>(sp_smem);
        uint64_t *K = X + A.x_keys;
        int32_t *gp = reinterpret_cast<int32_t *>(K + B);
        uint64_t k[ITEMS];
        const int n_keys = MS::active_keys(S);
        ms_load_keys_t<ITEMS>(SA, base, 0, fp, 0, S, n_keys, k);
        MS::sort_cta(k, X, n_keys);
        uint64_t *out = SA.keys_out + base + fp;
        for (int i = t; i < S; i += blockDim.x) {
            const uint64_t key = X[MS::pad(i)];
            K[i] = key;
            out[i] = key;
        }
        __syncthreads();
        G = form_hier_body(K, S, A.budget, A.rule, gp, sp_smem, s_scan, s_e2);
        __syncthreads();
        int32_t *gpo = A.gpos + spec_off(base, B, r, j);
        for (int i = t; i <= G; i += blockDim.x) gpo[i] = gp[i];
    }
    if (t == 0) __stcg(&A.G_tab[(int64_t)j * R + r], G);
    if (!A.eval_T) return;  // distributed mode: the tables of all processes are gathered first (k_spec_T_world)
    // ---- the last CTA of round j to arrive: Eq. 3 and the no-overflow check ----
    __threadfence();
    __syncthreads();
    if (t == 0) {
        s_flag = atomicAdd(&A.ctr[j], 1u) == (unsigned int)(R - 1);
        s_red[0] = 0;
        s_red[1] = 0x7fffffff;
    }
    __syncthreads();
    if (!s_flag) return;
    __threadfence();
    for (int q = t; q < R; q += blockDim.x) {
        const int g = __ldcg(&A.G_tab[(int64_t)j * R + q]);
        if (g > 0) {  // active set A = {r : G_r > 0}; its windows are non-empty
            const int64_t bq = SA.rank_ptr[q];
            const int nq = (int)(SA.rank_ptr[q + 1] - bq);
            const int sq = min(B, nq - (int)min((long long)j * B, (long long)nq));
            atomicMax(&s_red[0], g);
            atomicMin(&s_red[1], sq);
        }
    }
    __syncthreads();
    if (t == 0) {
        const int maxG = s_red[0];
        const int T = target_groups(maxG, s_red[1], A.slot_capacity);
        // every rank splits up to T (or idles): nothing is dropped, the next round starts without leftovers
        __stcg(&A.T_tab[j], T == maxG ? T : -1);
        A.ctr[j] = 0u;
        __threadfence();
        s_flag = atomicAdd(&A.ctr[kSpecMaxRounds], 1u) == (unsigned int)(A.n_rounds - 1);
        s_red[0] = A.n_rounds;
    }
    __syncthreads();
    if (!s_flag) return;
    // ---- the last CTA of the launch: j* and the step bases ----
    __threadfence();
    for (int q = t; q < A.n_rounds; q += blockDim.x)
        if (__ldcg(&A.T_tab[q]) < 0) atomicMin(&s_red[0], q);
    __syncthreads();
    const int js = s_red[0];
    int carry = 0;
    for (int q0 = 0; q0 < js; q0 += blockDim.x) {
        const int q = q0 + t;
        const int v = q < js ? __ldcg(&A.T_tab[q]) : 0;
        int tot;
        const int ex = block_excl_scan<int>(v, s_scan, tot);
        if (q < js) A.sb_tab[q] = carry + ex;
        carry += tot;
    }
    if (t == 0) {
        A.rec->j_star = js;
        A.rec->n_steps = carry;
        A.rec->complete = (js == A.n_rounds && A.terminal_after) ? 1 : 0;
        A.rec->pad_ = 0;
        A.ctr[kSpecMaxRounds] = 0u;
    }
}

__global__ void __launch_bounds__(kMsThreads) k_spec_commit(const SpecArgs A) {
    __shared__ RoundRec s_rec;
    __shared__ int s_state[3];
    const SortArgs &SA = A.sort;
    const int r = blockIdx.x, j = blockIdx.y, t = threadIdx.x, R = A.R, B = SA.buffer_size;
    if (j >= A.rec->j_star) return;
    const int T = A.T_tab[j], sb = A.sb_tab[j], G = A.G_tab[(int64_t)j * R + r];
    const int64_t base = SA.rank_ptr[r];
    const int n_r = (int)(SA.rank_ptr[r + 1] - base);
    const int fp = (int)min((long long)j * B, (long long)n_r);
    const int S = min(B, n_r - fp);
    const int64_t off = spec_off(base, B, r, j);
    if (t == 0) {
        s_rec.T = T;
        s_rec.done = 0;
        s_rec.n_finished = 0;
        s_state[0] = 0;
        s_state[1] = fp;
        s_state[2] = fp;
    }
    // A5: split up to T (G <= T in every committed round: the overflow branch is never taken)
    if (G > 0) align_body(S, G, T, A.gpos + off, A.agpos + off, A.agcnt + off, A.agorg + off, nullptr, SA.step_samples + sb);
    __syncthreads();
    RankView V;
    V.k = SA.keys_out + base + fp;
    V.ap = A.agpos + off;
    V.ac = A.agcnt + off;
    V.ag = A.agorg + off;
    V.ao = nullptr;
    V.pf = nullptr;
    V.S = S;
    V.Gr = G;
    V.cur = fp;
    V.n_r = n_r;
    V.base = base;
    V.n_left = &s_state[0];
    V.fetch_pos = &s_state[1];
    V.emit_cur = &s_state[2];
    commit_body(r, R, V, SA.step_samples, sb, j, A.join_mode, 0ll, 0ll, A.st_count, A.st_width, A.st_real, A.st_round,
                A.st_origin, A.emit_ids, SA.emit_pos, A.left_ids_w, &s_rec, true, 0, 1);
}

// Distributed mode (ranks over several processes): the same planner with ONE exchange for all its rounds instead of
// one per round.  Every process forms the windows of its ranks for the rounds [0, J) (k_spec_form, eval_T = 0), the
// G tables of all processes are all_gathered (layout [process][round][local rank]) next to every rank's stream
// length, and every process evaluates Eq. 3 and the no-overflow check of every round on the same gathered data
// (Lemma 3: identical decisions everywhere), commits its ranks' rounds before j* and goes on round by round from there.
__global__ void __launch_bounds__(1024)
k_spec_T_world(const int32_t *__restrict__ G_world, const int32_t *__restrict__ n_world, int n_procs, int R_local, int n_rounds,
               int B, int slot_capacity, int32_t *__restrict__ T_tab, int32_t *__restrict__ sb_tab, SpecRec *rec) {
    __shared__ int s_scan[34];
    __shared__ int s_js;
    const int t = threadIdx.x;
    if (t == 0) s_js = n_rounds;
    __syncthreads();
    for (int j = t; j < n_rounds; j += blockDim.x) {
        int maxG = 0, minS = 0x7fffffff;
        for (int p = 0; p < n_procs; ++p)
            for (int r = 0; r < R_local; ++r) {
                const int g = G_world[((int64_t)p * n_rounds + j) * R_local + r];
                if (g > 0) {  // active set A; its windows are non-empty
                    const int nq = n_world[p * R_local + r];
                    const int sq = min(B, nq - (int)min((long long)j * B, (long long)nq));
                    maxG = max(maxG, g);
                    minS = min(minS, sq);
                }
            }
        const int T = target_groups(maxG, minS, slot_capacity);
        const int v = (T == maxG && maxG > 0) ? T : -1;
        T_tab[j] = v;
        if (v < 0) atomicMin(&s_js, j);
    }
    __syncthreads();
    const int js = s_js;
    int carry = 0;
    for (int q0 = 0; q0 < js; q0 += blockDim.x) {
        const int q = q0 + t;
        const int v = q < js ? T_tab[q] : 0;
        int tot;
        const int ex = block_excl_scan<int>(v, s_scan, tot);
        if (q < js) sb_tab[q] = carry + ex;
        carry += tot;
    }
    if (t == 0) {
        rec->j_star = js;
        rec->n_steps = carry;
        rec->complete = js == n_rounds ? 1 : 0;
        rec->pad_ = 0;
    }
}

// the rank state the committed rounds leave behind: no leftovers, j* windows fetched and emitted
__global__ void k_spec_state(const SpecRec *rec, const int64_t *__restrict__ rank_ptr, int R, int B, int32_t *n_left,
                             int32_t *fetch_pos, int32_t *emit_cur) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    const int n_r = (int)(rank_ptr[r + 1] - rank_ptr[r]);
    const int fp = (int)min((long long)rec->j_star * B, (long long)n_r);
    n_left[r] = 0;
    fetch_pos[r] = fp;
    emit_cur[r] = fp;
}

// ---------------------------------------------------------------------------------------------
// A9 and the rank-major plan tables.
//
// k_fin_scan: one pass over the slots in rank-major order s = r * n_steps + k.  Tiles of kFinTile
// slots take a ticket (so every predecessor tile is running or done), transpose the step-major
// staging tables, and scan four int64 quantities with decoupled look-back: the 16-aligned block
// area (-> grp_offset), the sample count (-> grp_sample_ptr), count*width and the real tokens
// (-> totals).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kFinThreads)
k_fin_scan(int R, PlanDims *dims, const int32_t *__restrict__ st_count, const int32_t *__restrict__ st_width,
           const int32_t *__restrict__ st_real, const int32_t *__restrict__ st_round,
           const int32_t *__restrict__ st_origin, int32_t *__restrict__ grp_count, int32_t *__restrict__ grp_width,
           int32_t *__restrict__ grp_round, int32_t *__restrict__ grp_real, int32_t *__restrict__ grp_origin,
           int64_t *__restrict__ grp_offset, int64_t *__restrict__ grp_sample_ptr, ScanTile *tiles, unsigned int *ticket,
           CapCheck cap, int64_t n_total, int64_t *rank_off, PlanDims *h_dims_out, int epoch, RoundRec *clear_rec) {
    __shared__ long long s_scan64[34];
    __shared__ long long s_base[4];
    __shared__ int s_tile;
    if (!dims->complete) {  // enqueued behind a round that did not terminate the protocol
        if (h_dims_out && blockIdx.x == 0 && threadIdx.x == 0) {
            *h_dims_out = *dims;
            __threadfence_system();
        }
        return;
    }
    const int n_steps = dims->n_steps;
    const int64_t n_slots = (int64_t)R * n_steps;
    const int64_t n_tiles = max((n_slots + kFinTile - 1) / kFinTile, (int64_t)1);
    for (;;) {
        __syncthreads();  // everyone has read the previous s_tile / s_base
        if (threadIdx.x == 0) s_tile = (int)atomicAdd(ticket, 1u);
        __syncthreads();
        const int tile = s_tile;
        if ((int64_t)tile >= n_tiles) break;
        const int64_t s0 = (int64_t)tile * kFinTile + (int64_t)threadIdx.x * kFinItems;
        long long v[4][kFinItems];
        long long sum[4] = {0, 0, 0, 0};
#pragma unroll
        for (int i = 0; i < kFinItems; ++i) {
            const int64_t s = s0 + i;
            long long c = 0, w = 0, re = 0;
            if (s < n_slots) {
                const int r = (int)(s / n_steps);
                const int k = (int)(s - (int64_t)r * n_steps);
                const int64_t src = (int64_t)k * R + r;
                c = st_count[src];
                w = st_width[src];
                re = st_real[src];
                grp_count[s] = (int32_t)c;
                grp_width[s] = (int32_t)w;
                grp_real[s] = (int32_t)re;
                grp_round[s] = st_round[src];
                grp_origin[s] = st_origin[src];
            }
            const long long area = c * w;
            v[0][i] = (area + 15) / 16 * 16;
            v[1][i] = c;
            v[2][i] = area;
            v[3][i] = re;
#pragma unroll
            for (int q = 0; q < 4; ++q) sum[q] += v[q][i];
        }
        long long ex[4], total[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) ex[q] = block_excl_scan<long long>(sum[q], s_scan64, total[q]);
        ScanTile *me = tiles + tile;
        if (threadIdx.x == 0) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                me->agg[q] = total[q];
                if (tile == 0) me->inc[q] = total[q];
            }
            st_flag(&me->flag, (epoch << 2) | (tile == 0 ? 2 : 1));
            if (tile == 0) {
#pragma unroll
                for (int q = 0; q < 4; ++q) s_base[q] = 0;
            }
        }
        if (tile > 0 && threadIdx.x < 32) {  // warp 0 looks back over up to 32 predecessors at a time
            const int lane = threadIdx.x;
            long long acc[4] = {0, 0, 0, 0};
            int t = tile - 1;
            while (true) {
                const int tt = t - lane;
                int f = 2;  // tiles before the first count as "inclusive prefix 0"
                long long x[4] = {0, 0, 0, 0};
                if (tt >= 0) {
                    do {  // (a flag of an earlier launch counts as "nothing yet": the states are never cleared)
                        f = ld_flag(&tiles[tt].flag);
                    } while ((f >> 2) != epoch);
                    f &= 3;
#pragma unroll
                    for (int q = 0; q < 4; ++q) x[q] = (f == 2) ? __ldcg(&tiles[tt].inc[q]) : __ldcg(&tiles[tt].agg[q]);
                }
                const uint32_t done = __ballot_sync(ODB_FULL_MASK, f == 2);
                const int first = __ffs(done) - 1;  // nearest tile with an inclusive prefix (done != 0 once tt < 0)
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    long long y = (done == 0 || lane <= first) ? x[q] : 0;
#pragma unroll
                    for (int dlt = 16; dlt > 0; dlt >>= 1) y += __shfl_xor_sync(ODB_FULL_MASK, y, dlt);
                    acc[q] += y;
                }
                if (done) break;
                t -= 32;
            }
            if (lane == 0) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    s_base[q] = acc[q];
                    me->inc[q] = acc[q] + total[q];
                }
                st_flag(&me->flag, (epoch << 2) | 2);
            }
        }
        __syncthreads();
        long long run_o = s_base[0] + ex[0], run_p = s_base[1] + ex[1];
#pragma unroll
        for (int i = 0; i < kFinItems; ++i) {
            const int64_t s = s0 + i;
            if (s < n_slots) {
                grp_offset[s] = run_o;
                grp_sample_ptr[s] = run_p;
                if (rank_off && s % n_steps == 0) rank_off[s / n_steps] = run_o;  // arena offset of each rank's first slot
            }
            run_o += v[0][i];
            run_p += v[1][i];
        }
        if (threadIdx.x == 0 && (int64_t)tile == n_tiles - 1) {
            const long long tot_e = s_base[0] + total[0], tot_s = s_base[1] + total[1];
            grp_offset[n_slots] = tot_e;
            grp_sample_ptr[n_slots] = tot_s;
            if (rank_off) {
                rank_off[R] = tot_e;
                if (n_steps == 0)
                    for (int r = 0; r < R; ++r) rank_off[r] = 0;
            }
            dims->n_slots = n_slots;
            dims->total_elems = tot_e;
            dims->samples_emitted = tot_s;
            dims->padded_elems = s_base[2] + total[2];
            dims->real_tokens = (unsigned long long)(s_base[3] + total[3]);
            // Lemma 1: emitted + un-emitted = all (n_total < 0: an offline plan, no leftovers)
            dims->samples_left = n_total >= 0 ? n_total - tot_s : 0;
            // the caller's capacities (odb_run enqueues the collate kernels before the host sees the sizes)
            int err = 0;
            if (cap.arena >= 0 && tot_e > cap.arena) err = ODB_ERR_CAPACITY;
            if (cap.tiles >= 0 && (tot_e + kColTile - 1) / kColTile > cap.tiles) err = ODB_ERR_CAPACITY;
            if (cap.slots >= 0 && n_slots > cap.slots) err = ODB_ERR_CAPACITY;
            if (cap.ids >= 0 && tot_s > cap.ids) err = ODB_ERR_CAPACITY;
            if (cap.steps >= 0 && n_steps > cap.steps) err = ODB_ERR_CAPACITY;
            if (cap.left >= 0 && n_total >= 0 && n_total - tot_s > cap.left) err = ODB_ERR_CAPACITY;
            dims->err = err;
            // the sizes go straight to the caller's pinned copy: the host waits for an event behind this kernel, no
            // copy operation sits between the slot scan and the collate preparation
            if (h_dims_out) {
                *h_dims_out = *dims;
                __threadfence_system();
            }
            // the plan is complete: nothing reads the per-round status record any more; it is cleared here for the
            // next run (which then needs no clearing operation in front of its first kernel)
            if (clear_rec) {
                clear_rec->T = 0;
                clear_rec->T_emit = 0;
                clear_rec->quota_hit = 0;
                clear_rec->n_finished = 0;
                clear_rec->bad_length = 0;
                clear_rec->done = 0;
                clear_rec->emitted_round = 0;
            }
        }
    }
    // the last CTA to leave rewinds the ticket counter for the next launch (no clearing pass in front of this kernel)
    if (threadIdx.x == 0) {
        const unsigned int prev = atomicAdd(ticket + 1, 1u);
        if (prev == gridDim.x - 1u) {
            ticket[0] = 0u;
            ticket[1] = 0u;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// host launchers
// ---------------------------------------------------------------------------------------------
#define ODB_LAUNCH_CHECK(c)                       \
    do {                                          \
        (c)->launches++;                          \
        cudaError_t e_ = cudaGetLastError();      \
        if (e_ != cudaSuccess) return e_;         \
    } while (0)

cudaError_t launch_begin(odb_ctx *c, cudaStream_t st) {
    const int R = c->prm.n_ranks;  // (d_rec was zeroed when the run began)
    const int64_t step_cap = c->step_samples.p ? (int64_t)c->step_samples.cap : 0;
    const int64_t bound = std::max<int64_t>(std::max<int64_t>(c->n_total, R), step_cap);
    int blocks = (int)std::min<int64_t>((bound + 1023) / 1024, (int64_t)c->sm_count * 4);
    k_begin<<<std::max(blocks, 1), 256, 0, st>>>(c->d_lengths, c->n_total, R, c->n_left, c->fetch_pos, c->emit_cur, c->G,
                                                c->S, c->emit_pos, c->step_samples.p, step_cap, c->d_rec);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

static int max_window_bound(const odb_ctx *c) {
    int64_t m = c->max_nr;
    if (c->prm.buffer_size > 0 && m > c->prm.buffer_size) m = c->prm.buffer_size;
    return (int)m;
}

static size_t form_hier_smem_bytes(int maxS) {
    const size_t np = (size_t)maxS + ((size_t)maxS >> 5) + 2, npe = (np + 1) & ~(size_t)1;
    const size_t nb1 = ((size_t)maxS + 31) >> 5;
    return 3 * npe * 2 + ((nb1 + 1) & ~(size_t)1) * 2 + nb1 * 4 + 16;
}

static size_t form_smem_bytes(int maxS) {
    const size_t n1p = ((size_t)maxS + 1 + 7) & ~(size_t)7;
    const size_t words = ((size_t)maxS + 1 + 31) >> 5;
    return 4 * n1p + 4 * words;
}

// Segmented sort of arbitrary segments (used by the offline planners): the cluster sort when every segment has
// at most 65536 keys, else chunk sorts + merge passes through global memory.  A.keys_out / keyB: ping-pong buffers;
// *sorted receives the buffer that holds the result.  A.first must be 0 on the fallback path (no state reset there).
cudaError_t sort_segments_any(odb_ctx *c, const SortArgs &A, int64_t nseg, int maxS, uint64_t *keyB, uint64_t **sorted,
                              cudaStream_t st) {
    *sorted = A.keys_out;
    if (maxS == 0 || nseg == 0) return cudaSuccess;
    cudaError_t se = c->no_cluster_sort ? cudaErrorNotSupported : launch_sort_segments(c, A, nseg, maxS, st);
    if (se == cudaSuccess) return cudaSuccess;
    if (se != cudaErrorNotSupported) {
        (void)cudaGetLastError();
        c->no_cluster_sort = true;
    }
    if (nseg > 65535) return cudaErrorInvalidValue;  // (large segments and that many of them do not occur together)
    const int chunks = (maxS + kSortChunk - 1) / kSortChunk;
    k_chunk_sort_reg<<<dim3(chunks, (unsigned)nseg), kSortRegThreads, 0, st>>>(A.len, A.rank_ptr, A.n_left, A.fetch_pos,
                                                                             A.left_ids, A.arrived, A.buffer_size,
                                                                             A.keys_out, A.S_out, c->d_rec);
    ODB_LAUNCH_CHECK(c);
    uint64_t *src = A.keys_out, *dst = keyB;
    for (int64_t w = kSortChunk; w < maxS; w *= 2) {
        const int gx = (maxS + kMergeTile - 1) / kMergeTile;
        k_merge_pass<<<dim3(gx, (unsigned)nseg), kMergeThreads, 0, st>>>(src, dst, A.rank_ptr, A.S_out, (int)w);
        ODB_LAUNCH_CHECK(c);
        uint64_t *t = src;
        src = dst;
        dst = t;
    }
    *sorted = src;
    return cudaSuccess;
}

// A2 + A3 over arbitrary segments with the padded-area rule (the offline planners' greedy packing, App. I)
cudaError_t form_segments_maxfit(odb_ctx *c, const uint64_t *sorted, const int64_t *seg_ptr, const int32_t *S_arr,
                                 int64_t nseg, int maxS, int32_t *jA, int32_t *jB, uint8_t *mark, int32_t *gpos,
                                 int32_t *G_out, cudaStream_t st) {
    if (nseg == 0 || maxS == 0) return cudaSuccess;
    const uint32_t budget = (uint32_t)c->prm.budget;
    {
        const unsigned ns = (unsigned)nseg;  // (gridDim.x holds 2^31 - 1 blocks)
        const int64_t s0 = 0;
        if (maxS <= 32768) {
            if (!c->attr_form_hier) {
                cudaError_t e = cudaFuncSetAttribute(k_form_groups_hier, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                     (int)kFormSmemLimit);
                if (e != cudaSuccess) return e;
                c->attr_form_hier = true;
            }
            k_form_groups_hier<<<ns, kRankThreads, form_hier_smem_bytes(maxS), st>>>(sorted, seg_ptr + s0, S_arr + s0, budget,
                                                                                    ODB_RULE_MAXFIT_ASC, gpos, G_out + s0);
        } else {
            k_form_groups<<<ns, kRankThreads, 0, st>>>(sorted, seg_ptr + s0, S_arr + s0, budget, ODB_RULE_MAXFIT_ASC, jA, jB,
                                                       mark, gpos, G_out + s0);
        }
        ODB_LAUNCH_CHECK(c);
    }
    return cudaSuccess;
}

// the per-run state reset, when no sort launch has done it (no window anywhere, or the fallback sort)
cudaError_t flush_begin(odb_ctx *c, cudaStream_t st) {
    if (!c->begin_pending) return cudaSuccess;
    c->begin_pending = false;
    return launch_begin(c, st);
}

cudaError_t launch_round_form(odb_ctx *c, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    const int maxS = max_window_bound(c);
    if (maxS == 0) return flush_begin(c, st);
    // A0 + A1: one cluster launch (windows of up to 65536 keys); it also clears the per-run state in the
    // first round.  Larger windows: chunk sorts + merge passes through global memory.
    cudaError_t se = cudaErrorNotSupported;
    if (!c->no_cluster_sort) {
        se = launch_sort_window(c, maxS, c->begin_pending, st);
        if (se == cudaSuccess) c->begin_pending = false;
        else if (se != cudaErrorNotSupported) {  // e.g. a 16-CTA cluster the device will not schedule: fall back for good
            (void)cudaGetLastError();
            c->no_cluster_sort = true;
        }
    }
    if (se != cudaSuccess) {
        cudaError_t e = flush_begin(c, st);
        if (e != cudaSuccess) return e;
        const int chunks = (maxS + kSortChunk - 1) / kSortChunk;
        if (maxS > kSortChunk / 2)  // full-size chunks: the register-blocked network; small windows: the shared-memory one
            k_chunk_sort_reg<<<dim3(chunks, R), kSortRegThreads, 0, st>>>(c->d_lengths, c->d_rank_ptr, c->n_left, c->fetch_pos,
                                                                         c->left_ids, c->d_arrived, c->prm.buffer_size,
                                                                         c->keyA, c->S, c->d_rec);
        else
            k_chunk_sort<<<dim3(chunks, R), kSortThreads, 0, st>>>(c->d_lengths, c->d_rank_ptr, c->n_left, c->fetch_pos,
                                                                  c->left_ids, c->d_arrived, c->prm.buffer_size, c->keyA, c->S,
                                                                  c->d_rec);
        ODB_LAUNCH_CHECK(c);
        uint64_t *src = c->keyA, *dst = c->keyB;
        for (int64_t w = kSortChunk; w < maxS; w *= 2) {
            int gx = (maxS + kMergeTile - 1) / kMergeTile;
            k_merge_pass<<<dim3(gx, R), kMergeThreads, 0, st>>>(src, dst, c->d_rank_ptr, c->S, (int)w);
            ODB_LAUNCH_CHECK(c);
            uint64_t *t = src;
            src = dst;
            dst = t;
        }
        c->sorted = src;
    }
    // A2 + A3
    const size_t smem = form_smem_bytes(maxS);
    if (maxS <= 32768) {
        if (!c->attr_form_hier) {
            cudaError_t e = cudaFuncSetAttribute(k_form_groups_hier, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                 (int)kFormSmemLimit);
            if (e != cudaSuccess) return e;
            c->attr_form_hier = true;
        }
        k_form_groups_hier<<<R, kRankThreads, form_hier_smem_bytes(maxS), st>>>(c->sorted, c->d_rank_ptr, c->S,
                                                                               (uint32_t)c->prm.budget, c->prm.rule, c->gpos, c->G);
    } else if (smem <= kFormSmemLimit && maxS <= 65534) {
        if (!c->attr_form) {
            cudaError_t e = cudaFuncSetAttribute(k_form_groups_smem, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                 (int)kFormSmemLimit);
            if (e != cudaSuccess) return e;
            c->attr_form = true;
        }
        k_form_groups_smem<<<R, kRankThreads, smem, st>>>(c->sorted, c->d_rank_ptr, c->S, (uint32_t)c->prm.budget,
                                                          c->prm.rule, c->gpos, c->G);
    } else {
        k_form_groups<<<R, kRankThreads, 0, st>>>(c->sorted, c->d_rank_ptr, c->S, (uint32_t)c->prm.budget, c->prm.rule, c->jA,
                                                  c->jB, c->mark, c->gpos, c->G);
    }
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

static cudaError_t launch_align_kernel(odb_ctx *c, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    const size_t al_smem = (size_t)kAlignSmemKeys * sizeof(uint64_t);
    if (!c->attr_align) {
        cudaError_t e = cudaFuncSetAttribute(k_align, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)al_smem);
        if (e != cudaSuccess) return e;
        c->attr_align = true;
    }
    k_align<<<R, kRankThreads, al_smem, st>>>(c->d_rank_ptr, c->S, c->G, R, c->world_ranks ? c->gs_world : nullptr,
                                              c->world_ranks, c->prm.join_mode, c->prm.slot_capacity, c->gpos, c->agpos,
                                              c->agcnt, c->agorg, c->ovf, c->step_samples.p, c->n_steps, c->emit_cur, c->emit_snap,
                                              c->d_rec);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

static cudaError_t launch_commit_kernel(odb_ctx *c, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    k_commit<<<dim3(R, kCommitParts), kRankThreads, 0, st>>>(c->sorted, c->d_rank_ptr, c->S, c->G, R, c->agpos, c->agcnt, c->agorg, c->agoff,
                                         c->step_samples.p, c->n_steps, c->round, c->prm.join_mode,
                                         (long long)c->prm.sample_quota,
                                         (long long)c->prm.emitted_so_far + (long long)c->samples_emitted, c->st_count.p,
                                         c->st_width.p, c->st_real.p, c->st_round.p, c->st_origin.p, c->posflag,
                                         c->emit_ids, c->emit_pos, c->left_ids, c->n_left, c->fetch_pos, c->emit_cur,
                                         c->emit_snap, c->d_rec, c->world_ranks ? nullptr : c->d_dims, c->d_done_ctr,
                                         c->world_ranks ? nullptr : c->h_rec);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

cudaError_t launch_round_align(odb_ctx *c, cudaStream_t st) {
    cudaError_t e = launch_align_kernel(c, st);
    if (e != cudaSuccess) return e;
    return launch_commit_kernel(c, st);
}

cudaError_t launch_align_only(odb_ctx *c, cudaStream_t st) { return launch_align_kernel(c, st); }
cudaError_t launch_commit_only(odb_ctx *c, cudaStream_t st) { return launch_commit_kernel(c, st); }

// distributed mode: the local ranks' (G_r, S_r) pairs, the message of the per-round all_gather
__global__ void k_pack_summary(int R, const int32_t *__restrict__ G, const int32_t *__restrict__ S,
                               const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ fetch_pos,
                               int32_t *__restrict__ gs, RoundRec *rec) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q < R) {
        // status -1 "finished": nothing buffered and nothing pending; an empty window with views still
        // pending is status 0 "insufficient data".  Computed here, not in the sort kernel, because a
        // process whose ranks hold no sample at all never launches the sort.
        const int n_r = (int)(rank_ptr[q + 1] - rank_ptr[q]);
        const bool fin = S[q] == 0 && fetch_pos[q] >= n_r;
        gs[2 * q] = G[q];
        gs[2 * q + 1] = fin ? -1 : S[q];
    }
    if (q == 0) rec->done = 0;
}

cudaError_t launch_pack_summary(odb_ctx *c, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    k_pack_summary<<<(R + 127) / 128, 128, 0, st>>>(R, c->G, c->S, c->d_rank_ptr, c->fetch_pos, c->gs_local, c->d_rec);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

// The whole round loop in one cooperative launch (k_rounds).  cudaErrorNotSupported when the R CTAs cannot
// all be resident on this device (the caller then drives the rounds from the host).
// keys per thread of k_spec_form's window sort: 8 for grouping buffers of 512 samples and more, 4 below (measured
// planning stage with 4 / 8: buffer 256: 0.128 / 0.131 ms, 1024: 0.122 / 0.117 ms, 4096: 0.138 / 0.127 ms)
static int spec_items(const odb_ctx *c) { return c->prm.buffer_size >= 512 ? 8 : 4; }

static int host_active_keys(int S) {
    int n = 32 * kMsItems;
    while (n < S) n <<= 1;
    return std::min(n, kMsChunk);
}

// Arguments, block size and shared memory of the round-parallel planner's kernels for `spec_rounds` rounds.
static cudaError_t make_spec_args(odb_ctx *c, int spec_rounds, int eval_T, int terminal_after, cudaStream_t st, SpecArgs *out,
                                  int *threads_out, size_t *smem_out) {
    const int R = c->prm.n_ranks;
    const int B = c->prm.buffer_size;
    const int items = spec_items(c);
    int n_keys = 32 * items;
    while (n_keys < B) n_keys <<= 1;
    n_keys = std::min(n_keys, kMsChunk);
    // (measured: more threads per window are slower -- 256 / 512 / 1024 threads for 1024-key windows give a
    //  planning stage of 0.134 / 0.146 / 0.185 ms: the launch is throughput-bound, not latency-bound)
    *threads_out = std::max(n_keys / items, 128);
    const size_t x_keys = (size_t)n_keys + n_keys / items;
    const size_t x_bytes = std::max(x_keys * 8, (form_hier_smem_bytes(B) + 15) & ~(size_t)15);
    *smem_out = x_bytes + (size_t)B * 8 + ((size_t)B + 4) * 4;
    if (!c->spec_occ) {
        cudaError_t ae = cudaFuncSetAttribute(k_spec_form<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(96 * 1024));
        if (ae != cudaSuccess) return ae;
        ae = cudaFuncSetAttribute(k_spec_form<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(96 * 1024));
        if (ae != cudaSuccess) return ae;
        c->spec_occ = 1;
    }
    const size_t tab_fixed = 4 + (size_t)kSpecMaxRounds + 1;
    cudaError_t e = c->spec_tab.ensure(tab_fixed + 2 * ((size_t)kSpecMaxRounds + 1) + (size_t)spec_rounds * R, true, st);
    if (e != cudaSuccess) return e;
    SpecArgs P;
    memset(&P, 0, sizeof(P));
    P.sort.len = c->d_lengths;
    P.sort.rank_ptr = c->d_rank_ptr;
    P.sort.n_left = c->n_left;
    P.sort.fetch_pos = c->fetch_pos;
    P.sort.emit_cur = c->emit_cur;
    P.sort.left_ids = c->left_ids;
    P.sort.arrived = c->d_arrived;
    P.sort.buffer_size = B;
    P.sort.keys_out = c->keyA;
    P.sort.S_out = c->S;
    P.sort.rec = c->d_rec;
    P.sort.first = 1;
    P.sort.n_total = c->n_total;
    P.sort.emit_pos = c->emit_pos;
    P.sort.step_samples = c->step_samples.p;
    P.sort.step_cap = c->step_samples.p ? (int64_t)c->step_samples.cap : 0;
    P.R = R;
    P.n_rounds = spec_rounds;
    P.budget = (uint32_t)c->prm.budget;
    P.rule = c->prm.rule;
    P.join_mode = c->prm.join_mode;
    P.slot_capacity = c->prm.slot_capacity;
    P.x_keys = (int)(x_bytes / 8);
    P.eval_T = eval_T;
    P.terminal_after = terminal_after;
    P.gpos = c->gpos;
    P.agpos = c->agpos;
    P.agcnt = c->agcnt;
    P.agorg = c->agorg;
    P.st_count = c->st_count.p;
    P.st_width = c->st_width.p;
    P.st_real = c->st_real.p;
    P.st_round = c->st_round.p;
    P.st_origin = c->st_origin.p;
    P.emit_ids = c->emit_ids;
    P.left_ids_w = c->left_ids;
    P.rec = reinterpret_cast<SpecRec *>(c->spec_tab.p);
    P.ctr = reinterpret_cast<unsigned int *>(c->spec_tab.p + 4);
    P.T_tab = c->spec_tab.p + tab_fixed;
    P.sb_tab = P.T_tab + kSpecMaxRounds + 1;
    P.G_tab = P.sb_tab + kSpecMaxRounds + 1;
    *out = P;
    return cudaSuccess;
}

cudaError_t launch_rounds(odb_ctx *c, int spec_rounds, bool spec_terminal, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    const size_t smem = kRoundsSmem;
    if (c->rounds_max_ctas == 0) {
        int occ = 0, coop = 0;
        cudaError_t ae = cudaFuncSetAttribute(k_rounds, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (ae != cudaSuccess) return ae;
        cudaError_t e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_rounds, kMsThreads, smem);
        if (e != cudaSuccess) return e;
        c->rounds_max_ctas = coop ? std::max(occ * c->sm_count, 1) : -1;
    }
    if (c->rounds_max_ctas < R) return cudaErrorNotSupported;
    cudaError_t e = cudaSuccess;
    if (!c->gs_rounds) {
        e = cudaMalloc((void **)&c->gs_rounds, (size_t)4 * R * sizeof(int32_t) + 64);
        if (e != cudaSuccess) return e;
        // the barrier counter and the exit counter live behind the summary: zeroed once, rewound by the kernel itself
        e = cudaMemset(c->gs_rounds + (size_t)4 * R, 0, 64);
        if (e != cudaSuccess) return e;
    }
    unsigned int *bar = reinterpret_cast<unsigned int *>(c->gs_rounds + (size_t)4 * R);
    RoundsArgs A;
    memset(&A, 0, sizeof(A));
    A.sort.len = c->d_lengths;
    A.sort.rank_ptr = c->d_rank_ptr;
    A.sort.n_left = c->n_left;
    A.sort.fetch_pos = c->fetch_pos;
    A.sort.emit_cur = c->emit_cur;
    A.sort.left_ids = c->left_ids;
    A.sort.arrived = c->d_arrived;
    A.sort.buffer_size = c->prm.buffer_size;
    A.sort.keys_out = c->keyA;
    A.sort.S_out = c->S;
    A.sort.rec = c->d_rec;
    A.sort.first = 1;
    A.sort.n_total = c->n_total;
    A.sort.emit_pos = c->emit_pos;
    A.sort.step_samples = c->step_samples.p;
    A.sort.step_cap = c->step_samples.p ? (int64_t)c->step_samples.cap : 0;
    A.R = R;
    A.budget = (uint32_t)c->prm.budget;
    A.rule = c->prm.rule;
    A.join_mode = c->prm.join_mode;
    A.slot_capacity = c->prm.slot_capacity;
    A.quota = (long long)c->prm.sample_quota;
    A.emitted_before = (long long)c->prm.emitted_so_far;
    A.G = c->G;
    A.S = c->S;
    A.gpos = c->gpos;
    A.agpos = c->agpos;
    A.agcnt = c->agcnt;
    A.agorg = c->agorg;
    A.agoff = c->agoff;
    A.emit_snap = c->emit_snap;
    A.st_count = c->st_count.p;
    A.st_width = c->st_width.p;
    A.st_real = c->st_real.p;
    A.st_round = c->st_round.p;
    A.st_origin = c->st_origin.p;
    A.posflag = c->posflag;
    A.emit_ids = c->emit_ids;
    A.left_ids_w = c->left_ids;
    A.gs = c->gs_rounds;
    A.bar = bar;
    A.dims = c->d_dims;
    A.spec = nullptr;
    if (spec_rounds > 0) {
        // the rounds [0, spec_rounds) round-parallel; k_rounds resumes where the speculation stops
        SpecArgs P;
        int threads = 0;
        size_t sp_smem = 0;
        e = make_spec_args(c, spec_rounds, 1, spec_terminal ? 1 : 0, st, &P, &threads, &sp_smem);
        if (e != cudaSuccess) return e;
        if (spec_items(c) == 8) k_spec_form<8><<<dim3((unsigned)R, (unsigned)spec_rounds), threads, sp_smem, st>>>(P);
        else k_spec_form<4><<<dim3((unsigned)R, (unsigned)spec_rounds), threads, sp_smem, st>>>(P);
        ODB_LAUNCH_CHECK(c);
        k_spec_commit<<<dim3((unsigned)R, (unsigned)spec_rounds), std::max(host_active_keys(c->prm.buffer_size) / kMsItems, 128), 0, st>>>(P);
        ODB_LAUNCH_CHECK(c);
        A.sort.first = 0;
        A.spec = P.rec;
    }
    void *args[] = {(void *)&A};
    e = cudaLaunchCooperativeKernel((const void *)k_rounds, dim3((unsigned)R), dim3(kMsThreads), args, smem, st);
    if (e != cudaSuccess) return e;
    c->launches++;
    c->sorted = c->keyA;
    return cudaSuccess;
}

// distributed mode, first half: the local windows of the rounds [0, n_rounds) and their G table ([round][rank])
cudaError_t launch_dist_spec_form(odb_ctx *c, int n_rounds, int32_t **G_tab_out, cudaStream_t st) {
    SpecArgs P;
    int threads = 0;
    size_t sp_smem = 0;
    cudaError_t e = make_spec_args(c, n_rounds, 0, 1, st, &P, &threads, &sp_smem);
    if (e != cudaSuccess) return e;
    if (spec_items(c) == 8) k_spec_form<8><<<dim3((unsigned)c->prm.n_ranks, (unsigned)n_rounds), threads, sp_smem, st>>>(P);
    else k_spec_form<4><<<dim3((unsigned)c->prm.n_ranks, (unsigned)n_rounds), threads, sp_smem, st>>>(P);
    ODB_LAUNCH_CHECK(c);
    *G_tab_out = P.G_tab;
    c->sorted = c->keyA;
    return cudaSuccess;
}

// ... second half, behind the all_gather: Eq. 3 for every round on the gathered tables, split + commit of the
// local ranks' rounds before j*, the rank state for round j*
cudaError_t launch_dist_spec_commit(odb_ctx *c, int n_rounds, const int32_t *d_G_world, const int32_t *d_n_world, int n_procs,
                                    cudaStream_t st) {
    SpecArgs P;
    int threads = 0;
    size_t sp_smem = 0;
    cudaError_t e = make_spec_args(c, n_rounds, 0, 1, st, &P, &threads, &sp_smem);
    if (e != cudaSuccess) return e;
    const int R = c->prm.n_ranks;
    k_spec_T_world<<<1, 1024, 0, st>>>(d_G_world, d_n_world, n_procs, R, n_rounds, c->prm.buffer_size, c->prm.slot_capacity,
                                        P.T_tab, P.sb_tab, P.rec);
    ODB_LAUNCH_CHECK(c);
    k_spec_commit<<<dim3((unsigned)R, (unsigned)n_rounds), std::max(host_active_keys(c->prm.buffer_size) / kMsItems, 128), 0, st>>>(P);
    ODB_LAUNCH_CHECK(c);
    k_spec_state<<<(R + 127) / 128, 128, 0, st>>>(P.rec, c->d_rank_ptr, R, c->prm.buffer_size, c->n_left, c->fetch_pos,
                                                   c->emit_cur);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

// A9.  `slots_bound` >= the number of slots the plan can hold (the host may not have seen the plan yet);
// the grid is persistent: tiles are taken by ticket.
cudaError_t launch_finalize(odb_ctx *c, int64_t slots_bound, const CapCheck &cap, int64_t *rank_off, cudaStream_t st,
                            int64_t step_lo, int64_t slots_alloc) {
    const int R = c->prm.n_ranks;
    const int64_t so = step_lo * R;  // the staging tables are step-major: a step range is a contiguous piece
    const int64_t n_tiles = std::max<int64_t>((slots_bound + kFinTile - 1) / kFinTile, 1);
    // [0, 64): ticket + exit counter (rewound by the kernel's last CTA); then the tile states, whose flags carry the
    // launch's epoch, so nothing has to be cleared between launches (zeroed once, when the buffer grows)
    const int64_t tiles_alloc = std::max<int64_t>(n_tiles, (slots_alloc + kFinTile - 1) / kFinTile);
    cudaError_t e = c->scan_state.ensure((size_t)tiles_alloc * sizeof(ScanTile) + 64, true, st);
    if (e != cudaSuccess) return e;
    c->fin_epoch = (c->fin_epoch % 0x1ffffffe) + 1;  // 1 .. 2^29 - 1
    const int blocks = (int)std::min<int64_t>(n_tiles, (int64_t)c->sm_count * 2);
    k_fin_scan<<<blocks, kFinThreads, 0, st>>>(R, c->d_dims, c->st_count.p + so, c->st_width.p + so, c->st_real.p + so,
                                               c->st_round.p + so, c->st_origin.p + so, c->grp_count.p, c->grp_width.p, c->grp_round.p,
                                               c->grp_real.p, c->grp_origin.p, c->grp_offset.p, c->grp_sample_ptr.p,
                                               reinterpret_cast<ScanTile *>(c->scan_state.p + 64),
                                               reinterpret_cast<unsigned int *>(c->scan_state.p), cap,
                                               (c->offline || c->sub_mode) ? (int64_t)-1 : c->n_total, rank_off, c->h_dims, c->fin_epoch,
                                               (c->sub_mode || c->offline) ? nullptr : c->d_rec);
    if (!c->sub_mode && !c->offline) c->rec_clear_stream = st;  // (the host marks the record clean once it knows the plan was complete)
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

// ---------------------------------------------------------------------------------------------
// Step-range plans (odb_collate_steps): the steps [step_lo, step_lo + n) of the plan so far as a self-contained
// plan.  The slot scan above runs on that piece of the staging tables; what is left is the slot CSR's ids:
// a rank's slots are in emit order, so the rows of its steps [step_lo, ..) are the piece of its emit region
// that starts behind the samples of its earlier steps.
// ---------------------------------------------------------------------------------------------
__global__ void k_sub_dims(PlanDims *dims, int n_steps) {
    dims->n_steps = n_steps;
    dims->n_rounds = 0;
    dims->stop_reason = 0;
    dims->complete = 1;
    dims->err = 0;
    dims->bad_length = 0;
}

cudaError_t launch_sub_dims(odb_ctx *c, int n_steps, cudaStream_t st) {
    k_sub_dims<<<1, 1, 0, st>>>(c->d_dims, n_steps);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

__global__ void __launch_bounds__(1024)
k_sub_ids(const PlanDims *dims, int R, int step_lo, const int32_t *__restrict__ st_count, const int64_t *__restrict__ rank_ptr,
          const int32_t *__restrict__ emit_ids, const int64_t *__restrict__ grp_sample_ptr, int32_t *__restrict__ ids,
          int32_t *__restrict__ user_ids, const int64_t *__restrict__ full_sp, int full_K) {
    __shared__ long long s_scan64[34];
    if (!dims->complete || dims->err) return;
    const int r = blockIdx.x, n = dims->n_steps;
    long long e_lo;  // samples of rank r in the steps before the range
    if (full_sp) {   // the full plan's slot CSR knows it
        e_lo = full_sp[(int64_t)r * full_K + step_lo] - full_sp[(int64_t)r * full_K];
    } else {         // between rounds: sum the staging table's column
        long long part = 0;
        for (int k = threadIdx.x; k < step_lo; k += blockDim.x) part += st_count[(int64_t)k * R + r];
        (void)block_excl_scan<long long>(part, s_scan64, e_lo);
    }
    const int64_t base = rank_ptr[r];
    const int64_t q0 = grp_sample_ptr[(int64_t)r * n], q1 = grp_sample_ptr[(int64_t)(r + 1) * n];
    for (int64_t i = threadIdx.x; i < q1 - q0; i += blockDim.x) {
        const int32_t lid = emit_ids[base + e_lo + i];
        ids[q0 + i] = (int32_t)(base + lid);
        if (user_ids) user_ids[q0 + i] = lid;
    }
}

cudaError_t launch_sub_ids(odb_ctx *c, int step_lo, int32_t *user_ids, const int64_t *full_sp, int full_K, cudaStream_t st) {
    k_sub_ids<<<c->prm.n_ranks, 1024, 0, st>>>(c->d_dims, c->prm.n_ranks, step_lo, c->st_count.p, c->d_rank_ptr, c->emit_ids,
                                              c->grp_sample_ptr.p, c->grp_sample_ids.p, user_ids, full_sp, full_K);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

}  // namespace odb
