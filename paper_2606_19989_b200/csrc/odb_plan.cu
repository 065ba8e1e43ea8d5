// Planning kernels of the ODB hot path (rows A0..A9 of DESIGN.md): window fill + segmented sort,
// greedy successor, pointer-jumping list ranking, cross-rank reduction, split / overflow, step
// totals + quota cut, round commit, and the rank-major plan tables.  sm_100a only.
//
// Paper: /root/reference/PAPER.md (P:<line>).  Section 2.2 P:32-36 and Eq. 1 (grouping), Eq. 3
// (target), Alg. 1 P:258-279 (split / overflow), P:28 (IDLE slots), Thm 2 P:48 + P:347 (quota).
#include "odb_internal.cuh"

namespace odb {

// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t key_len(uint64_t k) { return (uint32_t)(k >> 32); }
__device__ __forceinline__ int32_t key_id(uint64_t k) { return (int32_t)(uint32_t)(k & 0xffffffffull); }

template <class V>
__device__ __forceinline__ V warp_incl_scan(V v) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        V n = __shfl_up_sync(ODB_FULL_MASK, v, d);
        if (lane >= d) v += n;
    }
    return v;
}

// Exclusive scan of one value per thread over the CTA.  `s` is shared scratch of 34 V's.
// Returns the exclusive prefix; `total` receives the CTA-wide sum.  Contains barriers: every
// thread of the CTA must call it.
template <class V>
__device__ __forceinline__ V block_excl_scan(V v, V *s, V &total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    V inc = warp_incl_scan(v);
    if (lane == 31) s[w] = inc;
    __syncthreads();
    if (w == 0) {
        V x = lane < nw ? s[lane] : (V)0;
        V xi = warp_incl_scan(x);
        s[lane] = xi - x;
        if (lane == 31) s[32] = xi;
    }
    __syncthreads();
    V r = inc - v + s[w];
    total = s[32];
    __syncthreads();
    return r;
}

// Stream compaction over i in [0, n): emit(i, k) for the k-th i with pred(i).  Returns the count.
template <class Pred, class Emit>
__device__ __forceinline__ int block_compact(int n, int *s, Pred pred, Emit emit) {
    int carry = 0;
    for (int base = 0; base < n; base += blockDim.x) {
        int i = base + threadIdx.x;
        int f = (i < n && pred(i)) ? 1 : 0;
        int tot;
        int ex = block_excl_scan<int>(f, s, tot);
        if (f) emit(i, carry + ex);
        carry += tot;
    }
    return carry;
}

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
__device__ __forceinline__ int window_size(int n_left, int fetch_pos, int n_r, int buffer_size) {
    long long avail = (long long)n_left + (long long)(n_r - fetch_pos);
    if (buffer_size > 0 && avail > buffer_size) avail = buffer_size;
    return (int)avail;
}

// ---------------------------------------------------------------------------------------------
// length validation (len >= 1), once per run
// ---------------------------------------------------------------------------------------------
__global__ void k_validate_lengths(const int32_t *__restrict__ len, int64_t n, RoundRec *rec) {
    int bad = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        if (len[i] < 1) bad = 1;
    if (__syncthreads_or(bad) && threadIdx.x == 0) rec->bad_length = 1;
}

// ---------------------------------------------------------------------------------------------
// A0 + A1a: fill the window and sort chunks of kSortChunk keys in shared memory.
// key = (len << 32) | local id, so ascending key order is the composite order (len, id) (U1).
// grid = (chunks of the largest possible window, R)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kSortThreads)
k_chunk_sort(const int32_t *__restrict__ len, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ n_left,
             const int32_t *__restrict__ fetch_pos, const int32_t *__restrict__ left_ids, int buffer_size,
             uint64_t *__restrict__ keys_out, int32_t *__restrict__ S_out) {
    __shared__ uint64_t sk[kSortChunk];
    const int r = blockIdx.y;
    const int64_t base = rank_ptr[r];
    const int n_r = (int)(rank_ptr[r + 1] - base);
    const int nl = n_left[r], fp = fetch_pos[r];
    const int S = window_size(nl, fp, n_r, buffer_size);
    if (blockIdx.x == 0 && threadIdx.x == 0) S_out[r] = S;
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

// A1b: one merge pass; runs of width w are merged pairwise.  Every element finds its output
// position by a binary search in the sibling run (keys are unique, so no tie handling).
__global__ void __launch_bounds__(kMergeThreads)
k_merge_pass(const uint64_t *__restrict__ src, uint64_t *__restrict__ dst, const int64_t *__restrict__ rank_ptr,
             const int32_t *__restrict__ S_arr, int w) {
    const int r = blockIdx.y;
    const int S = S_arr[r];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S) return;
    const uint64_t *s = src + rank_ptr[r];
    const long long run = i / w;
    const long long ps = (run & ~1ll) * (long long)w;
    const int mid = (int)min((long long)S, ps + w);
    const int end = (int)min((long long)S, ps + 2ll * w);
    const uint64_t key = s[i];
    int lo, hi;
    if (i < mid) {
        lo = mid;
        hi = end;
    } else {
        lo = (int)ps;
        hi = mid;
    }
    const int lo0 = lo;
    while (lo < hi) {  // lower bound of key in s[lo0, hi)
        int m = (lo + hi) >> 1;
        if (s[m] < key) lo = m + 1;
        else hi = m;
    }
    const int less = lo - lo0;
    const int pos = (i < mid) ? (i + less) : ((int)ps + (i - mid) + less);
    dst[rank_ptr[r] + pos] = key;
}

// ---------------------------------------------------------------------------------------------
// A2 + A3: successor array, pointer-jumping reachability from the head, candidate group starts.
// One CTA per rank.  Chase coordinate x in [0, S]:
//   THRESHOLD: x = position in the longest->shortest visit order; J[0] = 1 (t starts at 1),
//              J[x] = min(S, x + B(len(v[x-1]))), B from Eq. 1 (the group that starts at x closes
//              after B(l) samples, l = the last sample of the previous group).
//   MAXFIT:    x = ascending position; J[x] = largest e <= S with (e - x) * slen[e-1] <= L, >= x+1.
// Round p marks next^(k + 2^p)(0) for every marked next^k(0) and squares the jump array, so after
// ceil(log2 G) + 1 rounds exactly the orbit of 0 is marked.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kRankThreads)
k_form_groups(const uint64_t *__restrict__ keys, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ S_arr,
              long long budget, int rule, int32_t *jA, int32_t *jB, uint8_t *mark, uint8_t *__restrict__ flag,
              int32_t *__restrict__ gpos, int32_t *__restrict__ G_out) {
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
        int j;
        if (x == S) {
            j = S;
        } else if (rule == ODB_RULE_THRESHOLD) {
            if (x == 0) {
                j = 1;
            } else {
                long long l = (long long)key_len(k[S - x]);  // v[x-1] = ascending position S-1-(x-1)
                long long q = budget / (l > 0 ? l : 1);
                if (q < 1) q = 1;
                long long jj = (long long)x + q;
                j = (int)(jj < (long long)S ? jj : (long long)S);
            }
        } else {
            int lo = x + 1, hi = S;  // the singleton [x, x+1) is always accepted (U10)
            while (lo < hi) {
                int m = (lo + hi + 1) >> 1;
                if ((long long)(m - x) * (long long)key_len(k[m - 1]) <= budget) lo = m;
                else hi = m - 1;
            }
            j = lo;
        }
        cur[x] = j;
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
    // start flags in ascending coordinates; compact the start positions
    uint8_t *fl = flag + base;
    int32_t *gp = gpos + jb;
    int G = block_compact(
        S, s_scan,
        [&](int a) {
            bool f = (rule == ODB_RULE_THRESHOLD) ? (a == 0 || mk[S - a] != 0) : (mk[a] != 0);
            fl[a] = f ? 1 : 0;
            return f;
        },
        [&](int a, int kidx) { gp[kidx] = a; });
    if (threadIdx.x == 0) {
        gp[G] = S;
        G_out[r] = G;
    }
}

// ---------------------------------------------------------------------------------------------
// A4 + A5 + A6: T_grp (Eq. 3), split (the d rightmost non-start positions become starts, which is
// what Alg. 1's backward scan produces), overflow (sort groups by
// (count desc, index asc), keep the first T).  Output per rank: aligned groups in emit order as
// (agpos[k], agcnt[k]) over the sorted window, k < T.  Adds the counts into step_samples (A8a).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kRankThreads)
k_align(const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ S_arr, const int32_t *__restrict__ G_arr, int R,
        int slot_capacity, const uint8_t *__restrict__ flag, const int32_t *__restrict__ gpos, int32_t *__restrict__ agpos,
        int32_t *__restrict__ agcnt, uint64_t *ovf, int32_t *step_samples, int step_base, RoundRec *rec) {
    __shared__ int s_scan[34];
    __shared__ int s_maxG, s_minS;
    const int r = blockIdx.x;
    if (threadIdx.x == 0) {
        s_maxG = 0;
        s_minS = 0x7fffffff;
    }
    __syncthreads();
    for (int q = threadIdx.x; q < R; q += blockDim.x) {
        int g = G_arr[q];
        if (g > 0) {  // active set A = {r : G_r > 0}
            atomicMax(&s_maxG, g);
            int sq = S_arr[q];
            if (sq > 0) atomicMin(&s_minS, sq);
        }
    }
    __syncthreads();
    int T = s_maxG;
    if (slot_capacity > 0 && T > slot_capacity) T = slot_capacity;  // C+min (same C on every rank)
    if (T > s_minS) T = s_minS;                                     // S+min
    if (T < 1) T = 1;
    if (r == 0 && threadIdx.x == 0) rec->T = T;
    const int Gr = G_arr[r];
    if (Gr == 0) return;  // finished rank: IDLE slots are written by the commit kernel
    const int S = S_arr[r];
    const int64_t base = rank_ptr[r];
    const int64_t jb = base + r;
    const int32_t *gp = gpos + jb;
    int32_t *ap = agpos + jb, *ac = agcnt + jb;
    if (Gr <= T) {
        const int d = T - Gr;
        const uint8_t *fl = flag + base;
        int carry_old = 0, carry_new = 0;
        for (int b0 = 0; b0 < S; b0 += blockDim.x) {
            int a = b0 + threadIdx.x;
            int f = (a < S) ? fl[a] : 0;
            int tot_old, tot_new;
            int ex_old = block_excl_scan<int>(f, s_scan, tot_old) + carry_old;
            int nf = 0;
            if (a < S) {
                int nonstarts_right = (S - a) - (Gr - ex_old);  // non-start positions in [a, S)
                nf = (f || nonstarts_right <= d) ? 1 : 0;
            }
            int ex_new = block_excl_scan<int>(nf, s_scan, tot_new) + carry_new;
            if (nf) ap[ex_new] = a;
            carry_old += tot_old;
            carry_new += tot_new;
        }
        if (threadIdx.x == 0) ap[T] = S;
        __syncthreads();
        for (int k = threadIdx.x; k < T; k += blockDim.x) {
            int c = ap[k + 1] - ap[k];
            ac[k] = c;
            atomicAdd(&step_samples[step_base + k], c);
        }
    } else {
        uint64_t *ok = ovf + 2 * base;
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
            atomicAdd(&step_samples[step_base + k], c);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// A7 + A8a: commit the round.  Finds the quota cut k* (non-join), writes the step-major staging
// tables, appends the emitted ids to the rank's emit region, compacts the leftovers, advances the
// rank state and counts the ranks that will be finished next round.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kRankThreads)
k_commit(const uint64_t *__restrict__ keys, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ S_arr,
         const int32_t *__restrict__ G_arr, int R, const int32_t *__restrict__ agpos, const int32_t *__restrict__ agcnt,
         int32_t *__restrict__ agoff, const int32_t *__restrict__ step_samples, int step_base, int round, int join_mode,
         long long quota, long long emitted_before, int32_t *__restrict__ st_count, int32_t *__restrict__ st_width,
         int32_t *__restrict__ st_idoff, int32_t *__restrict__ st_round, uint8_t *__restrict__ posflag,
         int32_t *__restrict__ emit_ids, uint8_t *__restrict__ emitted, int32_t *__restrict__ left_ids, int32_t *n_left,
         int32_t *fetch_pos, int32_t *emit_cur, RoundRec *rec) {
    __shared__ int s_scan[34];
    __shared__ long long s_scan64[34];
    __shared__ int s_found;
    const int r = blockIdx.x;
    const int T = rec->T;
    int T_emit = T, quota_hit = 0;
    if (!join_mode && quota > 0) {
        if (threadIdx.x == 0) s_found = 0x7fffffff;
        __syncthreads();
        long long carry = 0;
        for (int b0 = 0; b0 < T; b0 += blockDim.x) {
            int k = b0 + threadIdx.x;
            long long v = (k < T) ? (long long)step_samples[step_base + k] : 0ll;
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
    if (r == 0) {  // round totals for the host
        long long part = 0;
        for (int k = threadIdx.x; k < T_emit; k += blockDim.x) part += step_samples[step_base + k];
        long long tot;
        (void)block_excl_scan<long long>(part, s_scan64, tot);
        if (threadIdx.x == 0) {
            rec->T_emit = T_emit;
            rec->quota_hit = quota_hit;
            rec->emitted_round = tot;
        }
    }
    const int Gr = G_arr[r];
    const int S = S_arr[r];
    const int64_t base = rank_ptr[r];
    const int n_r = (int)(rank_ptr[r + 1] - base);
    if (Gr == 0) {  // finished rank: IDLE slots (U14)
        for (int k = threadIdx.x; k < T_emit; k += blockDim.x) {
            int64_t idx = (int64_t)(step_base + k) * R + r;
            st_count[idx] = 0;
            st_width[idx] = 0;
            st_idoff[idx] = 0;
            st_round[idx] = round;
        }
        if (threadIdx.x == 0) atomicAdd(&rec->n_finished, 1);
        return;
    }
    const int64_t jb = base + r;
    const uint64_t *k_ = keys + base;
    const int32_t *ap = agpos + jb, *ac = agcnt + jb;
    int32_t *ao = agoff + jb;
    uint8_t *pf = posflag + base;
    const int cur = emit_cur[r];
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
            st_width[idx] = (int32_t)key_len(k_[p + c - 1]);  // rows ascending: the last row is the longest
            st_idoff[idx] = cur + ex;
            st_round[idx] = round;
            ao[k] = cur + ex;
        }
        carry += tot;
    }
    const int emitted_r = carry;
    __syncthreads();
    {  // copy ids: one warp per group
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
        for (int k = w; k < T_emit; k += nw) {
            int p = ap[k], c = ac[k], o = ao[k];
            for (int j = lane; j < c; j += 32) {
                int id = key_id(k_[p + j]);
                emit_ids[base + o + j] = id;
                emitted[base + id] = 1;
                pf[p + j] = 1;
            }
        }
    }
    __syncthreads();
    int32_t *lf = left_ids + base;
    int n_left_new = block_compact(
        S, s_scan, [&](int a) { return pf[a] == 0; }, [&](int a, int kidx) { lf[kidx] = key_id(k_[a]); });
    if (threadIdx.x == 0) {
        int nl_old = n_left[r], fp = fetch_pos[r];
        int fp_new = fp + (S - nl_old);
        emit_cur[r] = cur + emitted_r;
        n_left[r] = n_left_new;
        fetch_pos[r] = fp_new;
        if (n_left_new + (n_r - fp_new) == 0) atomicAdd(&rec->n_finished, 1);
    }
}

// ---------------------------------------------------------------------------------------------
// A9 and the rank-major plan tables
// ---------------------------------------------------------------------------------------------
__global__ void k_fin_slots(int R, int n_steps, const int32_t *__restrict__ st_count, const int32_t *__restrict__ st_width,
                            const int32_t *__restrict__ st_idoff, const int32_t *__restrict__ st_round,
                            int32_t *__restrict__ grp_count, int32_t *__restrict__ grp_width, int32_t *__restrict__ grp_round,
                            int32_t *__restrict__ grp_idoff, int64_t *__restrict__ grp_offset,
                            int64_t *__restrict__ grp_sample_ptr) {
    const int64_t n_slots = (int64_t)R * n_steps;
    for (int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; s < n_slots; s += (int64_t)gridDim.x * blockDim.x) {
        int r = (int)(s / n_steps);
        int k = (int)(s - (int64_t)r * n_steps);
        int64_t src = (int64_t)k * R + r;
        int c = st_count[src], w = st_width[src];
        grp_count[s] = c;
        grp_width[s] = w;
        grp_round[s] = st_round[src];
        grp_idoff[s] = st_idoff[src];
        int64_t area = (int64_t)c * (int64_t)w;
        grp_offset[s] = (area + 15) / 16 * 16;  // scanned in place by k_scan_slots
        grp_sample_ptr[s] = c;
    }
}

// In-place exclusive scans of grp_offset and grp_sample_ptr (n + 1 entries each) by one CTA, and the
// sum of count*width.  8 consecutive items per thread per iteration.
__global__ void __launch_bounds__(1024)
k_scan_slots(int64_t n, int64_t *grp_offset, int64_t *grp_sample_ptr, const int32_t *__restrict__ grp_count,
             const int32_t *__restrict__ grp_width, PlanTotals *tot) {
    __shared__ long long s_scan64[34];
    constexpr int ITEMS = 8;
    long long carry_o = 0, carry_p = 0, area_sum = 0;
    for (int64_t b0 = 0; b0 < n; b0 += (int64_t)blockDim.x * ITEMS) {
        int64_t i0 = b0 + (int64_t)threadIdx.x * ITEMS;
        long long vo[ITEMS], vp[ITEMS];
        long long so = 0, sp = 0;
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            int64_t i = i0 + j;
            vo[j] = (i < n) ? grp_offset[i] : 0;
            vp[j] = (i < n) ? grp_sample_ptr[i] : 0;
            if (i < n) area_sum += (long long)grp_count[i] * (long long)grp_width[i];
            so += vo[j];
            sp += vp[j];
        }
        long long to, tp;
        long long eo = block_excl_scan<long long>(so, s_scan64, to) + carry_o;
        long long ep = block_excl_scan<long long>(sp, s_scan64, tp) + carry_p;
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            int64_t i = i0 + j;
            if (i < n) {
                grp_offset[i] = eo;
                grp_sample_ptr[i] = ep;
            }
            eo += vo[j];
            ep += vp[j];
        }
        carry_o += to;
        carry_p += tp;
    }
    long long ta;
    (void)block_excl_scan<long long>(area_sum, s_scan64, ta);
    if (threadIdx.x == 0) {
        grp_offset[n] = carry_o;
        grp_sample_ptr[n] = carry_p;
        tot->total_elems = carry_o;
        tot->samples_emitted = carry_p;
        tot->padded_elems = ta;
    }
}

// One warp per slot: gather the slot's sample ids in row order and sum their lengths.
__global__ void k_gather_ids(int R, int n_steps, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ len,
                             const int32_t *__restrict__ emit_ids, const int32_t *__restrict__ grp_idoff,
                             const int32_t *__restrict__ grp_count, const int64_t *__restrict__ grp_sample_ptr,
                             int32_t *__restrict__ grp_sample_ids, int32_t *__restrict__ grp_real, PlanTotals *tot) {
    const int lane = threadIdx.x & 31;
    const int64_t n_slots = (int64_t)R * n_steps;
    const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    unsigned long long local = 0;
    for (int64_t s = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; s < n_slots; s += warps) {
        int r = (int)(s / n_steps);
        int64_t base = rank_ptr[r];
        int c = grp_count[s];
        int o = grp_idoff[s];
        int64_t q0 = grp_sample_ptr[s];
        long long sum = 0;
        for (int j = lane; j < c; j += 32) {
            int id = emit_ids[base + o + j];
            grp_sample_ids[q0 + j] = id;
            sum += len[base + id];
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(ODB_FULL_MASK, sum, d);
        if (lane == 0) {
            grp_real[s] = (int32_t)sum;
            local += (unsigned long long)sum;
        }
    }
    if (lane == 0 && local) atomicAdd(&tot->real_tokens, local);
}

// Un-emitted local ids per rank, ascending (Lemma 1: buffer + sampler-pending).
__global__ void __launch_bounds__(kRankThreads)
k_leftovers(int R, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ emit_cur,
            const uint8_t *__restrict__ emitted, int64_t *__restrict__ left_ptr, int32_t *__restrict__ left_out,
            PlanTotals *tot) {
    __shared__ int s_scan[34];
    __shared__ long long s_scan64[34];
    const int r = blockIdx.x;
    long long part = 0;
    for (int q = threadIdx.x; q < r; q += blockDim.x) part += (rank_ptr[q + 1] - rank_ptr[q]) - emit_cur[q];
    long long lbase;
    (void)block_excl_scan<long long>(part, s_scan64, lbase);
    const int64_t base = rank_ptr[r];
    const int n_r = (int)(rank_ptr[r + 1] - base);
    const uint8_t *em = emitted + base;
    int32_t *out = left_out + lbase;
    int cnt = block_compact(
        n_r, s_scan, [&](int i) { return em[i] == 0; }, [&](int i, int kidx) { out[kidx] = i; });
    if (threadIdx.x == 0) {
        left_ptr[r] = lbase;
        if (r == R - 1) {
            left_ptr[R] = lbase + cnt;
            tot->samples_left = lbase + cnt;
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

cudaError_t launch_validate_lengths(odb_ctx *c, cudaStream_t st) {
    if (c->n_total == 0) return cudaSuccess;
    int blocks = (int)std::min<int64_t>((c->n_total + 1023) / 1024, (int64_t)c->sm_count * 4);
    k_validate_lengths<<<blocks, 256, 0, st>>>(c->d_lengths, c->n_total, c->d_rec);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

static int max_window_bound(const odb_ctx *c) {
    int64_t m = c->max_nr;
    if (c->prm.buffer_size > 0 && m > c->prm.buffer_size) m = c->prm.buffer_size;
    return (int)m;
}

cudaError_t launch_round_form(odb_ctx *c, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    const int maxS = max_window_bound(c);
    if (maxS == 0) return cudaSuccess;
    const int chunks = (maxS + kSortChunk - 1) / kSortChunk;
    k_chunk_sort<<<dim3(chunks, R), kSortThreads, 0, st>>>(c->d_lengths, c->d_rank_ptr, c->n_left, c->fetch_pos, c->left_ids,
                                                          c->prm.buffer_size, c->keyA, c->S);
    ODB_LAUNCH_CHECK(c);
    uint64_t *src = c->keyA, *dst = c->keyB;
    for (int64_t w = kSortChunk; w < maxS; w *= 2) {
        int gx = (maxS + kMergeThreads - 1) / kMergeThreads;
        k_merge_pass<<<dim3(gx, R), kMergeThreads, 0, st>>>(src, dst, c->d_rank_ptr, c->S, (int)w);
        ODB_LAUNCH_CHECK(c);
        uint64_t *t = src;
        src = dst;
        dst = t;
    }
    c->sorted = src;
    k_form_groups<<<R, kRankThreads, 0, st>>>(c->sorted, c->d_rank_ptr, c->S, (long long)c->prm.budget, c->prm.rule, c->jA,
                                              c->jB, c->mark, c->flag, c->gpos, c->G);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

cudaError_t launch_round_align(odb_ctx *c, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    k_align<<<R, kRankThreads, 0, st>>>(c->d_rank_ptr, c->S, c->G, R, c->prm.slot_capacity, c->flag, c->gpos, c->agpos,
                                        c->agcnt, c->ovf, c->step_samples.p, c->n_steps, c->d_rec);
    ODB_LAUNCH_CHECK(c);
    k_commit<<<R, kRankThreads, 0, st>>>(c->sorted, c->d_rank_ptr, c->S, c->G, R, c->agpos, c->agcnt, c->agoff,
                                         c->step_samples.p, c->n_steps, c->round, c->prm.join_mode,
                                         (long long)c->prm.sample_quota,
                                         (long long)c->prm.emitted_so_far + (long long)c->samples_emitted, c->st_count.p,
                                         c->st_width.p, c->st_idoff.p, c->st_round.p, c->posflag, c->emit_ids, c->emitted,
                                         c->left_ids, c->n_left, c->fetch_pos, c->emit_cur, c->d_rec);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

cudaError_t launch_finalize(odb_ctx *c, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    const int64_t n_slots = (int64_t)R * c->n_steps;
    cudaError_t e = cudaMemsetAsync(c->d_tot, 0, sizeof(PlanTotals), st);
    if (e != cudaSuccess) return e;
    if (n_slots > 0) {
        int blocks = (int)std::min<int64_t>((n_slots + 255) / 256, (int64_t)c->sm_count * 8);
        k_fin_slots<<<blocks, 256, 0, st>>>(R, c->n_steps, c->st_count.p, c->st_width.p, c->st_idoff.p, c->st_round.p,
                                            c->grp_count.p, c->grp_width.p, c->grp_round.p, c->grp_idoff.p,
                                            c->grp_offset.p, c->grp_sample_ptr.p);
        ODB_LAUNCH_CHECK(c);
    }
    k_scan_slots<<<1, 1024, 0, st>>>(n_slots, c->grp_offset.p, c->grp_sample_ptr.p, c->grp_count.p, c->grp_width.p,
                                     c->d_tot);
    ODB_LAUNCH_CHECK(c);
    if (n_slots > 0) {
        int blocks = (int)std::min<int64_t>((n_slots * 32 + 255) / 256, (int64_t)c->sm_count * 8);
        k_gather_ids<<<blocks, 256, 0, st>>>(R, c->n_steps, c->d_rank_ptr, c->d_lengths, c->emit_ids, c->grp_idoff.p,
                                             c->grp_count.p, c->grp_sample_ptr.p, c->grp_sample_ids.p, c->grp_real.p,
                                             c->d_tot);
        ODB_LAUNCH_CHECK(c);
    }
    k_leftovers<<<R, kRankThreads, 0, st>>>(R, c->d_rank_ptr, c->emit_cur, c->emitted, c->left_ptr.p, c->left_out.p,
                                            c->d_tot);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

}  // namespace odb
