// the paper's OFFLINE comparators as planners -- GMT and BMT (App. I: global /
// bucketed max-token batchers on padded area, wrap-around repetition of the leading batches, rank striding) and
// HFG (App. J: megabatch length grouping with a fixed batch size, stride-sharded).  Index work only:
// they reuse the segmented sort (segments = the whole pool, the buckets, the megabatches), the padded-area
// successor + list ranking (MAXFIT_ASC), the slot scan and the collate path; what is new here is the map from
// the global batch list / index list to the rank-major slots.  A slot's ids are GLOBAL sample ids.
// Random draws (the epoch shuffle, the batch-shuffle keys) are inputs.  sm_100a only.
#include <cstring>

#include "odb_device.cuh"
#include "odb_internal.cuh"
#include "odb_sort.cuh"

namespace odb {

#define ODB_LAUNCH_CHECK(c)                       \
    do {                                          \
        (c)->launches++;                          \
        cudaError_t e_ = cudaGetLastError();      \
        if (e_ != cudaSuccess) return e_;         \
    } while (0)

__device__ __forceinline__ uint32_t of_len(uint64_t k) { return (uint32_t)(k >> 32); }
__device__ __forceinline__ int32_t of_id(uint64_t k) { return (int32_t)(uint32_t)(k & 0xffffffffull); }

// lengths in list order (the shuffled order for BMT / HFG), validated; segment tables
__global__ void k_of_gather(const int32_t *__restrict__ len, const int32_t *__restrict__ perm, int64_t N,
                            int32_t *__restrict__ plen, RoundRec *rec) {
    int bad = 0;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < N; p += (int64_t)gridDim.x * blockDim.x) {
        const int32_t l = len[perm ? perm[p] : p];
        plen[p] = l;
        if (l < 1) bad = 1;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) rec->bad_length = 1;
}

__global__ void k_of_segments(int64_t N, int64_t size, int64_t nseg, int64_t *__restrict__ seg_ptr, int32_t *__restrict__ tab) {
    for (int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; s <= nseg; s += (int64_t)gridDim.x * blockDim.x) {
        seg_ptr[s] = min(N, s * size);
        if (s < nseg) {
            tab[s] = 0;                      // n_left
            tab[nseg + s] = 0;               // fetch_pos
            tab[2 * nseg + s] = 0;           // emit_cur
            tab[3 * nseg + s] = 0x7fffffff;  // every view has arrived
        }
    }
}

// exclusive scan of the per-segment batch counts (one CTA; nseg <= N)
__global__ void __launch_bounds__(1024) k_of_scan(const int32_t *__restrict__ G, int64_t nseg, int32_t *__restrict__ boff) {
    __shared__ long long s_scan[34];
    long long carry = 0;
    for (int64_t b0 = 0; b0 < nseg; b0 += blockDim.x) {
        const int64_t s = b0 + threadIdx.x;
        const long long v = s < nseg ? G[s] : 0;
        long long tot;
        const long long ex = block_excl_scan<long long>(v, s_scan, tot);
        if (s < nseg) boff[s] = (int32_t)(carry + ex);
        carry += tot;
    }
    if (threadIdx.x == 0) boff[nseg] = (int32_t)carry;
}

// the flat batch table: first position in the sorted keys and sample count of every batch (a warp per segment)
__global__ void k_of_batches(int64_t nseg, const int64_t *__restrict__ seg_ptr, const int32_t *__restrict__ G,
                             const int32_t *__restrict__ boff, const int32_t *__restrict__ gpos,
                             int32_t *__restrict__ bstart, int32_t *__restrict__ bcnt) {
    const int lane = threadIdx.x & 31;
    const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; s < nseg; s += warps) {
        const int64_t base = seg_ptr[s];
        const int32_t *gp = gpos + base + s;
        const int g = G[s], b0 = boff[s];
        for (int i = lane; i < g; i += 32) {
            const int p = gp[i];
            bstart[b0 + i] = (int32_t)(base + p);
            bcnt[b0 + i] = gp[i + 1] - p;
        }
    }
}

struct OfflineMap {  // what a slot is made of
    int planner, W, size, bs;
    int64_t N, G, n_per;
    const uint64_t *sorted;
    const int32_t *perm, *bstart, *bcnt, *border;
};

// row i of slot (r, k): position of its key in `sorted` and the base of that key's segment
__device__ __forceinline__ void of_slot_range(const OfflineMap &M, int r, int k, int &cnt, int64_t &p0) {
    if (M.planner == ODB_PLANNER_HFG) {
        const int64_t i0 = (int64_t)k * M.bs;
        cnt = (int)max((int64_t)0, min((int64_t)M.bs, M.n_per - i0));
        p0 = i0;
    } else {
        int64_t j = ((int64_t)k * M.W + r) % M.G;  // wrap-around repetition of the leading batches, rank striding
        if (M.border) j = M.border[j];             // BMT: the batch shuffle
        cnt = M.bcnt[j];
        p0 = M.bstart[j];
    }
}
__device__ __forceinline__ int64_t of_row_pos(const OfflineMap &M, int r, int64_t p0, int i, int64_t &seg_base) {
    if (M.planner == ODB_PLANNER_HFG) {
        const int64_t t = ((p0 + i) * M.W + r) % M.N;  // the index list padded with its leading entries, stride-sharded
        seg_base = (t / M.size) * M.size;
        const int64_t n = min((int64_t)M.size, M.N - seg_base);
        return seg_base + (n - 1 - (t - seg_base));  // descending: the ascending order read backwards
    }
    seg_base = ((p0 + i) / M.size) * M.size;
    return p0 + i;
}

// step-major staging tables of every slot (a warp per slot) + the step totals
__global__ void k_of_slots(const OfflineMap M, int n_steps, int32_t *__restrict__ st_count, int32_t *__restrict__ st_width,
                           int32_t *__restrict__ st_real, int32_t *__restrict__ st_round, int32_t *__restrict__ st_origin,
                           int32_t *step_samples) {
    const int lane = threadIdx.x & 31;
    const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5, n_slots = (int64_t)M.W * n_steps;
    for (int64_t q = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; q < n_slots; q += warps) {
        const int k = (int)(q / M.W), r = (int)(q - (int64_t)k * M.W);
        int cnt;
        int64_t p0;
        of_slot_range(M, r, k, cnt, p0);
        uint32_t mx = 0, sum = 0;
        for (int i = lane; i < cnt; i += 32) {
            int64_t sb;
            const uint32_t l = of_len(M.sorted[of_row_pos(M, r, p0, i, sb)]);
            mx = max(mx, l);
            sum += l;
        }
        mx = __reduce_max_sync(ODB_FULL_MASK, mx);
        sum = __reduce_add_sync(ODB_FULL_MASK, sum);
        if (lane == 0) {
            const int64_t idx = (int64_t)k * M.W + r;
            st_count[idx] = cnt;
            st_width[idx] = (int32_t)mx;  // pad to the longest sample of the slot
            st_real[idx] = (int32_t)sum;
            st_round[idx] = 0;
            st_origin[idx] = k;
            atomicAdd(&step_samples[k], cnt);
        }
    }
}

// the slot CSR's ids (GLOBAL sample ids, row order), after the slot scan
__global__ void k_of_ids(const OfflineMap M, int n_steps, const int64_t *__restrict__ grp_sample_ptr,
                         int32_t *__restrict__ ids) {
    const int lane = threadIdx.x & 31;
    const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5, n_slots = (int64_t)M.W * n_steps;
    for (int64_t s = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; s < n_slots; s += warps) {
        const int r = (int)(s / n_steps), k = (int)(s - (int64_t)r * n_steps);
        int cnt;
        int64_t p0;
        of_slot_range(M, r, k, cnt, p0);
        const int64_t q0 = grp_sample_ptr[s];
        for (int i = lane; i < cnt; i += 32) {
            int64_t sb;
            const int64_t pos = of_row_pos(M, r, p0, i, sb);
            const int64_t list_pos = sb + of_id(M.sorted[pos]);  // the key's id is its position inside its segment
            ids[q0 + i] = M.perm ? M.perm[list_pos] : (int32_t)list_pos;
        }
    }
}

__global__ void k_of_border(const uint64_t *__restrict__ sorted, int64_t G, int32_t *__restrict__ border) {
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < G; t += (int64_t)gridDim.x * blockDim.x)
        border[t] = of_id(sorted[t]);
}

static OfflineMap make_map(const odb_ctx *c) {
    OfflineMap M;
    memset(&M, 0, sizeof(M));
    M.planner = c->offline_planner;
    M.W = c->prm.n_ranks;
    M.size = c->offline_size;
    M.bs = c->offline_bs;
    M.N = c->n_total;
    M.G = c->offline_G;
    M.n_per = (c->n_total + M.W - 1) / M.W;
    M.sorted = c->of_sorted;
    M.perm = c->offline_perm;
    M.bstart = c->of_bstart.p;
    M.bcnt = c->of_bcnt.p;
    M.border = c->offline_planner == ODB_PLANNER_BMT ? c->of_border.p : nullptr;
    return M;
}

cudaError_t launch_offline_ids(odb_ctx *c, cudaStream_t st) {
    const int64_t n_slots = (int64_t)c->prm.n_ranks * c->n_steps;
    if (n_slots == 0) return cudaSuccess;
    const int blocks = (int)std::min<int64_t>((n_slots * 32 + 255) / 256, (int64_t)c->sm_count * 16);
    k_of_ids<<<blocks, 256, 0, st>>>(make_map(c), c->n_steps, c->grp_sample_ptr.p, c->grp_sample_ids.p);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

#define OF_CU(expr)                          \
    do {                                     \
        cudaError_t e__ = (expr);            \
        if (e__ != cudaSuccess) return e__;  \
    } while (0)

// Builds the plan up to the step-major staging tables; *h_G receives the number of batches (GMT / BMT).
cudaError_t offline_build(odb_ctx *c, const odb_offline_params *P, const int32_t *d_lengths, int64_t N, cudaStream_t st) {
    const int64_t size = P->planner == ODB_PLANNER_GMT ? std::max<int64_t>(N, 1) : P->size;
    const int64_t nseg = N == 0 ? 0 : (N + size - 1) / size;
    const int maxS = (int)std::min<int64_t>(size, N);
    c->offline_size = (int)std::min<int64_t>(size, 0x7fffffff);
    OF_CU(cudaMemsetAsync(c->d_rec, 0, sizeof(RoundRec), st));
    OF_CU(c->of_plen.ensure((size_t)N + 1));
    OF_CU(c->of_seg_ptr.ensure((size_t)nseg + 2));
    OF_CU(c->of_seg_i32.ensure(7 * (size_t)nseg + 8));
    OF_CU(c->of_gpos.ensure((size_t)N + (size_t)nseg + 2));
    c->of_sorted = c->keyA;
    c->offline_G = 0;
    if (N == 0) return cudaSuccess;
    int32_t *tab = c->of_seg_i32.p;
    int32_t *S = tab + 4 * nseg, *G = tab + 5 * nseg, *boff = tab + 6 * nseg;
    {
        const int blocks = (int)std::min<int64_t>((N + 255) / 256, (int64_t)c->sm_count * 8);
        // (GMT works on the samples in their own order; BMT / HFG on the shuffled order)
        k_of_gather<<<blocks, 256, 0, st>>>(d_lengths, P->planner == ODB_PLANNER_GMT ? nullptr : P->d_perm, N, c->of_plen.p,
                                            c->d_rec);
        ODB_LAUNCH_CHECK(c);
        const int b2 = (int)std::min<int64_t>((nseg + 256) / 256, (int64_t)c->sm_count * 8);
        k_of_segments<<<b2, 256, 0, st>>>(N, size, nseg, c->of_seg_ptr.p, tab);
        ODB_LAUNCH_CHECK(c);
    }
    // segmented sort by (length, position inside the segment)
    SortArgs A;
    memset(&A, 0, sizeof(A));
    A.len = c->of_plen.p;
    A.rank_ptr = c->of_seg_ptr.p;
    A.n_left = tab;
    A.fetch_pos = tab + nseg;
    A.emit_cur = tab + 2 * nseg;
    A.left_ids = nullptr;
    A.arrived = tab + 3 * nseg;
    A.buffer_size = 0;
    A.keys_out = c->keyA;
    A.S_out = S;
    A.rec = c->d_rec;
    A.first = 0;
    OF_CU(sort_segments_any(c, A, nseg, maxS, c->keyB, &c->of_sorted, st));
    if (P->planner == ODB_PLANNER_HFG) return cudaSuccess;
    // greedy packing on padded area inside every segment, the flat batch table
    OF_CU(form_segments_maxfit(c, c->of_sorted, c->of_seg_ptr.p, S, nseg, maxS, c->jA, c->jB, c->mark, c->of_gpos.p, G, st));
    k_of_scan<<<1, 1024, 0, st>>>(G, nseg, boff);
    ODB_LAUNCH_CHECK(c);
    int32_t h_G = 0;
    OF_CU(cudaMemcpyAsync(&h_G, boff + nseg, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    OF_CU(cudaStreamSynchronize(st));  // an offline planner: the host sizes the batch tables
    c->offline_G = h_G;
    OF_CU(c->of_bstart.ensure((size_t)h_G + 1));
    OF_CU(c->of_bcnt.ensure((size_t)h_G + 1));
    {
        const int blocks = (int)std::min<int64_t>((nseg * 32 + 255) / 256, (int64_t)c->sm_count * 16);
        k_of_batches<<<blocks, 256, 0, st>>>(nseg, c->of_seg_ptr.p, G, boff, c->of_gpos.p, c->of_bstart.p, c->of_bcnt.p);
        ODB_LAUNCH_CHECK(c);
    }
    if (P->planner == ODB_PLANNER_BMT) {
        // batch shuffle: order the batches by (key of the batch index, batch index): one more sort, one segment
        OF_CU(c->of_border.ensure((size_t)h_G + 1));
        OF_CU(c->of_keyA.ensure((size_t)h_G + 1));
        OF_CU(c->of_keyB.ensure((size_t)h_G + 1));
        // (the bucket table is dead after k_of_batches: its first two entries become the one segment [0, G))
        const int64_t h_seg[2] = {0, h_G};
        int64_t *seg2 = c->of_seg_ptr.p;
        OF_CU(cudaMemcpyAsync(seg2, h_seg, sizeof(h_seg), cudaMemcpyHostToDevice, st));
        OF_CU(cudaStreamSynchronize(st));  // (h_seg lives on this stack frame)
        SortArgs B = A;
        B.len = P->d_shuffle_key;
        B.rank_ptr = seg2;
        B.keys_out = c->of_keyA.p;
        uint64_t *sorted2 = nullptr;
        OF_CU(sort_segments_any(c, B, 1, (int)h_G, c->of_keyB.p, &sorted2, st));
        const int blocks = (int)std::min<int64_t>((h_G + 255) / 256, (int64_t)c->sm_count * 8);
        k_of_border<<<std::max(blocks, 1), 256, 0, st>>>(sorted2, h_G, c->of_border.p);
        ODB_LAUNCH_CHECK(c);
    }
    return cudaSuccess;
}

cudaError_t offline_slots(odb_ctx *c, cudaStream_t st) {
    const int W = c->prm.n_ranks;
    const int64_t n_slots = (int64_t)W * c->n_steps;
    OF_CU(c->st_count.ensure((size_t)n_slots + 1));
    OF_CU(c->st_width.ensure((size_t)n_slots + 1));
    OF_CU(c->st_real.ensure((size_t)n_slots + 1));
    OF_CU(c->st_round.ensure((size_t)n_slots + 1));
    OF_CU(c->st_origin.ensure((size_t)n_slots + 1));
    OF_CU(c->step_samples.ensure((size_t)c->n_steps + 1));
    c->step_cap = std::min<int64_t>((int64_t)c->step_samples.cap, (int64_t)c->st_count.cap / std::max(W, 1));
    if (n_slots == 0) return cudaSuccess;
    OF_CU(cudaMemsetAsync(c->step_samples.p, 0, (size_t)c->n_steps * sizeof(int32_t), st));
    const int blocks = (int)std::min<int64_t>((n_slots * 32 + 255) / 256, (int64_t)c->sm_count * 16);
    k_of_slots<<<blocks, 256, 0, st>>>(make_map(c), c->n_steps, c->st_count.p, c->st_width.p, c->st_real.p, c->st_round.p,
                                       c->st_origin.p, c->step_samples.p);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

}  // namespace odb
