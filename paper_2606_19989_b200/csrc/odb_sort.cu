// A0 + A1 in ONE launch: window fill and the segmented sort of every rank's window by the composite key
// (length, local id) (paper section 2.2 P:36 "sorted ascending"; reading U1).  sm_100a only.
//
// A rank's window of up to CL * 4096 keys is sorted by a thread-block CLUSTER of CL CTAs (CL = 1, 2, 4, 8
// or 16): each CTA merge-sorts 4096 keys in its shared memory (1024 threads x 4 keys: a register sorting
// network, then ten merge-path levels with 4-step serial merges), then log2(CL) cross-CTA levels merge runs that live in the
// shared memory of neighbouring CTAs, read through distributed shared memory (DSMEM): a CTA cuts its
// 4096-key output tile out of the two runs with merge-path searches over DSMEM, stages the two input
// pieces locally with coalesced DSMEM loads, merges them from local shared memory, and the cluster
// barrier separates the levels.  The last level leaves through shared memory with coalesced stores.
// No global-memory round trip and no launch between the levels (the round-1 design was one chunk-sort
// launch plus one launch per merge level).
#include "odb_sort.cuh"

namespace odb {

#define ODB_LAUNCH_CHECK(c)                       \
    do {                                          \
        (c)->launches++;                          \
        cudaError_t e_ = cudaGetLastError();      \
        if (e_ != cudaSuccess) return e_;         \
    } while (0)

// grid = (CL, R), cluster (CL, 1, 1).  Dynamic shared memory: X (and Y when CL > 1), MsSort<ITEMS>::kPadded keys each.
// ITEMS keys per thread, 4096 / ITEMS threads per CTA.
template <int ITEMS>
__global__ void __launch_bounds__(MsSort<ITEMS>::kThreads) k_sort_window(const SortArgs A, int CL) {
    using MS = MsSort<ITEMS>;
    constexpr int kThreads = MS::kThreads;
    extern __shared__ __align__(16) unsigned char ms_smem[];
    uint64_t *X = reinterpret_cast<uint64_t *>(ms_smem);
    uint64_t *Y = X + MS::kPadded;
    __shared__ int s_cut[2];
    const int r_ = blockIdx.y, c = blockIdx.x, t = threadIdx.x;
    if (A.first)  // start of a run: the per-run state is cleared here instead of by a launch of its own
        ms_first_round_init(A, ((int64_t)r_ * gridDim.x + c) * kThreads + t, (int64_t)gridDim.x * gridDim.y * kThreads);
    const int64_t base = A.rank_ptr[r_];
    const int n_r = (int)(A.rank_ptr[r_ + 1] - base);
    const int nl = A.first ? 0 : A.n_left[r_], fp = A.first ? 0 : A.fetch_pos[r_];
    // only the views the workers have delivered so far can be drained (App. C.1; odb_set_available)
    const int S = ms_window_size(nl, fp, min(n_r, A.arrived[r_]), A.buffer_size);
    if (c == 0 && t == 0) {
        A.S_out[r_] = S;
        if (A.first) {
            A.n_left[r_] = 0;
            A.fetch_pos[r_] = 0;
            A.emit_cur[r_] = 0;
        }
        if (r_ == 0 && A.rec) A.rec->n_finished = 0;  // counted again by this round's commit
    }
    if (S == 0) return;  // the whole cluster leaves
    const int c0 = c * kMsChunk;
    const int cnt = max(0, min(kMsChunk, S - c0));
    uint64_t k[ITEMS];
    // (a lone CTA sorts only as many keys as its window needs; in a cluster every CTA sorts a full chunk)
    const int n_keys = CL == 1 ? MS::active_keys(cnt) : kMsChunk;
    ms_load_keys_t<ITEMS>(A, base, nl, fp, c0, cnt, n_keys, k);
    MS::sort_cta(k, X, n_keys);
    uint64_t *out = A.keys_out + base;
    if (CL == 1) {
        for (int i = t; i < cnt; i += kThreads) out[i] = X[MS::pad(i)];
        return;
    }
    // ---- cross-CTA levels: runs of m CTAs are merged pairwise; CTA c owns outputs [4096 c, 4096 (c + 1)) ----
    const uint32_t x_addr = smem_addr(X);
#pragma unroll 1
    for (int m = 1; m < CL; m <<= 1) {
        cluster_sync_all();  // every CTA's X holds the previous level
        const int p0 = c & ~(2 * m - 1);  // first CTA of the pair of runs
        const int na = m * kMsChunk, nb = m * kMsChunk;
        const int d0 = (c - p0) * kMsChunk, d1 = d0 + kMsChunk;
        if (t < 64) {  // warp 0: the cut of the tile's first diagonal, warp 1: of its last
            const int cut = MS::path_remote(x_addr, p0, na, p0 + m, nb, t < 32 ? d0 : d1);
            if ((t & 31) == 0) s_cut[t >> 5] = cut;
        }
        __syncthreads();
        const int a0 = s_cut[0], a1 = s_cut[1];
        const int b0 = d0 - a0;
        const int la = a1 - a0;  // + (b1 - b0) == 4096
        // stage the two pieces in Y: [0, la) from run A, [la, 4096) from run B (coalesced DSMEM loads)
        for (int i = t; i < kMsChunk; i += kThreads)
            Y[MS::pad(i)] = i < la ? MS::run_key(x_addr, p0, a0 + i) : MS::run_key(x_addr, p0 + m, b0 + (i - la));
        __syncthreads();
        const int ai = MS::path_local(Y, 0, la, la, kMsChunk - la, ITEMS * t);
        MS::merge_items(Y, ai, la, la + (ITEMS * t - ai), kMsChunk, k);
        cluster_sync_all();  // every CTA has read what it needs from the others' X
#pragma unroll
        for (int q = 0; q < ITEMS; ++q) X[MS::pad(ITEMS * t + q)] = k[q];
        __syncthreads();
    }
    for (int i = t; i < cnt; i += kThreads) out[c0 + i] = X[MS::pad(i)];
    cluster_sync_all();  // nobody leaves while a neighbour may still read its shared memory (none does; cheap insurance)
}

template <int ITEMS>
static cudaError_t launch_sort_segments_t(odb_ctx *c, const SortArgs &A0, int64_t nseg, int CL, bool *attr_done, cudaStream_t st) {
    using MS = MsSort<ITEMS>;
    const size_t smem = (size_t)(CL > 1 ? 2 : 1) * MS::kPadded * sizeof(uint64_t);
    if (!*attr_done) {
        cudaError_t e = cudaFuncSetAttribute(k_sort_window<ITEMS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)(2 * MS::kPadded * sizeof(uint64_t)));
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(k_sort_window<ITEMS>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
        *attr_done = true;
    }
    for (int64_t s0 = 0; s0 < nseg; s0 += 65535) {  // gridDim.y is limited to 65535
        const unsigned ns = (unsigned)std::min<int64_t>(nseg - s0, 65535);
        SortArgs A = A0;
        A.rank_ptr += s0;
        A.n_left += s0;
        A.fetch_pos += s0;
        A.emit_cur += s0;
        A.arrived += s0;
        A.S_out += s0;
        if (s0 > 0) A.first = 0;  // (the per-run state is cleared by the first batch of segments)
        if (CL == 1) {  // no cluster needed: a plain launch (the attribute path costs a few microseconds per launch)
            k_sort_window<ITEMS><<<dim3(1, ns), MS::kThreads, smem, st>>>(A, 1);
            ODB_LAUNCH_CHECK(c);
            continue;
        }
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3((unsigned)CL, ns, 1);
        cfg.blockDim = dim3(MS::kThreads, 1, 1);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)CL;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        cudaError_t e = cudaLaunchKernelEx(&cfg, k_sort_window<ITEMS>, A, CL);
        if (e != cudaSuccess) return e;
        c->launches++;
    }
    return cudaSuccess;
}

// Launches the cluster sort for `nseg` segments (rank windows; buckets / megabatches of the offline planners)
// of up to 16 * 4096 keys each.  Returns cudaErrorNotSupported when a segment can be larger (the caller falls
// back to chunk sorts + global merge passes).
cudaError_t launch_sort_segments(odb_ctx *c, const SortArgs &A0, int64_t nseg, int maxS, cudaStream_t st) {
    const int chunks = (maxS + kMsChunk - 1) / kMsChunk;
    int CL = 1;
    while (CL < chunks) CL <<= 1;
    if (CL > 16) return cudaErrorNotSupported;
    // keys per thread: 8 (512 threads per 4096-key chunk) for windows of 16 K keys and more, 4 (1024 threads) below.
    // Measured planning stage with 4 / 8 / 16 keys per thread: 32 x 32768-key windows 0.214 / 0.199 / 0.203 ms,
    // 16 x 16384 0.131 / 0.128 / 0.142 ms, 8 x 8192 0.107 / 0.107 / 0.120 ms.
    if (CL >= 4) return launch_sort_segments_t<8>(c, A0, nseg, CL, &c->attr_sort8, st);
    return launch_sort_segments_t<4>(c, A0, nseg, CL, &c->attr_sort, st);
}

cudaError_t launch_sort_window(odb_ctx *c, int maxS, bool first, cudaStream_t st) {
    SortArgs A;
    A.len = c->d_lengths;
    A.rank_ptr = c->d_rank_ptr;
    A.n_left = c->n_left;
    A.fetch_pos = c->fetch_pos;
    A.emit_cur = c->emit_cur;
    A.left_ids = c->left_ids;
    A.arrived = c->d_arrived;
    A.buffer_size = c->prm.buffer_size;
    A.keys_out = c->keyA;
    A.S_out = c->S;
    A.rec = c->d_rec;
    A.first = first ? 1 : 0;
    A.n_total = c->n_total;
    A.emit_pos = c->emit_pos;
    A.step_samples = c->step_samples.p;
    A.step_cap = c->step_samples.p ? (int64_t)c->step_samples.cap : 0;
    cudaError_t e = launch_sort_segments(c, A, c->prm.n_ranks, maxS, st);
    if (e == cudaSuccess) c->sorted = c->keyA;
    return e;
}

}  // namespace odb
