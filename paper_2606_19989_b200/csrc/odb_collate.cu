// Collation kernels (rows A10, A11 of DESIGN.md): every emitted slot becomes a dense, right-padded
// [count x width] block in four arenas (input_ids, attention_mask, position_ids, labels), with the
// pad fill, label shift, span masking and the valid-token count fused.  sm_100a only.
//
// Paper: collate_fn P:28; pad to the group max P:416-420; valid tokens t_r of Eq. 2 P:60-63.
// Tensor contract: BASELINE.json north_star (readings U16-U18).
#include <cstring>

#include "odb_internal.cuh"
#include "odb_device.cuh"

namespace odb {

#define ODB_LAUNCH_CHECK(c)                       \
    do {                                          \
        (c)->launches++;                          \
        cudaError_t e_ = cudaGetLastError();      \
        if (e_ != cudaSuccess) return e_;         \
    } while (0)

// ---------------------------------------------------------------------------------------------
// Collate preparation, ONE launch with three roles told apart by the block index (all sizes come from
// the device-resident PlanDims; the launch is skipped on the device when the plan is not complete or the
// caller's capacities are too small):
//
//   rows   one thread per sample (coalesced reads of sample_ptr / lengths / span CSR): the 32-byte
//          RowDesc of every emitted sample, stored at its rank's first row + its position in the rank's
//          emit region;
//   tiles  one warp per slot, a lane per 4096-element tile whose first element lies in the slot's
//          16-aligned region [grp_offset[s], grp_offset[s+1]) (IDLE slots own none): the 32-byte TileRec
//          the collate kernel starts a tile with.  These blocks also clear what the collate kernel
//          accumulates into (grp_valid, the work counters) and copy the plan tables into the caller's;
//   ids    one block per rank: the un-emitted local ids, ascending (Lemma 1: buffer + sampler-pending).
// ---------------------------------------------------------------------------------------------
constexpr int kPrepThreads = 1024;

struct PrepJob {
    void *dst;
    const void *src;
    int kind;  // words to copy: 0 = n_slots, 1 = 2 n_slots, 2 = 2 (n_slots + 1), 3 = n_steps, 4 = samples_emitted, 5 = 2 (R + 1)
};

struct PrepArgs {
    const PlanDims *dims;
    int R;
    // rows
    int offline_row_blocks;  // > 0: an offline plan (global ids): one thread per emitted ROW, that many blocks
    int rows_gx;  // blocks per rank
    const int64_t *rank_ptr;
    const int32_t *len;
    const int32_t *emit_pos;
    const int64_t *sample_ptr;
    const int64_t *span_ptr;
    const int32_t *span_lo;
    const int32_t *span_hi;
    const int64_t *grp_sample_ptr;
    RowDesc *rows;
    int64_t *row_sp;
    // tiles
    int tile_blocks;
    const int64_t *grp_offset;
    const int32_t *grp_count;
    const int32_t *grp_width;
    TileRec *tiles;
    int32_t *grp_valid;
    unsigned long long *tile_counter;
    int n_counters;
    PrepJob job[10];
    int n_jobs;
    // ids
    const int32_t *emit_cur;
    const int32_t *emit_ids;
    int32_t *grp_sample_ids, *user_ids;
    int64_t *left_ptr, *user_left_ptr;
    int32_t *left_out, *user_left;
};

__device__ __forceinline__ void prep_rows(const PrepArgs &A, int n_steps, int b) {
    const int r = b / A.rows_gx, bx = b - r * A.rows_gx;
    const int64_t base = A.rank_ptr[r];
    const int n_r = (int)(A.rank_ptr[r + 1] - base);
    const int i = bx * kPrepThreads + threadIdx.x;
    if (i >= n_r) return;
    const int64_t g = base + i;
    const int64_t q0 = A.grp_sample_ptr[(int64_t)r * n_steps];
    // the slot CSR's ids are the rank's emit region (slots of a rank are in emit order): entry i of it
    if (i < A.emit_cur[r]) {
        const int32_t id = A.emit_ids[g];
        A.grp_sample_ids[q0 + i] = id;
        if (A.user_ids) A.user_ids[q0 + i] = id;
    }
    const int p = A.emit_pos[g];
    if (p < 0) return;
    const int64_t q = q0 + p;
    RowDesc d;
    d.tok = A.sample_ptr[g];
    d.len = A.len[g];
    const int64_t sp = A.span_ptr ? A.span_ptr[g] : 0;
    const int ns = A.span_ptr ? (int)(A.span_ptr[g + 1] - sp) : 0;
    d.nspan = ns;
    d.lo0 = ns > 0 ? A.span_lo[sp] : 0;
    d.hi0 = ns > 0 ? A.span_hi[sp] : 0;
    d.lo1 = ns > 1 ? A.span_lo[sp + 1] : 0;
    d.hi1 = ns > 1 ? A.span_hi[sp + 1] : 0;
    A.rows[q] = d;
    if (ns > 2) A.row_sp[q] = sp;  // only read on the CSR path (more than two spans): skip the scattered 8-byte store
}

// offline plans (F4): the slot CSR holds GLOBAL sample ids and a sample may be emitted twice, so the row
// descriptors are gathered in emit order: one thread per emitted row
__device__ __forceinline__ void prep_rows_offline(const PrepArgs &A, int b) {
    const int64_t n_rows = A.dims->samples_emitted;
    for (int64_t q = (int64_t)b * kPrepThreads + threadIdx.x; q < n_rows; q += (int64_t)A.offline_row_blocks * kPrepThreads) {
        const int64_t g = A.grp_sample_ids[q];
        if (A.user_ids) A.user_ids[q] = (int32_t)g;
        RowDesc d;
        d.tok = A.sample_ptr[g];
        d.len = A.len[g];
        const int64_t sp = A.span_ptr ? A.span_ptr[g] : 0;
        const int ns = A.span_ptr ? (int)(A.span_ptr[g + 1] - sp) : 0;
        d.nspan = ns;
        d.lo0 = ns > 0 ? A.span_lo[sp] : 0;
        d.hi0 = ns > 0 ? A.span_hi[sp] : 0;
        d.lo1 = ns > 1 ? A.span_lo[sp + 1] : 0;
        d.hi1 = ns > 1 ? A.span_hi[sp + 1] : 0;
        A.rows[q] = d;
        if (ns > 2) A.row_sp[q] = sp;
    }
}

__device__ __forceinline__ void prep_tiles(const PrepArgs &A, int n_steps, int64_t n_slots, int b) {
    const int64_t tid = (int64_t)b * kPrepThreads + threadIdx.x, nth = (int64_t)A.tile_blocks * kPrepThreads;
    for (int64_t s = tid; s < n_slots; s += nth) A.grp_valid[s] = 0;
    if (tid < A.n_counters) A.tile_counter[tid] = 0ull;
    const int lane = threadIdx.x & 31;
    for (int64_t s = tid >> 5; s < n_slots; s += nth >> 5) {
        const int64_t o = A.grp_offset[s], on = A.grp_offset[s + 1];
        const int64_t t_lo = (o + kColTile - 1) / kColTile, t_hi = (on + kColTile - 1) / kColTile;
        if (t_lo >= t_hi) continue;
        TileRec rec;
        rec.off_s = o;
        rec.slot = (int32_t)s;
        rec.W = (uint32_t)A.grp_width[s];
        rec.area = (uint32_t)A.grp_count[s] * rec.W;
        rec.sp_s = (uint32_t)A.grp_sample_ptr[s];
        rec.pad_[0] = rec.pad_[1] = 0u;
        for (int64_t t = t_lo + lane; t < t_hi; t += 32) A.tiles[t] = rec;
    }
    for (int j = 0; j < A.n_jobs; ++j) {
        const int kind = A.job[j].kind;
        const int64_t words = kind == 0   ? n_slots
                              : kind == 1 ? 2 * n_slots
                              : kind == 2 ? 2 * (n_slots + 1)
                              : kind == 3 ? (int64_t)n_steps
                              : kind == 4 ? A.dims->samples_emitted
                                          : 2 * ((int64_t)A.R + 1);
        const uint32_t *__restrict__ src = reinterpret_cast<const uint32_t *>(A.job[j].src);
        uint32_t *__restrict__ dst = reinterpret_cast<uint32_t *>(A.job[j].dst);
        for (int64_t i = tid; i < words; i += nth) dst[i] = src[i];
    }
}

__device__ __forceinline__ void prep_ids(const PrepArgs &A, int n_steps, int r) {
    __shared__ int s_scan[34];
    __shared__ long long s_scan64[34];
    const int R = A.R;
    const int64_t base = A.rank_ptr[r];
    const int n_r = (int)(A.rank_ptr[r + 1] - base);
    const int ec = A.emit_cur[r];  // (the slot CSR's ids are copied by the row threads)
    long long part = 0;
    for (int q = threadIdx.x; q < r; q += blockDim.x) part += (A.rank_ptr[q + 1] - A.rank_ptr[q]) - A.emit_cur[q];
    long long lbase;
    (void)block_excl_scan<long long>(part, s_scan64, lbase);
    const int cnt = n_r - ec;
    if (cnt > 0) {
        const int32_t *ep = A.emit_pos + base;
        int32_t *out = A.left_out + lbase;
        int32_t *uout = A.user_left ? A.user_left + lbase : nullptr;
        (void)block_compact(
            n_r, s_scan, [&](int i) { return ep[i] < 0; },
            [&](int i, int kidx) {
                out[kidx] = i;
                if (uout) uout[kidx] = i;
            });
    }
    if (threadIdx.x == 0) {
        A.left_ptr[r] = lbase;
        if (A.user_left_ptr) A.user_left_ptr[r] = lbase;
        if (r == R - 1) {
            A.left_ptr[R] = lbase + cnt;
            if (A.user_left_ptr) A.user_left_ptr[R] = lbase + cnt;
        }
    }
}

__global__ void __launch_bounds__(kPrepThreads) k_prep(const PrepArgs A) {
    if (!A.dims->complete || A.dims->err) return;
    const int n_steps = A.dims->n_steps;
    const int64_t n_slots = (int64_t)A.R * n_steps;
    const int b = blockIdx.x;
    const int nb_rows = A.offline_row_blocks > 0 ? A.offline_row_blocks : A.rows_gx * A.R;
    if (b < nb_rows) {
        if (A.offline_row_blocks > 0) prep_rows_offline(A, b);
        else prep_rows(A, n_steps, b);
    } else if (b < nb_rows + A.tile_blocks) {
        prep_tiles(A, n_steps, n_slots, b - nb_rows);
    } else {
        prep_ids(A, n_steps, b - nb_rows - A.tile_blocks);
    }
}

// ---------------------------------------------------------------------------------------------
// collate
//
// The four arenas are treated as flat arrays.  A tile is kColTile = 4096 consecutive arena elements;
// each of a CTA's 8 warps owns a CHUNK of 512 consecutive elements.  Block offsets are multiples of
// 16, so a UNIT of 16 consecutive, 16-aligned elements never straddles two slots.
//
//   interior chunk (all 512 elements inside one slot's [count x width] block; > 95 % of the chunks
//   of the BASELINE.json configs): lane l owns unit l = elements [16 l, 16 l + 16) of the chunk and
//   writes them with two 256-bit stores per int32 arena (STG.256: each lane fills whole 32-byte
//   sectors) and one 16-byte store of the uint8 mask.  Tokens are fetched with four 16-byte ALIGNED
//   loads: a row's tokens start at an arbitrary 4-byte offset, so the lane loads the aligned vectors
//   that cover its first 16 tokens and takes the following vector (it holds the shifted label of the
//   last element) from its right-hand neighbour by shuffle, or loads it when the neighbour is in
//   another row; the 17 tokens t..t+16 are then picked by the skew (0..3 words).  Real / masked /
//   valid flags are 16-bit sets built with range arithmetic, not per-element compares, and units
//   that are all real / all valid / all ignored skip the per-element selects.
//   Units that cross a row end (one per row) are handled by the warp together, one element per
//   lane, while the aligned loads are in flight.
//
//   boundary chunk (slot change, alignment gap, block end, end of arena): the per-vector generic
//   path (4-element vectors, scalar loads, 4-byte mask stores).
//
// Work distribution: persistent CTAs take runs of up to kColGrab tiles from an atomic counter.
// A11: valid-token counts are integer sums: warp reduce, one atomicAdd per chunk and slot.
// ---------------------------------------------------------------------------------------------
struct RowRegs {
    int64_t tok;
    int32_t len, nspan, lo0, hi0, lo1, hi1;
};

__device__ __forceinline__ RowRegs load_row(const RowDesc *__restrict__ rows, int64_t q) {
    const int4 *p = reinterpret_cast<const int4 *>(rows + q);
    int4 a = __ldg(p), b = __ldg(p + 1);
    RowRegs r;
    r.tok = (int64_t)(((uint64_t)(uint32_t)a.y << 32) | (uint32_t)a.x);
    r.len = a.z;
    r.nspan = a.w;
    r.lo0 = b.x;
    r.hi0 = b.y;
    r.lo1 = b.z;
    r.hi1 = b.w;
    return r;
}

// 256-bit streaming store (.cs: the arenas are written once and not re-read by this kernel)
__device__ __forceinline__ void st256(int32_t *p, const int32_t (&v)[16], int o) {
    asm volatile("st.global.cs.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(v[o]), "r"(v[o + 1]), "r"(v[o + 2]),
                 "r"(v[o + 3]), "r"(v[o + 4]), "r"(v[o + 5]), "r"(v[o + 6]), "r"(v[o + 7])
                 : "memory");
}

template <int N>
__device__ __forceinline__ int clamp0(int v) {
    return min(max(v, 0), N);
}

// bits j in [0, N) with lo <= c0 + j < hi
template <int N>
__device__ __forceinline__ uint32_t range_bits(int lo, int hi, int c0) {
    const uint32_t below_hi = (1u << clamp0<N>(hi - c0)) - 1u;
    const uint32_t below_lo = (1u << clamp0<N>(lo - c0)) - 1u;
    return below_hi & ~below_lo;
}

// bits j in [0, N) whose position c0 + j lies in a masked span of the row
template <int N>
__device__ __forceinline__ uint32_t masked_bits(const RowRegs &r, int c0, const CollateArgs &A, int64_t q) {
    uint32_t m = range_bits<N>(r.lo0, r.hi0, c0) | range_bits<N>(r.lo1, r.hi1, c0);
    if (r.nspan > 2) {  // rare: walk the CSR
        const int64_t sp = A.row_sp[q];
        for (int j = 2; j < r.nspan; ++j) m |= range_bits<N>(A.span_lo[sp + j], A.span_hi[sp + j], c0);
    }
    return m;
}

// bit j -> byte j (4 bits -> 4 bytes of 0 / 1)
__device__ __forceinline__ uint32_t spread4(uint32_t bits) { return ((bits & 15u) * 0x00204081u) & 0x01010101u; }

// one output element (row r, column c)
template <bool SHIFT>
__device__ __forceinline__ void one_element(const CollateArgs &A, const RowRegs &r, int64_t q, int c, int32_t &id,
                                            int32_t &lab, int32_t &pos, uint32_t &m) {
    const int32_t *tp = A.tokens + r.tok;
    const bool real = c < r.len;
    id = real ? __ldg(tp + c) : A.pad_id;
    pos = real ? c : 0;
    m = real ? 1u : 0u;
    if (SHIFT) {
        const bool ok = (c + 1 < r.len) && !(masked_bits<1>(r, c + 1, A, q) & 1u);
        lab = ok ? __ldg(tp + c + 1) : A.ignore_index;
    } else {
        const bool ok = real && !(masked_bits<1>(r, c, A, q) & 1u);
        lab = ok ? id : A.ignore_index;
    }
}

// Boundary chunks: 4 consecutive elements starting at block element e, which may cross row ends
// (and, when `area` < e + 4, the end of the block): element by element.  Returns the mask bytes.
template <bool SHIFT>
__device__ __forceinline__ uint32_t straddle_vector(const CollateArgs &A, int64_t a, uint32_t e, uint32_t W, uint32_t area,
                                                    int64_t sp_s, int &acc) {
    uint32_t mw = 0;
#pragma unroll 1
    for (int j = 0; j < 4; ++j) {
        const uint32_t ee = e + j;
        if (ee >= area) break;
        const uint32_t bb = ee / W;
        const int c = (int)(ee - bb * W);
        const int64_t q = sp_s + bb;
        const RowRegs r = load_row(A.rows, q);
        int32_t id, lb, ps;
        uint32_t m;
        one_element<SHIFT>(A, r, q, c, id, lb, ps, m);
        A.ids[a + j] = id;
        A.labels[a + j] = lb;
        A.pos[a + j] = ps;
        mw |= m << (8 * j);
        acc += (lb != A.ignore_index) ? 1 : 0;
    }
    return mw;
}

// Boundary chunks: a 4-element vector inside one row from the 5 tokens x[0..4] = tokens t .. t+4.
template <bool SHIFT>
__device__ __forceinline__ void emit_vector(const CollateArgs &A, const RowRegs &r, int64_t q, int t, const int32_t (&x)[5],
                                            int64_t a, uint32_t &mword, int &acc) {
    const int nreal = clamp0<4>(r.len - t);  // elements t .. t+3 that are real tokens
    uint32_t ok;                              // elements whose label carries a loss term
    if (SHIFT) ok = ((1u << clamp0<4>(r.len - 1 - t)) - 1u) & ~masked_bits<4>(r, t + 1, A, q);
    else ok = ((1u << nreal) - 1u) & ~masked_bits<4>(r, t, A, q);
    acc += __popc(ok);
    const int4 oid = make_int4(nreal > 0 ? x[0] : A.pad_id, nreal > 1 ? x[1] : A.pad_id, nreal > 2 ? x[2] : A.pad_id,
                               nreal > 3 ? x[3] : A.pad_id);
    const int4 opos = make_int4(nreal > 0 ? t : 0, nreal > 1 ? t + 1 : 0, nreal > 2 ? t + 2 : 0, nreal > 3 ? t + 3 : 0);
    const int4 olab = make_int4((ok & 1u) ? x[SHIFT ? 1 : 0] : A.ignore_index, (ok & 2u) ? x[SHIFT ? 2 : 1] : A.ignore_index,
                                (ok & 4u) ? x[SHIFT ? 3 : 2] : A.ignore_index, (ok & 8u) ? x[SHIFT ? 4 : 3] : A.ignore_index);
    __stcs(reinterpret_cast<int4 *>(A.ids + a), oid);
    __stcs(reinterpret_cast<int4 *>(A.labels + a), olab);
    __stcs(reinterpret_cast<int4 *>(A.pos + a), opos);
    mword = spread4((1u << nreal) - 1u);
}

// ---- bulk (TMA) stores from shared memory: the alternative store form of the interior chunks ----
constexpr int kColStage = 3 * kColChunk * 4 + kColChunk;  // one warp's staging buffer: ids | labels | pos | mask
__device__ __forceinline__ void bulk_store(void *gdst, const void *ssrc, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst),
                 "r"((uint32_t)__cvta_generic_to_shared(ssrc)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// 16 consecutive int32 of a unit: two 256-bit streaming stores to the arena, or four 16-byte stores to the
// warp's staging buffer
template <bool BULK>
__device__ __forceinline__ void put16(int32_t *p, const int32_t (&o)[16]) {
    if (BULK) {
        int4 *q = reinterpret_cast<int4 *>(p);
#pragma unroll
        for (int i = 0; i < 4; ++i) q[i] = make_int4(o[4 * i], o[4 * i + 1], o[4 * i + 2], o[4 * i + 3]);
    } else {
        st256(p, o, 0);
        st256(p + 8, o, 8);
    }
}

// Interior chunks: a 16-element unit inside one row from the 17 tokens x[0..16] = tokens t .. t+16
// (anything beyond the sample), written at d_ids / d_lab / d_pos (the arenas, or the staging buffer).
// Returns the 16 mask bytes.
template <bool SHIFT, bool BULK>
__device__ __forceinline__ int4 emit_unit(const CollateArgs &A, const RowRegs &r, int64_t q, int t, const int32_t (&x)[17],
                                          int32_t *d_ids, int32_t *d_lab, int32_t *d_pos, int &acc) {
    const int nreal = clamp0<16>(r.len - t);  // elements t .. t+15 that are real tokens
    const uint32_t real = (1u << nreal) - 1u;
    uint32_t ok;  // elements whose label carries a loss term
    if (SHIFT) ok = ((1u << clamp0<16>(r.len - 1 - t)) - 1u) & ~masked_bits<16>(r, t + 1, A, q);
    else ok = real & ~masked_bits<16>(r, t, A, q);
    acc += __popc(ok);
    int32_t o[16];
    // input_ids
    if (nreal == 16) {
#pragma unroll
        for (int j = 0; j < 16; ++j) o[j] = x[j];
    } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) o[j] = j < nreal ? x[j] : A.pad_id;
    }
    put16<BULK>(d_ids, o);
    // position_ids
#pragma unroll
    for (int j = 0; j < 16; ++j) o[j] = j < nreal ? t + j : 0;
    put16<BULK>(d_pos, o);
    // labels
    if (ok == 0xFFFFu) {
#pragma unroll
        for (int j = 0; j < 16; ++j) o[j] = x[j + (SHIFT ? 1 : 0)];
    } else if (ok == 0u) {
#pragma unroll
        for (int j = 0; j < 16; ++j) o[j] = A.ignore_index;
    } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) o[j] = ((ok >> j) & 1u) ? x[j + (SHIFT ? 1 : 0)] : A.ignore_index;
    }
    put16<BULK>(d_lab, o);
    return make_int4((int)spread4(real), (int)spread4(real >> 4), (int)spread4(real >> 8), (int)spread4(real >> 12));
}

// BULK = false: the interior chunks leave the registers with 256-bit streaming stores (the adopted form);
// BULK = true: they are staged in shared memory (one 6.5 KB buffer per warp) and leave with four bulk (TMA)
// stores per chunk, one per arena (BASELINE.json's sketch of the store side; measured in profiles/r02_*).
template <bool SHIFT, bool BULK>
__global__ void __launch_bounds__(kColThreads, 3) k_collate(const CollateArgs A) {
    extern __shared__ __align__(128) unsigned char col_smem[];
    __shared__ long long s_grab;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // this warp's staging buffer (BULK only)
    int32_t *const s_ids = reinterpret_cast<int32_t *>(col_smem + (BULK ? (size_t)warp * kColStage : 0));
    int32_t *const s_lab = s_ids + kColChunk, *const s_pos = s_lab + kColChunk;
    uint8_t *const s_msk = reinterpret_cast<uint8_t *>(s_pos + kColChunk);
    constexpr int kWarps = kColThreads / 32;
    static_assert(kColChunk == 512 && kColTile == kWarps * kColChunk, "a chunk is one 16-element unit per lane");
    const int4 *tok4 = reinterpret_cast<const int4 *>(A.tokens);
    // a whole-arena launch reads its extent on the device (it may have been enqueued before the host saw
    // the plan) and does nothing when the plan is not complete or the caller's buffers are too small
    int64_t total_elems = A.total_elems, tile_hi = A.tile_hi;
    if (A.whole) {
        if (!A.dims->complete || A.dims->err) return;
        total_elems = A.dims->total_elems;
        tile_hi = (total_elems + kColTile - 1) / kColTile;
    }
    // tiles taken from the work counter at a time: kColGrab when there is plenty of work (the measured optimum on the
    // large configs), fewer when the launch holds only a few runs per CTA, so that small launches do not end with
    // half of the CTAs idle (configs[1] has 1.2 runs of 16 per CTA)
    const int64_t n_tiles_all = tile_hi - A.tile_lo;
    const int grab = (int)max((int64_t)1, min((int64_t)kColGrab, n_tiles_all / ((int64_t)gridDim.x * 8)));
    for (;;) {
        __syncthreads();  // everyone has read the previous s_grab
        if (threadIdx.x == 0) s_grab = (long long)atomicAdd(A.tile_counter, (unsigned long long)grab);
        __syncthreads();
        const int64_t tile_begin = A.tile_lo + s_grab;
        if (tile_begin >= tile_hi) break;
        const int64_t tile_end = min(tile_begin + grab, tile_hi);
#pragma unroll 1
        for (int64_t tile = tile_begin; tile < tile_end; ++tile) {
            const int64_t chunk = tile * kWarps + warp;
            const int64_t a0 = chunk * kColChunk;
            if (a0 >= total_elems) break;
            if (a0 + kColChunk <= A.elem_lo) continue;  // another launch's elements (odb_run_host pipelines ranks)
            // the tile's record: the slot that holds the tile's first element, and its geometry
            const int4 *tp = reinterpret_cast<const int4 *>(A.tiles + tile);
            const int4 c0 = __ldg(tp), c1 = __ldg(tp + 1);
            int64_t off_s = (int64_t)(((uint64_t)(uint32_t)c0.y << 32) | (uint32_t)c0.x);
            int64_t s = c0.z;
            uint32_t W = (uint32_t)c0.w, area = (uint32_t)c1.x;
            int64_t sp_s = (int64_t)(uint32_t)c1.y;
            if (a0 >= off_s + (((int64_t)area + 15) & ~15ll)) {
                // this warp's chunk starts in a later slot of the tile: find the slot j >= s + 1 whose region
                // [grp_offset[j], grp_offset[j + 1]) holds a0, 32 upper boundaries at a time (IDLE slots have
                // empty regions and are skipped over)
                int64_t cand = s + 1;
                const int64_t n_slots = A.dims->n_slots;
                for (;;) {  // warp-uniform
                    const int64_t idx = cand + 1 + lane;
                    const int64_t v = idx <= n_slots ? __ldg(A.grp_offset + idx) : 0x7fffffffffffffffll;
                    const uint32_t gt = __ballot_sync(ODB_FULL_MASK, v > a0);
                    if (gt) {
                        s = cand + (__ffs(gt) - 1);
                        break;
                    }
                    cand += 32;
                }
                off_s = __ldg(A.grp_offset + s);
                W = (uint32_t)__ldg(A.grp_width + s);
                area = (uint32_t)__ldg(A.grp_count + s) * W;
                sp_s = __ldg(A.grp_sample_ptr + s);
            }
            const int64_t e0 = a0 - off_s;
            int acc = 0;
            if (e0 + kColChunk <= (int64_t)area) {
                // ---------------- interior chunk: lane = one 16-element unit ----------------
                const uint32_t b0 = (uint32_t)e0 / W, t0 = (uint32_t)e0 - b0 * W;  // row / column of the chunk's first element
                const bool wide = W >= (uint32_t)kColChunk;  // then t0 + 16 l < 2 W: the row index grows by 0 or 1
                // ceil(2^32 / W): floor(n / W) == umulhi(n, M) for n < 1024 and 2 <= W < 512
                const uint32_t M = (W >= 2u && !wide) ? 0xFFFFFFFFu / W + 1u : 0u;
                const uint32_t n = t0 + 16u * (uint32_t)lane;  // column if the row never ended
                const uint32_t d = wide ? (n >= W ? 1u : 0u) : (W >= 2u ? __umulhi(n, M) : n);
                const int t = (int)(n - d * W);
                const uint32_t q = (uint32_t)sp_s + b0 + d;  // samples_emitted < 2^31
                const bool fast = (uint32_t)t + 16u <= W;
                const RowRegs r = load_row(A.rows, (int64_t)q);
                const int64_t g = r.tok + t;            // index of the unit's first token in d_tokens
                const int64_t qv = g >> 2;              // aligned vector that holds it
                const int64_t send = r.tok + r.len;     // one past the sample's last token
                const bool ld = fast && t < r.len;
                if (BULK) {  // the previous chunk's bulk stores have read the staging buffer
                    if (lane == 0) bulk_wait_read();
                    __syncwarp();
                }
                int4 v[4];
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    v[i] = (fast && ((qv + i) << 2) < send) ? __ldg(tok4 + qv + i) : make_int4(0, 0, 0, 0);
                // Units that cross a row end (one per row of the block: rare, but a dependent chain
                // of row-descriptor and token loads): the warp handles two of them per pass, one
                // element per lane, while the aligned loads above are in flight.
                int4 mv = make_int4(0, 0, 0, 0);
                uint32_t sb = __ballot_sync(ODB_FULL_MASK, !fast);
                while (sb) {  // warp-uniform
                    const int l0 = __ffs(sb) - 1;
                    sb &= sb - 1;
                    const int l1 = sb ? __ffs(sb) - 1 : -1;
                    if (sb) sb &= sb - 1;
                    const int src = lane < 16 ? l0 : l1;
                    uint32_t m = 0;
                    if (src >= 0) {
                        const int j = lane & 15;
                        const uint32_t ee = (uint32_t)e0 + 16u * (uint32_t)src + (uint32_t)j;
                        const uint32_t bb = ee / W;
                        const int c = (int)(ee - bb * W);
                        const int64_t qq = sp_s + bb;
                        const RowRegs rr = load_row(A.rows, qq);
                        int32_t id, lb, ps;
                        one_element<SHIFT>(A, rr, qq, c, id, lb, ps, m);
                        if (BULK) {
                            s_ids[16 * src + j] = id;
                            s_lab[16 * src + j] = lb;
                            s_pos[16 * src + j] = ps;
                        } else {
                            const int64_t aa = a0 + 16 * src + j;
                            A.ids[aa] = id;
                            A.labels[aa] = lb;
                            A.pos[aa] = ps;
                        }
                        acc += (lb != A.ignore_index) ? 1 : 0;
                        m <<= 8 * (j & 3);
                    }
                    // quad w of each half-warp assembles mask word w of its unit; hand the 4 words to the owner
                    m |= __shfl_xor_sync(ODB_FULL_MASK, m, 1);
                    m |= __shfl_xor_sync(ODB_FULL_MASK, m, 2);
                    const uint32_t w0 = __shfl_sync(ODB_FULL_MASK, m, 0), w1 = __shfl_sync(ODB_FULL_MASK, m, 4);
                    const uint32_t w2 = __shfl_sync(ODB_FULL_MASK, m, 8), w3 = __shfl_sync(ODB_FULL_MASK, m, 12);
                    const uint32_t u0 = __shfl_sync(ODB_FULL_MASK, m, 16), u1 = __shfl_sync(ODB_FULL_MASK, m, 20);
                    const uint32_t u2 = __shfl_sync(ODB_FULL_MASK, m, 24), u3 = __shfl_sync(ODB_FULL_MASK, m, 28);
                    if (lane == l0) mv = make_int4((int)w0, (int)w1, (int)w2, (int)w3);
                    if (lane == l1) mv = make_int4((int)u0, (int)u1, (int)u2, (int)u3);
                }
                // the vector after our four: the right-hand neighbour's first, when it is in the same
                // row and loaded it
                int4 nb;
                nb.x = __shfl_down_sync(ODB_FULL_MASK, v[0].x, 1);
                nb.y = __shfl_down_sync(ODB_FULL_MASK, v[0].y, 1);
                nb.z = __shfl_down_sync(ODB_FULL_MASK, v[0].z, 1);
                nb.w = __shfl_down_sync(ODB_FULL_MASK, v[0].w, 1);
                const uint32_t tag = ld ? q : 0xFFFFFFFFu;
                const uint32_t ntag = __shfl_down_sync(ODB_FULL_MASK, tag, 1);
                if (fast) {
                    if (!(lane < 31 && ntag == q))
                        nb = (ld && ((qv + 4) << 2) < send) ? __ldg(tok4 + qv + 4) : make_int4(0, 0, 0, 0);
                    const int32_t w[20] = {v[0].x, v[0].y, v[0].z, v[0].w, v[1].x, v[1].y, v[1].z, v[1].w, v[2].x, v[2].y,
                                           v[2].z, v[2].w, v[3].x, v[3].y, v[3].z, v[3].w, nb.x,   nb.y,   nb.z,   nb.w};
                    int32_t x[17];
                    switch ((int)g & 3) {  // the skew is the same for every unit of a row
                    case 0:
#pragma unroll
                        for (int j = 0; j < 17; ++j) x[j] = w[j];
                        break;
                    case 1:
#pragma unroll
                        for (int j = 0; j < 17; ++j) x[j] = w[j + 1];
                        break;
                    case 2:
#pragma unroll
                        for (int j = 0; j < 17; ++j) x[j] = w[j + 2];
                        break;
                    default:
#pragma unroll
                        for (int j = 0; j < 17; ++j) x[j] = w[j + 3];
                        break;
                    }
                    if (BULK) mv = emit_unit<SHIFT, true>(A, r, (int64_t)q, t, x, s_ids + 16 * lane, s_lab + 16 * lane, s_pos + 16 * lane, acc);
                    else mv = emit_unit<SHIFT, false>(A, r, (int64_t)q, t, x, A.ids + a0 + 16 * lane, A.labels + a0 + 16 * lane,
                                                      A.pos + a0 + 16 * lane, acc);
                }
                if (BULK) {
                    reinterpret_cast<int4 *>(s_msk)[lane] = mv;
                    fence_async_smem();  // the generic-proxy writes above, before the async proxy reads them
                    __syncwarp();
                    if (lane == 0) {
                        bulk_store(A.ids + a0, s_ids, kColChunk * 4);
                        bulk_store(A.labels + a0, s_lab, kColChunk * 4);
                        bulk_store(A.pos + a0, s_pos, kColChunk * 4);
                        bulk_store(A.mask + a0, s_msk, kColChunk);
                        bulk_commit();
                    }
                } else {
                    __stcs(reinterpret_cast<int4 *>(A.mask + a0 + 16 * lane), mv);
                }
                const int tot = __reduce_add_sync(ODB_FULL_MASK, acc);
                if (lane == 0 && tot != 0) atomicAdd(&A.grp_valid[s], tot);
            } else {
                // ---------------- boundary chunk: generic per-vector path ----------------
                int64_t off_n = A.grp_offset[s + 1];
                int64_t acc_slot = -1;
#pragma unroll 1
                for (int k = 0; k < 4; ++k) {
                    const int64_t a = a0 + (int64_t)(k * 32 + lane) * 4;
                    if (a >= total_elems) break;
                    if (a < A.elem_lo) continue;
                    bool moved = false;
                    while (a >= off_n) {
                        ++s;
                        off_s = off_n;
                        off_n = A.grp_offset[s + 1];
                        moved = true;
                    }
                    if (moved) {
                        W = (uint32_t)A.grp_width[s];
                        area = (uint32_t)A.grp_count[s] * W;
                        sp_s = A.grp_sample_ptr[s];
                    }
                    const uint32_t e = (uint32_t)(a - off_s);
                    if (e >= area) continue;  // alignment gap: never written
                    if (s != acc_slot) {
                        if (acc) atomicAdd(&A.grp_valid[acc_slot], acc);
                        acc = 0;
                        acc_slot = s;
                    }
                    const uint32_t b = e / W;
                    const uint32_t t = e - b * W;
                    uint32_t mw;
                    int nvalid = 4;
                    if (t + 4 <= W) {
                        const int64_t q = sp_s + b;
                        const RowRegs r = load_row(A.rows, q);
                        const int32_t *tp = A.tokens + r.tok + t;
                        const int nreal = max(0, min(5, r.len - (int)t));
                        int32_t x[5];
#pragma unroll
                        for (int j = 0; j < 5; ++j) x[j] = (j < nreal) ? __ldg(tp + j) : A.pad_id;
                        emit_vector<SHIFT>(A, r, q, (int)t, x, a, mw, acc);
                    } else {
                        mw = straddle_vector<SHIFT>(A, a, e, W, area, sp_s, acc);
                        nvalid = (int)min(4u, area - e);
                    }
                    if (nvalid == 4) {
                        __stcs(reinterpret_cast<unsigned int *>(A.mask + a), mw);
                    } else {
                        for (int j = 0; j < nvalid; ++j) A.mask[a + j] = (uint8_t)(mw >> (8 * j));
                    }
                }
                if (acc) atomicAdd(&A.grp_valid[acc_slot], acc);
            }
        }
    }
    if (BULK) {  // the staging buffers must outlive the bulk stores that read them
        if (lane == 0) bulk_wait_all();
        __syncwarp();
    }
}

// After the collate kernel, one launch: step_valid_tokens[k] = sum over ranks of grp_valid_tokens[r][k]
// (Eq. 2's T_tok per step), written to the library's table and the caller's, and the per-slot counts into
// the caller's table.  Sizes from PlanDims; skipped when the plan is not complete / the capacities too small.
// (Fusing this into the collate kernel's last CTA was tried: one CTA walking R x n_steps counts costs
// 40-200 us on the configs[4] cells against 12 us for this launch.)
__global__ void k_post(const PostArgs A) {
    if (!A.dims->complete || A.dims->err) return;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (int64_t)gridDim.x * blockDim.x;
    const int n_steps = A.dims->n_steps;
    const int64_t n_slots = (int64_t)A.R * n_steps;
    for (int64_t k = tid; k < n_steps; k += nth) {
        long long s = 0;
#pragma unroll 4
        for (int r = 0; r < A.R; ++r) s += A.grp_valid[(int64_t)r * n_steps + k];
        A.step_valid[k] = s;
        if (A.user_step_valid) A.user_step_valid[k] = s;
    }
    if (A.user_grp_valid)
        for (int64_t i = tid; i < n_slots; i += nth) A.user_grp_valid[i] = A.grp_valid[i];
}

// ---------------------------------------------------------------------------------------------
// host launchers
// ---------------------------------------------------------------------------------------------
cudaError_t launch_prep(odb_ctx *c, const int64_t *d_sample_ptr, const int64_t *d_span_ptr, const int32_t *d_span_lo,
                        const int32_t *d_span_hi, const odb_outputs *u, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    PrepArgs A;
    memset(&A, 0, sizeof(A));
    A.dims = c->d_dims;
    A.R = R;
    A.rows_gx = std::max((c->max_nr + kPrepThreads - 1) / kPrepThreads, 1);
    A.rank_ptr = c->d_rank_ptr;
    A.len = c->d_lengths;
    A.emit_pos = c->emit_pos;
    A.sample_ptr = d_sample_ptr;
    A.span_ptr = d_span_ptr;
    A.span_lo = d_span_lo;
    A.span_hi = d_span_hi;
    A.grp_sample_ptr = c->grp_sample_ptr.p;
    A.rows = c->rows.p;
    A.row_sp = c->row_sp.p;
    // one warp per slot; the bound on the slot count is what the tables were sized for
    const int64_t slots_bound = (int64_t)c->grp_count.cap;
    A.tile_blocks = (int)std::max<int64_t>(1, std::min<int64_t>((slots_bound * 32 + kPrepThreads - 1) / kPrepThreads,
                                                                (int64_t)c->sm_count * 2));
    A.grp_offset = c->grp_offset.p;
    A.grp_count = c->grp_count.p;
    A.grp_width = c->grp_width.p;
    A.tiles = c->tiles.p;
    A.grp_valid = c->grp_valid.p;
    A.tile_counter = c->d_tile_counter;
    A.n_counters = R + 1;
    auto job = [&](void *dst, const void *src, int kind) {
        if (!dst) return;
        A.job[A.n_jobs].dst = dst;
        A.job[A.n_jobs].src = src;
        A.job[A.n_jobs].kind = kind;
        A.n_jobs++;
    };
    if (u) {
        job(u->d_grp_count, c->grp_count.p, 0);
        job(u->d_grp_width, c->grp_width.p, 0);
        job(u->d_grp_round, c->grp_round.p, 0);
        job(u->d_grp_real_tokens, c->grp_real.p, 0);
        job(u->d_grp_origin, c->grp_origin.p, 0);
        job(u->d_grp_offset, c->grp_offset.p, 1);
        job(u->d_grp_sample_ptr, c->grp_sample_ptr.p, 2);
        job(u->d_step_samples, c->step_samples.p + (c->sub_mode ? c->sub_step_lo : 0), 3);
    }
    A.emit_cur = c->emit_cur;
    A.emit_ids = c->emit_ids;
    A.grp_sample_ids = c->grp_sample_ids.p;
    A.left_ptr = c->left_ptr.p;
    A.left_out = c->left_out.p;
    if (u) {
        A.user_ids = u->d_grp_sample_ids;
        A.user_left_ptr = u->d_left_ptr;
        A.user_left = u->d_left_ids;
    }
    int blocks = A.rows_gx * R + A.tile_blocks + R;
    if (c->offline || c->sub_mode) {  // rows in emit order; no leftovers (left_ptr was zeroed by odb_plan_query)
        // (a step range: the host may not know its row count yet; the blocks beyond it leave at once)
        const int64_t n_rows = std::max<int64_t>(c->sub_mode ? c->n_total : c->info.samples_emitted, 1);
        A.offline_row_blocks = (int)std::min<int64_t>((n_rows + kPrepThreads - 1) / kPrepThreads, (int64_t)c->sm_count * 8);
        A.user_ids = (u && !c->sub_mode) ? u->d_grp_sample_ids : nullptr;  // (a step range: written by k_sub_ids, local ids)
        if (u && u->d_left_ptr && !c->sub_mode) {
            A.job[A.n_jobs].dst = u->d_left_ptr;
            A.job[A.n_jobs].src = c->left_ptr.p;
            A.job[A.n_jobs].kind = 5;
            A.n_jobs++;
        }
        blocks = A.offline_row_blocks + A.tile_blocks;
    }
    k_prep<<<blocks, kPrepThreads, 0, st>>>(A);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

template <bool SHIFT, bool BULK>
static cudaError_t launch_collate_t(odb_ctx *c, const CollateArgs &args, cudaStream_t st) {
    const int v = (SHIFT ? 1 : 0) + (BULK ? 2 : 0);
    const size_t smem = BULK ? (size_t)(kColThreads / 32) * kColStage : 0;
    if (c->col_occ[v] == 0) {
        if (BULK) {
            cudaError_t e = cudaFuncSetAttribute(k_collate<SHIFT, BULK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->col_occ[v], k_collate<SHIFT, BULK>, kColThreads, smem);
        if (e != cudaSuccess) return e;
        if (c->col_occ[v] < 1) c->col_occ[v] = 1;
    }
    // tiles the launch can have to visit: known for a ranged launch, bounded by the caller's arena otherwise
    const int64_t n_tiles = args.tile_hi - args.tile_lo;
    if (n_tiles <= 0 && !args.whole) return cudaSuccess;
    const int blocks = (int)std::min<int64_t>(std::max<int64_t>((n_tiles + kColGrab - 1) / kColGrab, 1),
                                              (int64_t)c->sm_count * c->col_occ[v]);
    k_collate<SHIFT, BULK><<<blocks, kColThreads, smem, st>>>(args);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

cudaError_t launch_collate(odb_ctx *c, const CollateArgs &args, cudaStream_t st) {
    const bool sh = args.shift_labels != 0;
    if (c->collate_bulk) return sh ? launch_collate_t<true, true>(c, args, st) : launch_collate_t<false, true>(c, args, st);
    return sh ? launch_collate_t<true, false>(c, args, st) : launch_collate_t<false, false>(c, args, st);
}

cudaError_t launch_post(odb_ctx *c, const PostArgs &args, cudaStream_t st) {
    // the grid is sized by what the tables can hold (the host may not have seen the plan yet)
    const int64_t work = std::max<int64_t>((int64_t)c->grp_valid.cap, 1);
    int blocks = (int)std::min<int64_t>((work + 255) / 256, (int64_t)c->sm_count * 8);
    k_post<<<blocks, 256, 0, st>>>(args);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

}  // namespace odb
