// Collation kernels (rows A10, A11 of DESIGN.md): every emitted slot becomes a dense, right-padded
// [count x width] block in four arenas (input_ids, attention_mask, position_ids, labels), with the
// pad fill, label shift, span masking and the valid-token count fused.  sm_100a only.
//
// Paper: collate_fn P:28; pad to the group max P:416-420; valid tokens t_r of Eq. 2 P:60-63.
// Tensor contract: BASELINE.json north_star (readings U16-U18).
#include "odb_internal.cuh"

namespace odb {

#define ODB_LAUNCH_CHECK(c)                       \
    do {                                          \
        (c)->launches++;                          \
        cudaError_t e_ = cudaGetLastError();      \
        if (e_ != cudaSuccess) return e_;         \
    } while (0)

// ---------------------------------------------------------------------------------------------
// row descriptors: one warp per slot walks the slot's rows
// ---------------------------------------------------------------------------------------------
__global__ void k_row_desc(int R, int n_steps, const int64_t *__restrict__ rank_ptr, const int32_t *__restrict__ len,
                           const int64_t *__restrict__ sample_ptr, const int64_t *__restrict__ span_ptr,
                           const int32_t *__restrict__ span_lo, const int32_t *__restrict__ span_hi,
                           const int32_t *__restrict__ grp_count, const int64_t *__restrict__ grp_sample_ptr,
                           const int32_t *__restrict__ grp_sample_ids, RowDesc *__restrict__ rows,
                           int64_t *__restrict__ row_sp) {
    const int lane = threadIdx.x & 31;
    const int64_t n_slots = (int64_t)R * n_steps;
    const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; s < n_slots; s += warps) {
        const int r = (int)(s / n_steps);
        const int64_t base = rank_ptr[r];
        const int c = grp_count[s];
        const int64_t q0 = grp_sample_ptr[s];
        for (int j = lane; j < c; j += 32) {
            const int64_t g = base + grp_sample_ids[q0 + j];
            RowDesc d;
            d.tok = sample_ptr[g];
            d.len = len[g];
            const int64_t sp = span_ptr ? span_ptr[g] : 0;
            const int ns = span_ptr ? (int)(span_ptr[g + 1] - sp) : 0;
            d.nspan = ns;
            d.lo0 = ns > 0 ? span_lo[sp] : 0;
            d.hi0 = ns > 0 ? span_hi[sp] : 0;
            d.lo1 = ns > 1 ? span_lo[sp + 1] : 0;
            d.hi1 = ns > 1 ? span_hi[sp + 1] : 0;
            rows[q0 + j] = d;
            row_sp[q0 + j] = sp;
        }
    }
}

// tile t (elements [t*kColTile, (t+1)*kColTile) of the arenas) -> the slot that contains its first
// element.  One thread per slot fills the tiles that start inside the slot's [offset, next offset).
__global__ void k_tile_slots(int64_t n_slots, const int64_t *__restrict__ grp_offset, int32_t *__restrict__ tile_slot) {
    for (int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; s < n_slots; s += (int64_t)gridDim.x * blockDim.x) {
        const int64_t lo = grp_offset[s], hi = grp_offset[s + 1];
        for (int64_t t = (lo + kColTile - 1) / kColTile; t * kColTile < hi; ++t) tile_slot[t] = (int32_t)s;
    }
}

// ---------------------------------------------------------------------------------------------
// collate, version 1: direct global loads, 16-byte streaming stores.
// A warp covers 128 consecutive arena elements per iteration (lane = 4 elements = one int4 store
// per int32 arena and one 4-byte store of the uint8 mask); a CTA's 8 warps cover 1024 consecutive
// elements; a tile is 4 such iterations.  Block offsets are multiples of 16, so a lane's vector never
// straddles two slots.  Persistent CTAs stride over the tiles.
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

__device__ __forceinline__ bool masked_at(const RowRegs &r, int c, const CollateArgs &A, int64_t q) {
    if (r.nspan <= 2) return (c >= r.lo0 && c < r.hi0) || (c >= r.lo1 && c < r.hi1);
    const int64_t sp = A.row_sp[q];
    for (int j = 0; j < r.nspan; ++j)
        if (c >= A.span_lo[sp + j] && c < A.span_hi[sp + j]) return true;
    return false;
}

// one output element (row r, column c); used by the slow path
__device__ __forceinline__ void one_element(const CollateArgs &A, const RowRegs &r, int64_t q, int c, int32_t &id,
                                            int32_t &lab, int32_t &pos, uint32_t &m) {
    const int32_t *tp = A.tokens + r.tok;
    const bool real = c < r.len;
    id = real ? __ldg(tp + c) : A.pad_id;
    pos = real ? c : 0;
    m = real ? 1u : 0u;
    if (A.shift_labels) {
        const bool ok = (c + 1 < r.len) && !masked_at(r, c + 1, A, q);
        lab = ok ? __ldg(tp + c + 1) : A.ignore_index;
    } else {
        const bool ok = real && !masked_at(r, c, A, q);
        lab = ok ? id : A.ignore_index;
    }
}

__global__ void __launch_bounds__(kColThreads, 4) k_collate_v1(const CollateArgs A) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int kWarps = kColThreads / 32;
    constexpr int kIters = kColTile / (kWarps * 128);
    for (int64_t tile = A.tile_lo + blockIdx.x; tile < A.tile_hi; tile += gridDim.x) {
        int64_t s = A.tile_slot[tile];
        int64_t off_s = A.grp_offset[s], off_n = A.grp_offset[s + 1];
        int64_t s_loaded = -1;
        uint32_t W = 0, area = 0;
        int64_t sp_s = 0;
        int acc = 0;
        int64_t acc_slot = -1;
#pragma unroll 1
        for (int it = 0; it < kIters; ++it) {
            const int64_t a = tile * kColTile + (int64_t)(it * kWarps + warp) * 128 + lane * 4;
            if (a >= A.total_elems) break;
            while (a >= off_n) {
                ++s;
                off_s = off_n;
                off_n = A.grp_offset[s + 1];
            }
            if (s != s_loaded) {
                W = (uint32_t)A.grp_width[s];
                area = (uint32_t)A.grp_count[s] * W;
                sp_s = A.grp_sample_ptr[s];
                s_loaded = s;
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
            if (t + 4 <= W) {
                // fast path: the vector lies inside one row (and therefore inside the block)
                const int64_t q = sp_s + b;
                const RowRegs r = load_row(A.rows, q);
                const int32_t *tp = A.tokens + r.tok + t;
                const int nreal = max(0, min(5, r.len - (int)t));  // tokens t .. t+4 that exist
                int32_t v[5];
#pragma unroll
                for (int j = 0; j < 5; ++j) v[j] = (j < nreal) ? __ldg(tp + j) : A.pad_id;
                int4 oid, olab, opos;
                uint32_t om = 0;
                int32_t lab[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int c = (int)t + j;
                    const bool real = c < r.len;
                    if (real) om |= 1u << (8 * j);
                    if (A.shift_labels) {
                        const bool ok = (c + 1 < r.len) && !masked_at(r, c + 1, A, q);
                        lab[j] = ok ? v[j + 1] : A.ignore_index;
                    } else {
                        const bool ok = real && !masked_at(r, c, A, q);
                        lab[j] = ok ? v[j] : A.ignore_index;
                    }
                    acc += (lab[j] != A.ignore_index) ? 1 : 0;
                }
                oid = make_int4(v[0], v[1], v[2], v[3]);  // v[j] is pad_id beyond the sample
                opos = make_int4((int)t < r.len ? (int)t : 0, (int)t + 1 < r.len ? (int)t + 1 : 0,
                                 (int)t + 2 < r.len ? (int)t + 2 : 0, (int)t + 3 < r.len ? (int)t + 3 : 0);
                olab = make_int4(lab[0], lab[1], lab[2], lab[3]);
                __stcs(reinterpret_cast<int4 *>(A.ids + a), oid);
                __stcs(reinterpret_cast<int4 *>(A.labels + a), olab);
                __stcs(reinterpret_cast<int4 *>(A.pos + a), opos);
                __stcs(reinterpret_cast<unsigned int *>(A.mask + a), om);
            } else {
                // slow path: the vector crosses a row end and / or the end of the block
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
                    one_element(A, r, q, c, id, lb, ps, m);
                    A.ids[a + j] = id;
                    A.labels[a + j] = lb;
                    A.pos[a + j] = ps;
                    A.mask[a + j] = (uint8_t)m;
                    acc += (lb != A.ignore_index) ? 1 : 0;
                }
            }
        }
        // A11: one integer atomic per warp per tile when the whole warp stayed in one slot
        const int64_t slot0 = __shfl_sync(ODB_FULL_MASK, acc_slot, 0);
        const bool same = __all_sync(ODB_FULL_MASK, acc_slot == slot0);
        if (same) {
            const int tot = __reduce_add_sync(ODB_FULL_MASK, acc);
            if (lane == 0 && tot != 0) atomicAdd(&A.grp_valid[slot0], tot);
        } else if (acc) {
            atomicAdd(&A.grp_valid[acc_slot], acc);
        }
    }
}

// step_valid_tokens[k] = sum over ranks of grp_valid_tokens[r][k]  (Eq. 2's T_tok per step)
__global__ void k_step_valid(int R, int n_steps, const int32_t *__restrict__ grp_valid, int64_t *__restrict__ step_valid) {
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_steps; k += gridDim.x * blockDim.x) {
        long long s = 0;
        for (int r = 0; r < R; ++r) s += grp_valid[(int64_t)r * n_steps + k];
        step_valid[k] = s;
    }
}

// ---------------------------------------------------------------------------------------------
// host launchers
// ---------------------------------------------------------------------------------------------
cudaError_t launch_row_desc(odb_ctx *c, const int64_t *d_sample_ptr, const int64_t *d_span_ptr,
                            const int32_t *d_span_lo, const int32_t *d_span_hi, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    const int64_t n_slots = (int64_t)R * c->n_steps;
    if (n_slots == 0) return cudaSuccess;
    int blocks = (int)std::min<int64_t>((n_slots * 32 + 255) / 256, (int64_t)c->sm_count * 8);
    k_row_desc<<<blocks, 256, 0, st>>>(R, c->n_steps, c->d_rank_ptr, c->d_lengths, d_sample_ptr, d_span_ptr, d_span_lo,
                                       d_span_hi, c->grp_count.p, c->grp_sample_ptr.p, c->grp_sample_ids.p, c->rows.p,
                                       c->row_sp.p);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

cudaError_t launch_tile_slots(odb_ctx *c, int64_t n_tiles, cudaStream_t st) {
    const int64_t n_slots = (int64_t)c->prm.n_ranks * c->n_steps;
    if (n_slots == 0 || n_tiles == 0) return cudaSuccess;
    int blocks = (int)std::min<int64_t>((n_slots + 255) / 256, (int64_t)c->sm_count * 8);
    k_tile_slots<<<blocks, 256, 0, st>>>(n_slots, c->grp_offset.p, c->tile_slot.p);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

cudaError_t launch_collate(odb_ctx *c, const CollateArgs &args, cudaStream_t st) {
    const int64_t n_tiles = args.tile_hi - args.tile_lo;
    if (n_tiles <= 0) return cudaSuccess;
    static int occ = 0;
    if (occ == 0) {
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_collate_v1, kColThreads, 0);
        if (e != cudaSuccess) return e;
        if (occ < 1) occ = 1;
    }
    int blocks = (int)std::min<int64_t>(n_tiles, (int64_t)c->sm_count * occ);
    k_collate_v1<<<blocks, kColThreads, 0, st>>>(args);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

cudaError_t launch_step_valid(odb_ctx *c, int64_t *d_step_valid, cudaStream_t st) {
    if (c->n_steps == 0) return cudaSuccess;
    int blocks = std::min((c->n_steps + 255) / 256, c->sm_count * 4);
    k_step_valid<<<blocks, 256, 0, st>>>(c->prm.n_ranks, c->n_steps, c->grp_valid.p, d_step_valid);
    ODB_LAUNCH_CHECK(c);
    return cudaSuccess;
}

}  // namespace odb
