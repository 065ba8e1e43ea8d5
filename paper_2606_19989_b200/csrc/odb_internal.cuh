// Internal declarations shared by the translation units of libodb (CUDA path only).
// Nothing here is used by, or shared with, the CPU oracle under oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <atomic>
#include <vector>

#include "odb.h"

#define ODB_FULL_MASK 0xffffffffu

namespace odb {

// ---------------------------------------------------------------------------------------------
// compile-time configuration
// ---------------------------------------------------------------------------------------------
constexpr int kSortChunk = 4096;    // keys sorted in shared memory by one CTA (A1)
constexpr int kSortThreads = 512;
constexpr int kMergeThreads = 256;
constexpr int kRankThreads = 1024;  // one CTA per rank for A2..A8
constexpr int kCommitParts = 4;     // CTAs per rank that share k_commit's scan-free fast path
constexpr size_t kFormSmemLimit = 231424;  // dynamic shared memory of k_form_groups_smem (227 KB - static)
constexpr int kAlignSmemKeys = 8192;       // overflow sort keys kept in shared memory by k_align
constexpr int kFinThreads = 512;           // k_fin_scan: tile = kFinThreads * kFinItems slots
constexpr int kFinItems = 1;
constexpr int kFinTile = kFinThreads * kFinItems;
constexpr int kColThreads = 256;    // collate CTA (A10)
constexpr int kColTile = 4096;      // arena elements per collate tile (one CTA iteration)
constexpr int kColChunk = 512;      // arena elements per warp per tile (one 16-element unit per lane)
constexpr int kColGrab = 16;        // tiles a CTA takes from the work counter at a time
constexpr int kTimingRing = 64;     // timed runs whose stage events are kept (odb_get_timing_at)

// Per-round status record: written by the round's kernels, copied to pinned host memory (A7).
struct RoundRec {
    int32_t T;           // Eq. 3 target of the round
    int32_t T_emit;      // steps actually emitted (== T unless the quota cut fired)
    int32_t quota_hit;   // 1 if the non-join sample quota was reached in this round
    int32_t n_finished;  // ranks that will be "finished" (status -1) at the start of the next round
    int32_t bad_length;  // some length < 1 was seen
    int32_t done;        // distributed mode: the world summary of this round says "terminated" (no emission)
    int64_t emitted_round;  // samples emitted in this round over all ranks
};

// Sizes of the plan, DEVICE-RESIDENT: written by the planning kernels (the host uploads the first four
// fields in the staged path, where it has read them round by round), read by every later kernel, so that
// nothing after the round loop needs a size from the host.  A pinned host copy is filled by the slot scan.
struct PlanDims {
    int32_t n_steps;      // slots per rank
    int32_t n_rounds;     // protocol rounds including the terminal check
    int32_t stop_reason;  // ODB_STOP_*
    int32_t complete;     // 1 = the protocol has terminated: the tables may be finalised and collated
    int32_t err;          // ODB_ERR_CAPACITY flagged by the slot scan against the caller's capacities
    int32_t bad_length;
    int64_t n_slots;
    int64_t total_elems;
    int64_t samples_emitted;
    int64_t padded_elems;
    unsigned long long real_tokens;
    int64_t samples_left;
};

// Result of the speculative, round-parallel planner (k_spec_form): the protocol rounds [0, j_star) have been
// formed under the assumption "no leftovers so far", which holds as long as no round overflows; round j_star
// is the first that does (the sequential round loop resumes there) or the terminal check (complete = 1).
struct SpecRec {
    int32_t j_star;    // rounds committed by k_spec_commit
    int32_t n_steps;   // steps those rounds emit (sum of their T)
    int32_t complete;  // 1 = round j_star is the terminal check: the protocol is over
    int32_t pad_;
};

// The caller's output capacities, checked on the device by the slot scan (odb_run enqueues the collate
// kernels before the host has seen the plan sizes).
struct CapCheck {
    int64_t arena, slots, ids, steps, left;  // < 0 = not checked
    int64_t tiles;                           // capacity of the library's tile table
};

// State of one tile of the slot scan (decoupled look-back): flag 0 = nothing, 1 = agg valid,
// 2 = inc (inclusive prefix) valid.
struct __align__(16) ScanTile {
    long long agg[4];
    long long inc[4];
    int flag;
    int pad_[3];
};

// One emitted row (sample) as the collate kernel wants it: 32 bytes, two 16-byte loads.
struct __align__(16) RowDesc {
    int64_t tok;    // offset of the sample's first token in d_tokens
    int32_t len;    // realized length
    int32_t nspan;  // number of masked spans; the first two are inlined below
    int32_t lo0, hi0, lo1, hi1;
};

// Where a 4096-element tile of the arenas starts: the slot that holds the tile's first element (or the
// alignment gap behind that slot's block) and its geometry.  32 bytes, two 16-byte loads; a warp derives
// (row, column) of its own 512-element chunk from it with one division.
struct __align__(16) TileRec {
    int64_t off_s;   // grp_offset of the slot
    int32_t slot;
    uint32_t W;      // grp_width
    uint32_t area;   // count * width
    uint32_t sp_s;   // grp_sample_ptr of the slot (index of its first row)
    uint32_t pad_[2];
};

struct CollateArgs {
    const int32_t *tokens;
    const RowDesc *rows;
    const int64_t *row_sp;  // first span index of each row (only read when nspan > 2)
    const int32_t *span_lo;
    const int32_t *span_hi;
    const int64_t *grp_offset;      // n_slots + 1
    const int64_t *grp_sample_ptr;  // n_slots + 1
    const int32_t *grp_count;
    const int32_t *grp_width;
    const TileRec *tiles;
    const PlanDims *dims;  // non-NULL: the launch covers the whole arena, whose size is read on the device
    int32_t *ids;
    int32_t *labels;
    int32_t *pos;
    uint8_t *mask;
    int32_t *grp_valid;
    unsigned long long *tile_counter;  // work counter of the launch (zeroed before it)
    int64_t total_elems;       // arena elements [elem_lo, total_elems) are written by this launch
    int64_t elem_lo;
    int64_t tile_lo, tile_hi;  // tiles [tile_lo, tile_hi) are visited by this launch
    int32_t pad_id, ignore_index, shift_labels;
    int32_t whole;  // 1: the launch covers the whole arena, extent read from dims (skipped if the plan is not usable)
};

// k_post: the per-step valid-token totals and the caller's valid-token tables
struct PostArgs {
    int R;
    const PlanDims *dims;
    const int32_t *grp_valid;
    int64_t *step_valid;
    int64_t *user_step_valid;
    int32_t *user_grp_valid;
};

// growable device buffer (cudaMalloc on growth only)
// cudaMalloc calls made by the growable tables below, process-wide (diagnostics: odb_debug_read(ctx, 5, ..); a test
// uses it to show that a pass of step ranges does not allocate after its first range)
inline std::atomic<long long> g_table_allocs{0};

template <class T>
struct DevBuf {
    T *p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t n, bool zero = false, cudaStream_t st = 0) {
        if (n <= cap) return cudaSuccess;
        if (p) {
            cudaError_t e = cudaFree(p);
            p = nullptr;
            cap = 0;
            if (e != cudaSuccess) return e;
        }
        size_t want = n + n / 4 + 16;
        g_table_allocs.fetch_add(1, std::memory_order_relaxed);
        cudaError_t e = cudaMalloc((void **)&p, want * sizeof(T));
        if (e != cudaSuccess) {
            p = nullptr;
            return e;
        }
        cap = want;
        if (zero) return cudaMemsetAsync(p, 0, want * sizeof(T), st);
        return cudaSuccess;
    }
    void release() {
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
    }
};

}  // namespace odb

// A second (and third) set of the rank-major plan tables: odb_collate_steps builds the self-contained plan of a
// STEP RANGE in one of them (swapped in for the duration of the enqueue), so the full plan's tables stay valid
// and two step ranges can be in flight at once (double-buffered streaming output).
struct SubTabs {
    odb::DevBuf<int32_t> grp_count, grp_width, grp_round, grp_valid, grp_real, grp_origin;
    odb::DevBuf<unsigned char> scan_state;
    odb::DevBuf<int64_t> grp_offset, grp_sample_ptr;
    odb::DevBuf<int32_t> grp_sample_ids, left_out;
    odb::DevBuf<int64_t> left_ptr, step_valid;
    odb::DevBuf<odb::RowDesc> rows;
    odb::DevBuf<int64_t> row_sp;
    odb::DevBuf<odb::TileRec> tiles;
    odb::PlanDims *d_dims = nullptr, *h_dims = nullptr;
    unsigned long long *d_tile_counter = nullptr;
    cudaEvent_t ev_plan = nullptr;
    bool ready = false;
};

// The context.  Host-side state machine + device scratch.
struct odb_ctx {
    odb_params prm;
    int device = 0;
    int64_t n_max = 0;  // max_samples_total
    int sm_count = 148;
    int last_cuda_error = 0;
    int64_t launches = 0;
    int timing = 0;
    // timing: a ring of kTimingRing event quadruples, one per timed run, so that a caller can read the stage
    // times of many back-to-back runs AFTER they have all been enqueued (no per-step wait)
    std::vector<cudaEvent_t> evring;  // 4 * kTimingRing, created by odb_set_timing
    int64_t ev_seq = 0;               // timed runs completed (ev[3] recorded) since odb_set_timing
    cudaEvent_t *ev = nullptr;        // the current run's quadruple inside evring
    bool ev_valid = false;
    cudaEvent_t ev_status = nullptr;
    cudaStream_t last_stream = nullptr;
    int col_occ[4] = {0, 0, 0, 0};  // resident collate CTAs per SM (shift 0 / 1, + 2 for the bulk-store form)
    bool collate_bulk = false;      // odb_set_option(ODB_OPT_COLLATE_BULK_STORES)
    bool attr_form = false, attr_form_hier = false, attr_align = false, attr_sort = false, attr_sort8 = false;  // cudaFuncSetAttribute done
    bool no_cluster_sort = false;  // the cluster sort could not be launched on this device: use the fallback
    bool begin_pending = false;    // a run has started and its per-run device state is not cleared yet
    bool no_rounds_kernel = false; // the persistent round-loop kernel could not be launched on this device
    int rounds_max_ctas = 0;       // resident CTAs of k_rounds on this device (0 = not asked yet, -1 = no cooperative launch)
    int32_t *gs_rounds = nullptr;  // k_rounds: the double-buffered per-round summary + the grid-barrier counter
    odb::DevBuf<int32_t> spec_tab;  // round-parallel planner: SpecRec, per-round T / step base / arrival counters, G table
    int spec_occ = 0;               // k_spec_form's shared-memory attribute is set
    bool round_parallel = true;     // odb_set_option(ODB_OPT_ROUND_PARALLEL)
    bool spec_used = false;         // the last run went through the round-parallel planner (spec_tab holds its SpecRec)
    int32_t dist_spec_rounds = 0;   // distributed mode: rounds formed by odb_dist_spec_form (state 7 / 8)
    int32_t *dist_spec_G = nullptr; //   ... their local G table inside spec_tab
    int32_t *h_spec = nullptr;      // pinned: SpecRec + the committed rounds' T (read back by odb_dist_spec_status)

    // inputs fixed by the first odb_form_groups after create / reset
    const int32_t *d_lengths = nullptr;
    std::vector<int64_t> h_rank_ptr;
    int64_t n_total = 0;
    int32_t max_nr = 0;

    // distributed layout (odb_dist_config): this context holds ranks [rank_offset, rank_offset + R) of
    // world_ranks; 0 = single-process mode
    int32_t world_ranks = 0, rank_offset = 0, world_max_window = 0, gs_world_cap = 0;
    int32_t round_window = 0;  // step totals this round may touch: step_samples[n_steps .. n_steps + round_window)
    int32_t *gs_local = nullptr;  // 2 R: (G_r, S_r) pairs of the local ranks, input of the all_gather
    int32_t *gs_world = nullptr;  // 2 world_ranks: the gathered pairs

    // state machine: 0 = fresh, 1 = groups formed, 2 = aligned (status pending), 3 = status read,
    // 4 = terminated, 5 = plan queried, 6 = aligned but not committed (distributed mode)
    int state = 0;
    int32_t round = 0;     // rounds fully processed (emitting rounds)
    int32_t n_rounds = 0;  // including the terminal check once terminated
    int32_t n_steps = 0;
    int64_t samples_emitted = 0;
    int32_t n_finished = 0;
    int32_t last_T = 0;
    int stop_reason = 0;
    odb_plan_info info;
    bool info_valid = false;

    // device scratch sized by n_max (+ R)
    int64_t *d_rank_ptr = nullptr;      // R+1
    uint64_t *keyA = nullptr, *keyB = nullptr;  // n_max
    uint64_t *sorted = nullptr;         // = keyA or keyB after the merge passes
    uint64_t *ovf = nullptr;            // 2*n_max + 2 (overflow sort keys)
    int32_t *jA = nullptr, *jB = nullptr;  // n_max + R
    uint8_t *mark = nullptr;            // n_max + R
    uint8_t *posflag = nullptr;         // n_max
    int32_t *emit_pos = nullptr;        // n_max: index in the rank's emit region, -1 = not emitted
    int32_t *gpos = nullptr;            // n_max + R
    int32_t *agpos = nullptr, *agcnt = nullptr, *agoff = nullptr, *agorg = nullptr;  // n_max + R
    int32_t *left_ids = nullptr, *emit_ids = nullptr;              // n_max
    int32_t *n_left = nullptr, *fetch_pos = nullptr, *emit_cur = nullptr, *G = nullptr, *S = nullptr;  // R
    int32_t *emit_snap = nullptr;  // R: emit_cur as seen by k_align (read by every CTA of k_commit)
    int32_t *d_arrived = nullptr;  // R: views of the rank's stream that have arrived (odb_set_available)
    std::vector<int32_t> h_arrived;
    std::vector<int32_t> h_arrived_dev;  // what d_arrived holds (empty = unknown)
    bool dev_rank_ptr_valid = false;     // d_rank_ptr holds h_rank_ptr
    cudaStream_t dev_meta_stream = nullptr;  // ... uploaded on this stream
    bool arrived_set = false;
    odb::RoundRec *d_rec = nullptr;
    odb::RoundRec *h_rec = nullptr;  // pinned
    odb::PlanDims *d_dims = nullptr;
    odb::PlanDims *h_dims = nullptr;     // pinned: the device's sizes, copied back behind the slot scan
    odb::PlanDims *h_dims_up = nullptr;  // pinned: the host's sizes on their way up (staged path)
    unsigned int *d_done_ctr = nullptr;  // "last CTA" counter of k_commit (self-resetting)
    cudaEvent_t ev_plan = nullptr;       // recorded behind the slot scan's read-back
    unsigned long long *d_tile_counter = nullptr;
    int fin_epoch = 0;                   // launch counter of k_fin_scan (tags its tile flags)
    bool rec_clean = false;              // d_rec was cleared by the slot scan of the last (complete) plan ...
    cudaStream_t rec_clear_stream = nullptr;  // ... enqueued on this stream

    // step-major staging tables [step * R + r], growable
    odb::DevBuf<int32_t> st_count, st_width, st_real, st_round, st_origin, step_samples;
    int64_t step_cap = 0;

    // rank-major plan tables built by odb_plan_query
    odb::DevBuf<int32_t> grp_count, grp_width, grp_round, grp_valid, grp_real, grp_origin;
    bool collated = false;  // grp_valid holds the counts of a completed collate
    odb::DevBuf<unsigned char> scan_state;
    odb::DevBuf<int64_t> grp_offset, grp_sample_ptr;
    odb::DevBuf<int32_t> grp_sample_ids, left_out;
    odb::DevBuf<int64_t> left_ptr, step_valid;
    odb::DevBuf<odb::RowDesc> rows;
    odb::DevBuf<int64_t> row_sp;
    odb::DevBuf<odb::TileRec> tiles;

    // step-range plans (odb_collate_steps)
    SubTabs sub[2];
    int sub_seq = 0;
    bool sub_mode = false;     // the tables swapped in belong to a step range: rows are gathered through the slot CSR
    int32_t sub_step_lo = 0;   // its first step

    // offline planners (odb_offline.cu): the plan's slots hold GLOBAL sample ids
    bool offline = false;
    int offline_planner = 0, offline_size = 0, offline_bs = 0;
    int64_t offline_G = 0;             // batches in the global list (GMT / BMT)
    const int32_t *offline_perm = nullptr;
    odb::DevBuf<int64_t> of_seg_ptr;   // nseg + 1
    odb::DevBuf<int32_t> of_seg_i32;   // 5 x nseg: zeros (n_left), zeros (fetch_pos), zeros (emit_cur), "all arrived", S; then G, boff (nseg + 1)
    odb::DevBuf<int32_t> of_plen;      // N: lengths in list order; later the batch-shuffle keys
    odb::DevBuf<int32_t> of_gpos;      // N + nseg + 1
    odb::DevBuf<int32_t> of_bstart, of_bcnt, of_border;  // per batch: first position in the sorted keys, count; the shuffled order
    odb::DevBuf<uint64_t> of_keyA, of_keyB;               // the batch shuffle's sort buffers
    uint64_t *of_sorted = nullptr;

    // device staging for odb_run_host
    odb::DevBuf<int32_t> hs_lengths, hs_tokens, hs_span_lo, hs_span_hi, hs_ids, hs_labels, hs_pos;
    odb::DevBuf<int64_t> hs_sample_ptr, hs_span_ptr;
    odb::DevBuf<uint8_t> hs_mask;
    cudaStream_t aux_stream = nullptr;   // collate preparation: chunk table + id tables beside the row descriptors
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaStream_t copy_stream = nullptr;  // host -> device
    cudaStream_t d2h_stream = nullptr;   // device -> host
    cudaEvent_t copy_ev = nullptr;
    std::vector<cudaEvent_t> ev_pool;         // odb_run_host: tokens landed / rank collated / piece collated / piece copied
    odb::DevBuf<unsigned long long> piece_ctr;  // one work counter per output piece
    int64_t host_staging_elems = 1ll << 25;   // arena elements per staging piece (ODB_OPT_HOST_STAGING_ELEMS)
    bool host_device_arenas = false;          // odb_run_host: the four arenas of `h_out_bufs` are DEVICE memory
    int64_t *h_rank_off = nullptr;            // pinned, R+1: arena offset of each rank's first slot
};

namespace odb {
// ---- launchers implemented in odb_plan.cu ----------------------------------------------------
cudaError_t launch_begin(odb_ctx *c, cudaStream_t st);  // per-run state reset + length validation
cudaError_t flush_begin(odb_ctx *c, cudaStream_t st);   // ... if no sort launch has done it
cudaError_t launch_round_form(odb_ctx *c, cudaStream_t st);   // A0..A3
// A0 + A1 in one launch (odb_sort.cu): cluster merge sort; cudaErrorNotSupported for windows > 65536 keys
cudaError_t launch_sort_window(odb_ctx *c, int maxS, bool first, cudaStream_t st);
cudaError_t launch_round_align(odb_ctx *c, cudaStream_t st);  // A4..A8a + commit (single-process mode)
// every protocol round in one cooperative launch; cudaErrorNotSupported if R CTAs cannot be resident
// `spec_rounds` > 0: the rounds [0, spec_rounds) are first formed and committed round-parallel (k_spec_form /
// k_spec_commit) and the persistent kernel resumes where that speculation stops
// (spec_terminal: the round behind them is the terminal check -- false when a sample quota ends the speculation)
cudaError_t launch_rounds(odb_ctx *c, int spec_rounds, bool spec_terminal, cudaStream_t st);
// scratch entries per rank-sized table (gpos, agpos, ...): every (rank, round) window of the round-parallel
// planner owns S + 1 entries
inline size_t plan_table_entries(size_t N, size_t R) { return N + N / 8 + 2 * R + 64; }
constexpr int kSpecMinWindow = 8;       // smallest buffer_size the round-parallel planner takes
constexpr int kSpecMaxRounds = 65535;   // (gridDim.y)
cudaError_t launch_pack_summary(odb_ctx *c, cudaStream_t st);   // distributed: (G_r, S_r) pairs for the all_gather
// distributed, batched exchange: the local G table of the rounds [0, n_rounds); then, from the gathered tables,
// Eq. 3 of every round, split + commit of the rounds before the first that overflows, the rank state behind them
cudaError_t launch_dist_spec_form(odb_ctx *c, int n_rounds, int32_t **G_tab_out, cudaStream_t st);
cudaError_t launch_dist_spec_commit(odb_ctx *c, int n_rounds, const int32_t *d_G_world, const int32_t *d_n_world, int n_procs,
                                    cudaStream_t st);
cudaError_t launch_align_only(odb_ctx *c, cudaStream_t st);     // distributed: A4..A6 from the world summary
cudaError_t launch_commit_only(odb_ctx *c, cudaStream_t st);    // distributed: A7 + A8a after the all_reduce
// A9: rank-major tables, offsets, totals (sizes from the device-resident PlanDims)
// (step_lo: the slot scan covers the steps [step_lo, step_lo + PlanDims.n_steps) of the staging tables;
//  slots_alloc: size the scan's tile records for at least that many slots, so that later, larger scans do not grow them)
cudaError_t launch_finalize(odb_ctx *c, int64_t slots_bound, const CapCheck &cap, int64_t *rank_off, cudaStream_t st,
                            int64_t step_lo = 0, int64_t slots_alloc = 0);
// step-range plans: PlanDims of the range, and the slot CSR's ids of its rows (global in the library's table, local
// in the caller's)
cudaError_t launch_sub_dims(odb_ctx *c, int n_steps, cudaStream_t st);
// (full_sp: the full plan's grp_sample_ptr over full_K steps per rank when it exists, else NULL)
cudaError_t launch_sub_ids(odb_ctx *c, int step_lo, int32_t *user_ids, const int64_t *full_sp, int full_K, cudaStream_t st);
// ---- segment-level pieces shared with the offline planners (odb_offline.cu) -------------------------
struct SortArgs;
cudaError_t launch_sort_segments(odb_ctx *c, const SortArgs &A, int64_t nseg, int maxS, cudaStream_t st);
cudaError_t sort_segments_any(odb_ctx *c, const SortArgs &A, int64_t nseg, int maxS, uint64_t *keyB, uint64_t **sorted,
                              cudaStream_t st);
cudaError_t form_segments_maxfit(odb_ctx *c, const uint64_t *sorted, const int64_t *seg_ptr, const int32_t *S_arr,
                                 int64_t nseg, int maxS, int32_t *jA, int32_t *jB, uint8_t *mark, int32_t *gpos,
                                 int32_t *G_out, cudaStream_t st);
// ---- odb_offline.cu -------------------------------------------------------------------------------
cudaError_t offline_build(odb_ctx *c, const odb_offline_params *P, const int32_t *d_lengths, int64_t N, cudaStream_t st);
cudaError_t offline_slots(odb_ctx *c, cudaStream_t st);
cudaError_t launch_offline_ids(odb_ctx *c, cudaStream_t st);
// ---- launchers implemented in odb_collate.cu -------------------------------------------------
// collate preparation in ONE launch: row descriptors, tile table, slot-id / leftover tables, table copies
cudaError_t launch_prep(odb_ctx *c, const int64_t *d_sample_ptr, const int64_t *d_span_ptr, const int32_t *d_span_lo,
                        const int32_t *d_span_hi, const odb_outputs *user, cudaStream_t st);
cudaError_t launch_collate(odb_ctx *c, const CollateArgs &args, cudaStream_t st);
cudaError_t launch_post(odb_ctx *c, const PostArgs &args, cudaStream_t st);
// ---- odb_scale.cu ------------------------------------------------------------------------------
cudaError_t launch_loss_weights(odb_ctx *c, int mode, double *d_weights, cudaStream_t st);
cudaError_t launch_loss_numerators(odb_ctx *c, int mode, double *d_num, cudaStream_t st);
cudaError_t launch_loss_normalize(odb_ctx *c, const double *d_num_world, int world_ranks, int rank_offset,
                                  double *d_weights, cudaStream_t st);
}  // namespace odb
