/*
 * odb.h -- C ABI of the B200-native ODB hot path: group -> align -> collate.
 *
 * What it computes (paper: "Online Dynamic Batching", /root/reference/PAPER.md, cited P:<line>):
 *   for R data-parallel ranks (virtual ranks: independent segments on ONE GPU), given the realized
 *   post-tokenization sample lengths and the ragged token buffers,
 *     1. per rank, sort the buffered window by length and form variable-size token-budget groups
 *        (section 2.2, Eq. 1; worked example App. D);
 *     2. align the per-rank group counts to the common target T_grp with the Max-Based
 *        Bidirectional Group Alignment protocol (section 2.3; Eq. 3; Alg. 1):
 *        split upward, overflow + recirculation downward, IDLE slots for finished ranks,
 *        join (default, Thm 1) or non-join termination with sample-quota closure (Thm 2);
 *     3. collate every aligned group into padded tensors input_ids / attention_mask /
 *        position_ids / labels (collate_fn P:28; pad to the group max P:416-420) and count the
 *        valid tokens per group for token-level loss scaling (Eq. 2).
 *   All work is integer / index work; results are bit-exact and run-to-run deterministic.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The caller owns every
 *     buffer it passes; the library never frees or reallocates them.  The library owns only the
 *     scratch inside odb_ctx.
 *   - `stream` is a cudaStream_t passed as void* (0 = the legacy default stream).  Kernel launches
 *     are asynchronous on it; the calls documented as "synchronises" wait for that stream.
 *   - Samples are laid out rank-major: rank r owns samples h_rank_ptr[r] .. h_rank_ptr[r+1]-1 in
 *     sampler order; a "local id" is the index inside the rank.
 *   - d_sample_ptr[g] .. d_sample_ptr[g+1] are the token offsets of global sample g in d_tokens and
 *     must equal the prefix sum of d_lengths.  d_tokens must be 16-byte aligned; a buffer of exactly n_tokens
 *     words is enough.  The collate kernel fetches tokens with aligned 16-byte loads, so when n_tokens is not a
 *     multiple of 4 the 16-byte unit that holds the last token is read whole: that unit starts at a 16-byte
 *     boundary inside the caller's mapping and cannot cross a page, so the load cannot fault; the up to 3 words
 *     behind the last token are whatever the caller keeps there, and they are discarded, never copied to an output
 *     (tests/test_gpu_parity.py::test_token_buffer_of_exactly_n_tokens).
 *   - Masked spans (labels -> ignore_index) are CSR per sample: spans d_span_ptr[g] .. d_span_ptr[g+1]-1,
 *     half-open [lo,hi) token positions, sorted and disjoint.
 *   - Every call returns an ODB_* status (0 = OK).  No exceptions, no abort, nothing printed.
 *   - There is no CPU fallback: without a CUDA device odb_create returns ODB_ERR_CUDA.
 *
 * Output layout
 *   Slot index s = r * n_steps + k (rank-major; step k of rank r).  Every rank holds exactly
 *   n_steps slots; an IDLE slot has count 0 and width 0 (reading U14).  Slot s is a dense
 *   row-major [grp_count[s] x grp_width[s]] block, right-padded, placed at element offset
 *   grp_offset[s] (a multiple of 16) in each of the four arenas; the <= 15 gap elements between
 *   blocks are never written.  Rows are the group's samples ascending by (length, local id).
 */
#ifndef ODB_H_
#define ODB_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* exported symbol (the library is built with -fvisibility=hidden) */
#if defined(__GNUC__)
#define ODB_API __attribute__((visibility("default")))
#else
#define ODB_API
#endif

typedef struct odb_ctx odb_ctx;

enum {
    ODB_OK = 0,
    ODB_ERR_INVALID_ARG = 1,
    ODB_ERR_BAD_LENGTH = 2, /* some length < 1 */
    ODB_ERR_CAPACITY = 3,   /* an output arena or table is too small; nothing is written past capacity */
    ODB_ERR_CUDA = 4,       /* a CUDA call failed (odb_last_cuda_error gives the code) */
    ODB_ERR_STATE = 5       /* call order violated */
};
enum {
    ODB_RULE_THRESHOLD = 0, /* paper section 2.2: threshold carry-over greedy (default) */
    ODB_RULE_MAXFIT_ASC = 1 /* App. I: longest ascending run with count*max_len <= budget */
};
enum { /* loss-scaling modes (section 2.3; App. B) */
    ODB_SCALE_SAMPLE = 1,       /* w = n_{r,k} / N_k */
    ODB_SCALE_TOKEN_APPROX = 2, /* w from t_adj = n_adj * (t_orig / n_orig) of the slot's candidate group */
    ODB_SCALE_TOKEN_EXACT = 3   /* Eq. 2: w = t_{r,k} / T_tok,k from post-alignment valid-token counts (default) */
};
enum {
    ODB_STOP_ALL_FINISHED = 0, /* join: every rank drained (Thm 1) */
    ODB_STOP_LOGICAL = 1,      /* non-join: some rank advertised "finished" */
    ODB_STOP_QUOTA = 2         /* non-join: cumulative emitted samples reached sample_quota (Thm 2) */
};

typedef struct {
    int32_t n_ranks;        /* R = W >= 1 */
    int32_t rule;           /* ODB_RULE_* */
    int32_t join_mode;      /* 1 = join (default), 0 = non-join */
    int32_t buffer_size;    /* per-round window per rank (the paper's grouping buffer); 0 = all */
    int32_t slot_capacity;  /* C_r, output slots per round (Eq. 3); 0 = unlimited */
    int32_t pad_id;         /* input_ids pad value */
    int32_t ignore_index;   /* label of pad / masked positions (-100) */
    int32_t shift_labels;   /* 1: labels[t] = token t+1 (default); 0: labels[t] = token t */
    int64_t budget;         /* L_max, 1 .. 2^31-1 */
    int64_t sample_quota;   /* non-join only; <= 0 = no quota */
    int64_t emitted_so_far; /* non-join only; S_emit carried in from earlier logical iterations */
} odb_params;

typedef struct { /* host-side; filled by odb_plan_query / odb_run */
    int32_t n_rounds;    /* protocol rounds including the terminal check */
    int32_t n_steps;     /* slots per rank = sum over rounds of T_grp */
    int32_t stop_reason; /* ODB_STOP_* */
    int32_t reserved;
    int64_t n_slots;         /* R * n_steps */
    int64_t total_elems;     /* elements per output arena (sum of round_up(count*width, 16)) */
    int64_t samples_emitted; /* S_emit of this call */
    int64_t samples_left;    /* un-emitted samples (non-join) */
    int64_t real_tokens;     /* sum of lengths of emitted samples */
    int64_t padded_elems;    /* sum of count*width */
} odb_plan_info;

typedef struct { /* device outputs, caller-allocated; any table pointer may be NULL (not wanted) */
    int32_t *d_input_ids;
    int32_t *d_labels;
    int32_t *d_position_ids;
    uint8_t *d_attention_mask;
    int64_t arena_capacity; /* elements available in each of the four arenas */
    /* per-slot tables, n_slots entries each (d_grp_sample_ptr: n_slots+1) */
    int32_t *d_grp_count;
    int32_t *d_grp_width;
    int32_t *d_grp_round;
    int32_t *d_grp_valid_tokens; /* #{labels != ignore_index} in the slot (Eq. 2's t_{r,k}) */
    int32_t *d_grp_real_tokens;  /* sum of the slot's sample lengths */
    int32_t *d_grp_origin;       /* step index of the first slot of the same rank cut from the same pre-alignment
                                    candidate group (== own step unless the slot is a split singleton; App. B) */
    int64_t *d_grp_offset;
    int64_t *d_grp_sample_ptr;
    int64_t slot_capacity_alloc; /* slots available in the per-slot tables */
    int32_t *d_grp_sample_ids;   /* local sample ids, row order, samples_emitted entries */
    int64_t ids_capacity;
    /* per-step tables, n_steps entries */
    int32_t *d_step_samples;      /* e_k = sum over ranks of count */
    int64_t *d_step_valid_tokens; /* T_tok,k = sum over ranks of valid tokens (Eq. 2) */
    int64_t step_capacity_alloc;
    /* un-emitted local ids per rank, ascending (non-join): d_left_ptr R+1, d_left_ids samples_left */
    int64_t *d_left_ptr;
    int32_t *d_left_ids;
    int64_t left_capacity;
} odb_outputs;

/* Create a context on CUDA device `device` for at most max_samples_total samples over all ranks.
 * Validates params (ODB_ERR_INVALID_ARG).  Allocates scratch (~70 bytes per sample). */
ODB_API int odb_create(const odb_params *params, int device, int64_t max_samples_total, odb_ctx **out);
ODB_API int odb_destroy(odb_ctx *ctx);
/* Forget all rounds and start over with the same params; keeps scratch. */
ODB_API int odb_reset(odb_ctx *ctx);

/* One protocol round, first half (section 2.2): fill each rank's window (recirculated leftovers +
 * the next un-fetched samples, up to buffer_size), sort it by (length, id), compute the greedy
 * successor of every start position and extract the candidate groups and G_r.  Lengths only; no
 * token is touched.  The first call after create/reset fixes d_lengths / h_rank_ptr (R+1 entries,
 * h_rank_ptr[R] <= max_samples_total) for the following rounds.  Asynchronous. */
ODB_API int odb_form_groups(odb_ctx *ctx, const int32_t *d_lengths, const int64_t *h_rank_ptr, void *stream);

/* Arrival state of the streams (the asynchronous side of App. C.1: a sampler view sits in the
 * worker queue until the workers deliver it).  h_arrived[r] = how many views of rank r's stream (in
 * sampler order) have arrived so far; only those can be drained into the window by the next
 * odb_form_groups.  A rank whose window is empty while views are pending advertises n_groups = 0
 * ("insufficient data"): it is not finished and gets IDLE slots; a round in which no rank has a
 * group is a skip round (T_grp = 0, nothing emitted; Lemma 2) -- the caller must let arrivals
 * progress, or the loop never terminates.  NULL = everything has arrived (the default after create /
 * reset, and what odb_run uses).  Values must not decrease.  Call between rounds only (before the first
 * odb_form_groups or after odb_round_status; ODB_ERR_STATE otherwise).  h_arrived: host, n_ranks entries. */
ODB_API int odb_set_available(odb_ctx *ctx, const int64_t *h_arrived, void *stream);

/* Online operation, the caller's side of the loop (App. C.1).  h_emitted[r] (host, n_ranks entries) = how
 * many views of rank r's stream have been emitted so far: the size of E_r in the paper's per-rank state machine
 * (a view that overflowed or was cut by the quota is back in the window and does not count).  Between rounds only:
 * after odb_reset (all 0), after odb_round_status, after termination; ODB_ERR_STATE inside a round and for offline
 * plans.  Waits for one small device-to-host copy on the stream the rounds were enqueued on. */
ODB_API int odb_emitted_counts(odb_ctx *ctx, int64_t *h_emitted);

/* The outstanding-depth envelope: the iterator schedules Fetch so that the views fetched but not yet
 * emitted, |Q_r + B_r|, stay within D = max(prefetch_factor * num_workers, buffer_size) -- the max is the clamp of
 * App. P: a loader configured with fewer outstanding views than one grouping buffer could never fill
 * it.  h_fetch_upto[r] = min(n_r, h_emitted[r] + D), n_r = h_rank_ptr[r+1] - h_rank_ptr[r]: how far into rank r's
 * stream the caller's workers may have fetched by now.  With buffer_size 0 (the window is the whole stream) the
 * envelope does not bind and h_fetch_upto[r] = n_r.  Lemma 2 is why skip rounds are finite under this
 * rule: D >= buffer_size >= 1 lets every unfinished rank fetch beyond what it has emitted.  Takes the job's
 * parameters (n_ranks, buffer_size), not a context: host arithmetic on host arrays of n_ranks (+ 1) entries, no device
 * work, usable on a machine without a GPU.  ODB_ERR_INVALID_ARG for negative arguments or h_emitted[r] outside
 * [0, n_r]. */
ODB_API int odb_fetch_quota(const odb_params *params, const int64_t *h_rank_ptr, int32_t prefetch_factor,
                            int32_t num_workers, const int64_t *h_emitted, int64_t *h_fetch_upto);

/* Second half (section 2.3, Alg. 1): T_grp by an on-device reduction over the R ranks, split /
 * overflow, IDLE slots, step totals, the non-join quota cut, leftovers.  Asynchronous. */
ODB_API int odb_align(odb_ctx *ctx, void *stream);

/* Synchronises.  *h_done != 0 when the protocol has terminated (no further round may be formed);
 * *h_T = T_grp of the round just aligned (0 if the round was the terminal check).  Must be called
 * after every odb_align.  Returns ODB_ERR_BAD_LENGTH if some length < 1. */
ODB_API int odb_round_status(odb_ctx *ctx, int32_t *h_done, int32_t *h_T);

/* Synchronises.  Builds the rank-major slot tables and block offsets; fills *h_out so the caller
 * can size the output arenas.  Only after termination (ODB_ERR_STATE otherwise). */
ODB_API int odb_plan_query(odb_ctx *ctx, odb_plan_info *h_out);

/* Collate every emitted slot (C.4 in DESIGN.md) and fill the tables of `out`.  Requires
 * odb_plan_query.  ODB_ERR_CAPACITY if an arena or table is too small.  Asynchronous. */
ODB_API int odb_collate(odb_ctx *ctx, const int32_t *d_tokens, const int64_t *d_sample_ptr, const int64_t *d_span_ptr,
                const int32_t *d_span_lo, const int32_t *d_span_hi, const odb_outputs *out, void *stream);

/* The whole plan without collation: reset, every protocol round until termination (on the device where odb_run
 * would run them there: the round-parallel planner and the persistent round loop for grouping buffers of at most
 * 4096 samples; host-driven rounds otherwise), the slot scan.  Synchronises for the plan sizes (*h_out);
 * afterwards the context is where odb_plan_query leaves it: odb_collate and odb_collate_steps may follow, and
 * odb_loss_weights once a full odb_collate has counted the valid tokens (not after odb_collate_steps alone). */
ODB_API int odb_plan(odb_ctx *ctx, const int32_t *d_lengths, const int64_t *h_rank_ptr, odb_plan_info *h_out, void *stream);

/* Streaming output (section 2.3: a round's aligned groups go to the trainer while the next window is being
 * grouped): collate the steps [step_lo, step_hi) of the plan SO FAR as a self-contained plan into `out` -- slots
 * s' = r * n + (k - step_lo), n = step_hi - step_lo, block offsets from 0 (the exclusive scan of
 * round_up(count * width, 16) over s'), every table of `out` indexed by s' (d_grp_origin keeps plan-wide step
 * indices, d_grp_round plan-wide rounds, d_grp_sample_ids rank-local ids, d_step_samples / d_step_valid_tokens the
 * n steps of the range; no leftover tables).  Allowed between rounds of the staged calls (after odb_round_status:
 * the steps emitted so far) and after termination (odb_plan / odb_plan_query / odb_run); the context's state and the
 * full plan's tables are untouched, so a trainer can pull a long plan through output buffers of bounded size, or
 * take every round's batches as soon as the round is committed.  *h_out describes the range (n_steps = n, n_slots,
 * total_elems, samples_emitted, real_tokens, padded_elems; n_rounds / stop_reason of the plan so far).  Waits only
 * for those sizes; the collate kernel is then running on `stream`.  The library keeps TWO sets of range tables and
 * alternates between them, so two ranges can be in flight at once (double buffering: a call reuses the tables of
 * the call before the previous one and must be ordered behind it -- same stream, or that call's work complete).
 * After odb_plan / odb_run each set is sized for the whole plan on its first use, so later ranges (a longer chunk, a
 * larger arena) allocate nothing; between rounds of the staged calls a range larger than any before it grows the set
 * (cudaFree + cudaMalloc: a device-wide synchronisation).
 * Null arenas: a sizing call (ODB_ERR_CAPACITY with *h_out filled unless the range is empty); it does not count in
 * the alternation -- the call that follows it uses the same set and should use the same stream.
 * The range's grp_valid_tokens / step_valid_tokens go to `out` only: the loss-scaling calls (odb_loss_weights,
 * odb_loss_numerators, odb_loss_normalize) need one full odb_collate of the plan and return ODB_ERR_STATE after
 * step-range collation alone.  ODB_ERR_CAPACITY
 * (nothing written) if an arena or table of `out` is too small; ODB_ERR_STATE for offline plans and distributed
 * mode. */
ODB_API int odb_collate_steps(odb_ctx *ctx, int32_t step_lo, int32_t step_hi, const int32_t *d_tokens,
                              const int64_t *d_sample_ptr, const int64_t *d_span_ptr, const int32_t *d_span_lo,
                              const int32_t *d_span_hi, const odb_outputs *out, odb_plan_info *h_out, void *stream);

/* Everything: reset, the round loop until termination, plan query, one collate over all emitted
 * steps.  With the four arenas given, the rounds run on the device and the slot scan, the collate preparation and
 * the collate kernel are enqueued behind them without a host round trip -- grouping buffers of at most 4096 samples
 * (the paper's regime): the round-parallel planner + the persistent round loop (ODB_OPT_ROUND_PARALLEL);
 * whole-stream windows: one round closed on the device -- and the call waits only for the plan sizes; otherwise
 * (a sizing call with NULL arenas, windows in between, too many ranks for a cooperative launch) the host drives the
 * rounds and synchronises once per round (a few bytes of status).  Returns with the collate kernels enqueued on
 * `stream`.  On ODB_ERR_CAPACITY *h_out is still filled. */
ODB_API int odb_run(odb_ctx *ctx, const int32_t *d_lengths, const int64_t *h_rank_ptr, const int32_t *d_tokens,
            const int64_t *d_sample_ptr, const int64_t *d_span_ptr, const int32_t *d_span_lo,
            const int32_t *d_span_hi, const odb_outputs *out, odb_plan_info *h_out, void *stream);

/* End-to-end variant with HOST buffers (pinned memory recommended): copies lengths, sample_ptr,
 * spans and tokens host->device, runs the whole path, copies the four arenas and every non-NULL
 * table of `h_out_bufs` (same struct, HOST pointers) back.  The device memory it uses does not grow
 * with the job: tokens pass through a ring of three rank-sized buffers, the arenas through a ring of
 * three fixed-size pieces (ODB_OPT_HOST_STAGING_ELEMS), uploads, collate launches and downloads overlapping
 * on three streams.  Synchronises before returning.  n_spans = h_span_ptr[N]. */
ODB_API int odb_run_host(odb_ctx *ctx, const int32_t *h_lengths, const int64_t *h_rank_ptr, const int32_t *h_tokens,
                 const int64_t *h_sample_ptr, const int64_t *h_span_ptr, const int32_t *h_span_lo,
                 const int32_t *h_span_hi, const odb_outputs *h_out_bufs, odb_plan_info *h_out, void *stream);

/* Loss-scaling weights (section 2.3 "Loss scaling", Eq. 2; modes P:738): d_weights[r * n_steps + k]
 * = w_{r,k} in fp64, one per slot; rank r prescales its mean loss of step k by W * w_{r,k} so that DDP's
 * average equals the per-token reference loss (Eq. 2).  Every quotient, product and sum is one IEEE fp64
 * operation, sums over ranks run in the order r = 0..R-1, a step whose denominator is 0 gets weight 0:
 * results are bit-identical to the CPU oracle.  Requires a completed odb_collate / odb_run on this
 * context (valid-token counts; ODB_ERR_STATE otherwise).  d_weights: device, n_slots doubles, caller-owned.
 * Asynchronous on `stream`. */
ODB_API int odb_loss_weights(odb_ctx *ctx, int mode, double *d_weights, void *stream);

/* The two halves of odb_loss_weights, for a job whose ranks live in several processes: numerators of
 * the local slots (d_num: n_slots doubles); after the caller has gathered the numerators of all ranks
 * into d_num_world (rank-major [world_ranks][n_steps]; rows [rank_offset, rank_offset + n_ranks) are this
 * context's), odb_loss_normalize sums each step's column in the order r = 0..world_ranks-1 and writes the
 * local weights (d_weights may alias the local rows of d_num_world). */
ODB_API int odb_loss_numerators(odb_ctx *ctx, int mode, double *d_num, void *stream);
ODB_API int odb_loss_normalize(odb_ctx *ctx, const double *d_num_world, int32_t world_ranks, int32_t rank_offset,
                               double *d_weights, void *stream);

/* ---- ranks spread over several processes / GPUs -------------------------------
 * The paper runs one rank per process and exchanges, once per round, every rank's status and group
 * counts with ONE unconditional all_gather (section 2.3; message layout P:250; deadlock-freedom
 * Lemma 3), then evaluates Eq. 3 and the termination predicates on that shared tensor.  Here a
 * context holds n_ranks consecutive ranks of a job of world_ranks ranks (equal n_ranks in every
 * process); the library never communicates: it exposes the device buffers, the CALLER runs the
 * collectives (torch.distributed over NCCL / NVLink) between the calls:
 *
 *   odb_dist_config(ctx, world_ranks, rank_offset, world_max_window)      once per run (resets the ctx)
 *   per round:
 *     odb_form_groups(...)         local windows, groups; packs (G_r, S_r) pairs into d_summary_local
 *     all_gather(d_summary_world <- d_summary_local)                       [collective 1, 8 bytes per rank]
 *     odb_align(...)               Eq. 3 and the termination predicates from d_summary_world; split / overflow
 *     all_reduce(SUM, d_step_samples_round[0 .. step_window))              [collective 2, global e_k, P:347]
 *     odb_commit(...)              quota cut on the global totals, staging tables, leftovers
 *     odb_round_status(...)        identical on every process
 *   odb_plan_query / odb_collate   local slots only
 *   all_reduce(SUM, the caller's out->d_step_valid_tokens[0 .. n_steps))   [Eq. 2's T_tok per step]
 *
 * world_max_window = max over ALL ranks of the job of min(n_r, buffer_size or n_r): bounds T_grp of a
 * round (a process whose ranks are all finished still emits T IDLE slots).  odb_plan_info then counts
 * the local ranks only, except n_rounds / n_steps / stop_reason, which are global.  In this mode
 * odb_run / odb_run_host return ODB_ERR_STATE. */
typedef struct {
    int32_t *d_summary_local;      /* 2 * n_ranks int32: (G_r, S_r) per local rank */
    int32_t *d_summary_world;      /* 2 * world_ranks int32 */
    int32_t summary_local_count, summary_world_count;
    int32_t *d_step_samples_round; /* valid between odb_form_groups and odb_commit of a round */
    int32_t step_window;
    int32_t spec_G_count;          /* batched exchange: n_rounds * n_ranks */
    int32_t *d_spec_G_local;       /* batched exchange: G of the local ranks, [round][rank] (after odb_dist_spec_form) */
} odb_dist_bufs;
ODB_API int odb_dist_config(odb_ctx *ctx, int32_t world_ranks, int32_t rank_offset, int32_t world_max_window);
ODB_API int odb_dist_buffers(odb_ctx *ctx, odb_dist_bufs *out);
/* Distributed mode only (ODB_ERR_STATE otherwise): second half of odb_align, after collective 2. */
ODB_API int odb_commit(odb_ctx *ctx, void *stream);

/* Distributed mode, BATCHED EXCHANGE: the round-parallel planner (ODB_OPT_ROUND_PARALLEL) over several processes.
 * A round depends on its predecessors only through the leftovers, and there are none until a round
 * overflows; until then the window of round j of rank r is the views [j B, (j + 1) B) of its stream, so the
 * per-round exchange of P:52 can be done for ALL those rounds at once: 3 collectives for J rounds instead of 2 J.
 *
 *   all_gather(every rank's stream length n_r)                             [the caller; once per run]
 *   odb_dist_spec_form(ctx, d_lengths, h_rank_ptr, J, max n_r, stream)     local windows of the rounds [0, J): sort,
 *                                                                          candidate groups, G table (odb_dist_buffers:
 *                                                                          d_spec_G_local, spec_G_count, [round][rank])
 *   all_gather(G_world <- d_spec_G_local)                                  [layout [process][round][local rank]]
 *   odb_dist_spec_commit(ctx, G_world, n_world, n_procs, stream)           Eq. 3 and the no-overflow check of every round
 *                                                                          on the gathered data (identical everywhere,
 *                                                                          Lemma 3), split + commit of the rounds before
 *                                                                          the first that overflows
 *   all_reduce(SUM, d_step_samples_round[0 .. max n_r))                    [global e_k of those rounds' steps]
 *   odb_dist_spec_status(ctx, &rounds, &steps, h_T, capacity, &done)       synchronises; rounds committed (0 .. J), their
 *                                                                          steps and T_grp.  done = 1: all J were, round J
 *                                                                          is the terminal check -- known to every process
 *                                                                          from the same data, so it needs no exchange:
 *                                                                          the protocol is over (odb_plan_query next);
 *                                                                          done = 0: the per-round calls go on with round
 *                                                                          `rounds` (odb_form_groups ...)
 *
 * J = rounds that are certainly not the terminal check: join ceil(max n_r / B), non-join ceil(min n_r / B), over ALL
 * ranks of the job (1 .. 65535).  Requirements (ODB_ERR_INVALID_ARG / ODB_ERR_STATE otherwise): distributed mode,
 * a fresh run (after odb_dist_config / odb_reset), buffer_size in 8 .. 4096, no sample quota, no arrival schedule,
 * every process holds the same number of ranks (world_ranks = n_procs * n_ranks). */
ODB_API int odb_dist_spec_form(odb_ctx *ctx, const int32_t *d_lengths, const int64_t *h_rank_ptr, int32_t n_rounds,
                               int64_t world_max_stream, void *stream);
ODB_API int odb_dist_spec_commit(odb_ctx *ctx, const int32_t *d_G_world, const int32_t *d_n_world, int32_t n_procs,
                                 void *stream);
ODB_API int odb_dist_spec_status(odb_ctx *ctx, int32_t *h_rounds, int32_t *h_steps, int32_t *h_T, int32_t T_capacity,
                                 int32_t *h_done);

/* Device times of the last odb_run / odb_collate on this context, in milliseconds, measured with
 * CUDA events on the launching stream: ms[0] = planning (all rounds, plan query, row descriptors and
 * the tile table), ms[1] = the collate kernel alone, ms[2] = what follows it (step totals, table
 * copies).  Synchronises.  Enabled by odb_set_timing(ctx, 1); off by default. */
ODB_API int odb_set_timing(odb_ctx *ctx, int enable);
ODB_API int odb_get_timing(odb_ctx *ctx, float *ms3);
/* The same for the timed run `back` runs before the latest one (0 = the latest, up to 63): the events of
 * the last 64 runs are kept, so a benchmark can enqueue many runs back to back and read their stage times
 * afterwards instead of waiting on every run.  ODB_ERR_STATE if that run does not exist (any more). */
ODB_API int odb_get_timing_at(odb_ctx *ctx, int back, float *ms3);
/* ---- the paper's offline comparators as planners ---------------------------------
 * GMT and BMT (App. I) and HFG (App. J) build their batches from a GLOBAL scalar length array (the
 * paper's "oracle cache"), not from per-rank streams; every rank computes the same list and takes its share by
 * striding.  odb_offline_plan plans such a job for the context's n_ranks = W ranks and budget (padded-area
 * feasibility max_i l_i * |b| <= budget, over-budget singletons allowed); afterwards odb_plan_query /
 * odb_collate / odb_loss_weights work as for an ODB plan, with these differences: a slot's ids
 * (d_grp_sample_ids) are GLOBAL sample ids; d_sample_ptr / d_span_ptr of odb_collate are indexed by global
 * sample id; a sample may sit in two slots (wrap-around repetition); there are no leftovers; n_rounds = 1.
 *   GMT: ascending (length, id) sort of all samples, greedy packing; the batch list is padded to a multiple of W
 *        by repeating its leading batches (at most W - 1) and batch j goes to rank j mod W, step j div W.
 *   BMT: the shuffled order d_perm is cut into buckets of `size` samples, each bucket is sorted by (length,
 *        position in the shuffled order) and packed on its own, the batches are then ordered by (d_shuffle_key[j],
 *        j), j = the batch's index before the shuffle; padding and striding as GMT.
 *   HFG: d_perm is cut into megabatches of `size` samples, each sorted by length DESCENDING (the reverse of the
 *        ascending (length, position) order), concatenated, padded to a multiple of W with its leading entries;
 *        rank r takes every W-th index from r, and steps are runs of `batch_size` consecutive entries.
 * The random draws are inputs: d_perm = a permutation of 0 .. n_samples - 1, d_shuffle_key = n_samples keys in
 * [0, 2^31) (device pointers, caller-owned, must stay valid until odb_collate).  Synchronises (an offline
 * planner: the host sizes the batch tables).  ODB_ERR_BAD_LENGTH if some length < 1. */
enum { ODB_PLANNER_GMT = 0, ODB_PLANNER_BMT = 1, ODB_PLANNER_HFG = 2 };
typedef struct {
    int32_t planner;    /* ODB_PLANNER_* */
    int32_t size;       /* BMT: samples per bucket; HFG: samples per megabatch */
    int32_t batch_size; /* HFG: the fixed batch size */
    int32_t reserved;
    const int32_t *d_perm;        /* BMT, HFG */
    const int32_t *d_shuffle_key; /* BMT */
} odb_offline_params;
ODB_API int odb_offline_plan(odb_ctx *ctx, const odb_offline_params *params, const int32_t *d_lengths, int64_t n_samples,
                             void *stream);

/* ---- for callers that cannot allocate device memory ------------------------------------------------
 * Some users of this library are guests on a GPU they do not manage: a data-loading plugin inside a trainer whose
 * framework has already claimed the whole HBM for its caching allocator (a second party's cudaMalloc then fails, or
 * works and makes the trainer run out of memory later), or code running in the middle of a training step, where
 * cudaMalloc / cudaFree hold up every stream of the device.  They cannot call odb_create (the context allocates
 * ~70 bytes per sample).  odb_slot_offsets_static is the one entry point made for them: it takes no context, calls no
 * cudaMalloc / cudaFree and no library routine that allocates, and keeps the scan's tile records in a fixed
 * 128.25 KiB array that is part of the library image (every GPU that loads libodb.so holds it until the process ends).
 *
 * It computes the output offsets of a plan (A9; a group's padded block is count x width), as
 * odb_plan_query / odb_run do for out->d_grp_offset:
 *     d_grp_offset[s] = sum over s' < s of round_up(d_grp_count[s'] * d_grp_width[s'], 16),   s = 0 .. n_slots,
 * so d_grp_offset[n_slots] is odb_plan_info.total_elems.  d_grp_count, d_grp_width: device, n_slots int32 each,
 * caller-owned, read only; d_grp_offset: device, n_slots + 1 int64, caller-owned, written.  n_slots = 0 is allowed
 * (writes d_grp_offset[0] = 0).  Asynchronous on `stream`, on the device that is current when it is called.
 *
 * Limit: n_slots <= ODB_STATIC_MAX_SLOTS (odb_static_max_slots() returns it).  More slots than that: ODB_ERR_CAPACITY,
 * nothing launched, nothing written -- the fixed array has no tile records for them.  Bad pointers or n_slots < 0:
 * ODB_ERR_INVALID_ARG.  A failing CUDA call: ODB_ERR_CUDA, with the cudaError_t in odb_static_last_cuda_error()
 * (per host thread).
 *
 * First call on each device: it asks the CUDA runtime for the array's address on that device (a one-time set-up,
 * kept for later calls).  Make that first call before you start capturing a stream.
 * Sharing: all calls on a device use the same array, and each call starts by clearing the part it needs (two small
 * kernels per call: the clear, then the scan).  Two calls whose kernels may run at the same time on one device --
 * different streams with no ordering between them, or two host threads -- corrupt each other's result: put them on
 * one stream or order them with events. */
#define ODB_STATIC_MAX_SLOTS 4194304 /* 2^22 slots (the largest BASELINE.json config has ~2 * 10^5) */
ODB_API int odb_slot_offsets_static(const int32_t *d_grp_count, const int32_t *d_grp_width, int64_t n_slots,
                                    int64_t *d_grp_offset, void *stream);
ODB_API int64_t odb_static_max_slots(void);
ODB_API int odb_static_last_cuda_error(void);

/* Tuning / measurement switches.  ODB_OPT_COLLATE_BULK_STORES (value 0 / 1, default 0): the collate kernel stages
 * the interior chunks of each arena in shared memory and stores them with bulk asynchronous copies
 * (cp.async.bulk.global.shared::cta, the store side of BASELINE.json's "TMA bulk copies") instead of 256-bit
 * streaming stores from registers.  Same results bit for bit; the measured comparison is in profiles/.
 * ODB_OPT_HOST_STAGING_ELEMS (value >= 1, default 2^25): arena elements per device staging piece of odb_run_host
 * (three pieces of 13 bytes per element are held; rounded down to a multiple of 4096, at least 4096).
 * ODB_OPT_ROUND_PARALLEL (value 0 / 1, default 1): with a grouping buffer of 8 .. 4096 samples (the paper's
 * operating point) odb_run forms and commits the protocol rounds round-parallel -- a round depends on its
 * predecessors only through the leftovers, and there are none until a round overflows -- and the
 * sequential round loop resumes at the first round that does (with a sample quota: at the latest at the round whose
 * cumulative emission reaches it); 0 = every round in the sequential loop.  Same results bit for bit.
 * ODB_OPT_HOST_DEVICE_ARENAS (value 0 / 1, default 0): the four arena pointers of odb_run_host's `h_out_bufs` are
 * DEVICE memory (16-byte aligned, arena_capacity elements): the inputs still come from host buffers rank by rank,
 * but every rank's slots are collated in place as soon as its tokens have landed and the batches stay on the device
 * for the trainer; only the tables (still HOST pointers) come back.  No output staging is allocated.
 * ODB_ERR_INVALID_ARG for an unknown option. */
enum { ODB_OPT_COLLATE_BULK_STORES = 1, ODB_OPT_HOST_STAGING_ELEMS = 2, ODB_OPT_ROUND_PARALLEL = 3,
       ODB_OPT_HOST_DEVICE_ARENAS = 4 };
ODB_API int odb_set_option(odb_ctx *ctx, int option, int64_t value);

/* Bandwidth probes (measurement utility, not part of the method): the collate kernel's byte mix -- 4 bytes read
 * and 13 written per element -- with trivial indexing.  kind 0: the mix with 256-bit streaming stores; 1: the mix
 * with bulk stores from shared memory; 2 / 3: the 13 bytes of stores alone in the two forms; 4: a copy (4 bytes
 * read, 4 written).  d_in: n_elems int32 (kinds 0, 1, 4); d_out0..2: n_elems int32, d_out3: n_elems bytes (kind 4
 * writes d_out0 only); all 16-byte aligned; n_elems is rounded down to a multiple of 512.  Runs 1 + reps launches
 * on `stream` and writes the average milliseconds per launch to *h_ms.  Synchronises. */
ODB_API int odb_probe_bandwidth(int kind, const int32_t *d_in, int32_t *d_out0, int32_t *d_out1, int32_t *d_out2,
                                uint8_t *d_out3, int64_t n_elems, int reps, void *stream, float *h_ms);

/* Number of kernels this context has launched since odb_create (diagnostics / bench accounting). */
ODB_API int64_t odb_kernel_launches(const odb_ctx *ctx);

/* Diagnostics: copy an internal device table to the host (synchronises).  `what`: 0 = G_r (int32[R])
 * of the last round, 1 = S_r (int32[R]), 2 = sorted keys of the last round ((len<<32)|id, uint64[N],
 * rank regions at h_rank_ptr), 3 = views emitted so far per rank (int32[R]; valid between rounds of the staged calls),
 * 4 = the record of the round-parallel planner of the last odb_run (int32[4]: rounds it committed, steps they emit,
 * 1 if it ended the protocol, 0; < 0 is returned when that run did not use it),
 * 5 = how many times the library's growable device tables have called cudaMalloc in this process so far (int64; a
 * host-side counter, no synchronisation).
 * Returns bytes copied or < 0. */
ODB_API int64_t odb_debug_read(odb_ctx *ctx, int what, void *h_dst, int64_t max_bytes);

/* Synthetic-input utility (benchmarks / tests; not part of the method): d_tokens[j] for j in
 * [0, count) = the counter-based id of global token index start + j,
 *   ((mix64(seed * 0x9E3779B97F4A7C15 + start + j) >> 32) * vocab) >> 32,  mix64 = SplitMix64 finaliser
 * (DESIGN.md "Input recipe").  Asynchronous on `stream`. */
ODB_API int odb_synth_tokens(int32_t *d_tokens, int64_t start, int64_t count, uint64_t seed, int32_t vocab, void *stream);

ODB_API int odb_last_cuda_error(const odb_ctx *ctx);
ODB_API const char *odb_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* ODB_H_ */
