// C ABI of libodb (include/odb.h): argument checks, the host-side round loop / state machine,
// scratch management.  Every step of the path runs in the kernels of odb_plan.cu / odb_collate.cu;
// there is no CPU fallback.
#include <algorithm>
#include <cstddef>
#include <cstring>
#include <new>

#include "odb_internal.cuh"

using namespace odb;

#define CU(c, expr)                                 \
    do {                                            \
        cudaError_t e__ = (expr);                   \
        if (e__ != cudaSuccess) {                   \
            (c)->last_cuda_error = (int)e__;        \
            (void)cudaGetLastError();               \
            return ODB_ERR_CUDA;                    \
        }                                           \
    } while (0)

template <class T>
static cudaError_t dev_alloc(T **p, size_t n) {
    return cudaMalloc((void **)p, std::max<size_t>(n, 1) * sizeof(T));
}

// grow a step-major staging table, preserving `used` entries and zero-filling the rest
template <class T>
static cudaError_t grow_preserve(DevBuf<T> &b, size_t want, size_t used, cudaStream_t st) {
    if (want <= b.cap) return cudaSuccess;
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    T *np = nullptr;
    e = cudaMalloc((void **)&np, want * sizeof(T));
    if (e != cudaSuccess) return e;
    e = cudaMemset(np, 0, want * sizeof(T));
    if (e != cudaSuccess) return e;
    if (b.p && used) {
        e = cudaMemcpy(np, b.p, used * sizeof(T), cudaMemcpyDeviceToDevice);
        if (e != cudaSuccess) return e;
    }
    if (b.p) cudaFree(b.p);
    b.p = np;
    b.cap = want;
    return cudaSuccess;
}

template <class T>
static cudaError_t copy_tab(T *dst, const T *src, size_t n, cudaStream_t st) {
    if (!dst || n == 0) return cudaSuccess;
    return cudaMemcpyAsync(dst, src, n * sizeof(T), cudaMemcpyDeviceToDevice, st);
}

static void free_all(odb_ctx *c) {
    cudaFree(c->d_rank_ptr);
    cudaFree(c->keyA);
    cudaFree(c->keyB);
    cudaFree(c->ovf);
    cudaFree(c->jA);
    cudaFree(c->jB);
    cudaFree(c->mark);
    cudaFree(c->posflag);
    cudaFree(c->emit_pos);
    cudaFree(c->gpos);
    cudaFree(c->agpos);
    cudaFree(c->agcnt);
    cudaFree(c->agoff);
    cudaFree(c->agorg);
    cudaFree(c->left_ids);
    cudaFree(c->emit_ids);
    cudaFree(c->n_left);
    cudaFree(c->fetch_pos);
    cudaFree(c->emit_cur);
    cudaFree(c->G);
    cudaFree(c->S);
    cudaFree(c->emit_snap);
    cudaFree(c->d_arrived);
    cudaFree(c->d_rec);
    cudaFree(c->d_dims);
    cudaFree(c->d_done_ctr);
    cudaFree(c->d_tile_counter);
    cudaFree(c->gs_local);
    cudaFree(c->gs_world);
    cudaFree(c->gs_rounds);
    if (c->h_rec) cudaFreeHost(c->h_rec);
    if (c->h_dims) cudaFreeHost(c->h_dims);
    if (c->h_dims_up) cudaFreeHost(c->h_dims_up);
    if (c->ev_plan) cudaEventDestroy(c->ev_plan);
    c->st_count.release();
    c->st_width.release();
    c->st_real.release();
    c->st_round.release();
    c->st_origin.release();
    c->step_samples.release();
    c->grp_count.release();
    c->grp_width.release();
    c->grp_round.release();
    c->grp_valid.release();
    c->grp_real.release();
    c->grp_origin.release();
    c->scan_state.release();
    c->grp_offset.release();
    c->grp_sample_ptr.release();
    c->grp_sample_ids.release();
    c->left_out.release();
    c->left_ptr.release();
    c->step_valid.release();
    c->rows.release();
    c->row_sp.release();
    c->tiles.release();
    c->hs_lengths.release();
    c->hs_tokens.release();
    c->hs_span_lo.release();
    c->hs_span_hi.release();
    c->hs_ids.release();
    c->hs_labels.release();
    c->hs_pos.release();
    c->hs_sample_ptr.release();
    c->hs_span_ptr.release();
    c->hs_mask.release();
    for (cudaEvent_t e : c->evring) cudaEventDestroy(e);
    if (c->ev_status) cudaEventDestroy(c->ev_status);
    if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
    if (c->copy_ev) cudaEventDestroy(c->copy_ev);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    c->piece_ctr.release();
    c->spec_tab.release();
    if (c->h_rank_off) cudaFreeHost(c->h_rank_off);
    if (c->h_spec) cudaFreeHost(c->h_spec);
    for (SubTabs &t : c->sub) {
        t.grp_count.release();
        t.grp_width.release();
        t.grp_round.release();
        t.grp_valid.release();
        t.grp_real.release();
        t.grp_origin.release();
        t.scan_state.release();
        t.grp_offset.release();
        t.grp_sample_ptr.release();
        t.grp_sample_ids.release();
        t.left_out.release();
        t.left_ptr.release();
        t.step_valid.release();
        t.rows.release();
        t.row_sp.release();
        t.tiles.release();
        cudaFree(t.d_dims);
        cudaFree(t.d_tile_counter);
        if (t.h_dims) cudaFreeHost(t.h_dims);
        if (t.ev_plan) cudaEventDestroy(t.ev_plan);
    }
}

// the context's plan tables <-> a step-range set (odb_collate_steps): kernels take the pointers at launch, so the
// full plan's tables are back as soon as the range has been enqueued
static void swap_tabs(odb_ctx *c, SubTabs &t) {
    std::swap(c->grp_count, t.grp_count);
    std::swap(c->grp_width, t.grp_width);
    std::swap(c->grp_round, t.grp_round);
    std::swap(c->grp_valid, t.grp_valid);
    std::swap(c->grp_real, t.grp_real);
    std::swap(c->grp_origin, t.grp_origin);
    std::swap(c->scan_state, t.scan_state);
    std::swap(c->grp_offset, t.grp_offset);
    std::swap(c->grp_sample_ptr, t.grp_sample_ptr);
    std::swap(c->grp_sample_ids, t.grp_sample_ids);
    std::swap(c->left_out, t.left_out);
    std::swap(c->left_ptr, t.left_ptr);
    std::swap(c->step_valid, t.step_valid);
    std::swap(c->rows, t.rows);
    std::swap(c->row_sp, t.row_sp);
    std::swap(c->tiles, t.tiles);
    std::swap(c->d_dims, t.d_dims);
    std::swap(c->h_dims, t.h_dims);
    std::swap(c->d_tile_counter, t.d_tile_counter);
    std::swap(c->ev_plan, t.ev_plan);
}

extern "C" {

const char *odb_status_string(int status) {
    switch (status) {
    case ODB_OK: return "ok";
    case ODB_ERR_INVALID_ARG: return "invalid argument";
    case ODB_ERR_BAD_LENGTH: return "bad length (some sample length < 1)";
    case ODB_ERR_CAPACITY: return "output capacity too small";
    case ODB_ERR_CUDA: return "CUDA error";
    case ODB_ERR_STATE: return "call order violated";
    default: return "unknown status";
    }
}

int odb_last_cuda_error(const odb_ctx *ctx) { return ctx ? ctx->last_cuda_error : 0; }
int64_t odb_kernel_launches(const odb_ctx *ctx) { return ctx ? ctx->launches : 0; }

int odb_create(const odb_params *p, int device, int64_t max_samples_total, odb_ctx **out) {
    if (!p || !out) return ODB_ERR_INVALID_ARG;
    *out = nullptr;
    if (p->n_ranks < 1 || p->n_ranks > 65535 || p->budget < 1 || p->budget > 0x7fffffffll ||
        (p->rule != ODB_RULE_THRESHOLD && p->rule != ODB_RULE_MAXFIT_ASC) || p->buffer_size < 0 || p->slot_capacity < 0 ||
        max_samples_total < 0 || max_samples_total > 0x7fffff00ll || (p->join_mode != 0 && p->join_mode != 1) ||
        (p->shift_labels != 0 && p->shift_labels != 1))
        return ODB_ERR_INVALID_ARG;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) {
        (void)cudaGetLastError();
        return ODB_ERR_CUDA;  // no CPU fallback
    }
    odb_ctx *c = new (std::nothrow) odb_ctx();
    if (!c) return ODB_ERR_CUDA;
    c->prm = *p;
    c->device = device;
    c->n_max = max_samples_total;
    memset(&c->info, 0, sizeof(c->info));
    cudaError_t e = cudaSetDevice(device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
    if (e == cudaSuccess) c->sm_count = prop.multiProcessorCount;
    const size_t N = (size_t)max_samples_total, R = (size_t)p->n_ranks;
    if (e == cudaSuccess) e = dev_alloc(&c->d_rank_ptr, R + 1);
    if (e == cudaSuccess) e = dev_alloc(&c->keyA, N);
    if (e == cudaSuccess) e = dev_alloc(&c->keyB, N);
    if (e == cudaSuccess) e = dev_alloc(&c->ovf, 2 * N + 2);
    if (e == cudaSuccess) e = dev_alloc(&c->jA, N + R);
    if (e == cudaSuccess) e = dev_alloc(&c->jB, N + R);
    if (e == cudaSuccess) e = dev_alloc(&c->mark, N + R);
    if (e == cudaSuccess) e = dev_alloc(&c->posflag, N);
    if (e == cudaSuccess) e = dev_alloc(&c->emit_pos, N);
    if (e == cudaSuccess) e = dev_alloc(&c->gpos, plan_table_entries(N, R));
    if (e == cudaSuccess) e = dev_alloc(&c->agpos, plan_table_entries(N, R));
    if (e == cudaSuccess) e = dev_alloc(&c->agcnt, plan_table_entries(N, R));
    if (e == cudaSuccess) e = dev_alloc(&c->agoff, plan_table_entries(N, R));
    if (e == cudaSuccess) e = dev_alloc(&c->agorg, plan_table_entries(N, R));
    if (e == cudaSuccess) e = dev_alloc(&c->left_ids, N);
    if (e == cudaSuccess) e = dev_alloc(&c->emit_ids, N);
    if (e == cudaSuccess) e = dev_alloc(&c->n_left, R);
    if (e == cudaSuccess) e = dev_alloc(&c->fetch_pos, R);
    if (e == cudaSuccess) e = dev_alloc(&c->emit_cur, R);
    if (e == cudaSuccess) e = dev_alloc(&c->G, R);
    if (e == cudaSuccess) e = dev_alloc(&c->S, R);
    if (e == cudaSuccess) e = dev_alloc(&c->emit_snap, R);
    if (e == cudaSuccess) e = dev_alloc(&c->d_arrived, R);
    if (e == cudaSuccess) e = dev_alloc(&c->d_rec, 1);
    if (e == cudaSuccess) e = dev_alloc(&c->d_dims, 1);
    if (e == cudaSuccess) e = cudaMemset(c->d_dims, 0, sizeof(PlanDims));
    if (e == cudaSuccess) e = dev_alloc(&c->d_done_ctr, 2);
    if (e == cudaSuccess) e = cudaMemset(c->d_done_ctr, 0, 2 * sizeof(unsigned int));
    if (e == cudaSuccess) e = dev_alloc(&c->d_tile_counter, R + 1);  // one work counter per pipelined launch
    if (e == cudaSuccess) e = cudaMallocHost((void **)&c->h_rec, sizeof(RoundRec));
    if (e == cudaSuccess) e = cudaMallocHost((void **)&c->h_dims, sizeof(PlanDims));
    if (e == cudaSuccess) e = cudaMallocHost((void **)&c->h_dims_up, sizeof(PlanDims));
    if (e == cudaSuccess) e = cudaMallocHost((void **)&c->h_rank_off, (R + 1) * sizeof(int64_t));
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_plan, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_status, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        free_all(c);
        delete c;
        return ODB_ERR_CUDA;
    }
    *out = c;
    return ODB_OK;
}

int odb_destroy(odb_ctx *c) {
    if (!c) return ODB_ERR_INVALID_ARG;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    free_all(c);
    delete c;
    return ODB_OK;
}

int odb_reset(odb_ctx *c) {
    if (!c) return ODB_ERR_INVALID_ARG;
    c->state = 0;
    c->round = 0;
    c->n_rounds = 0;
    c->n_steps = 0;
    c->samples_emitted = 0;
    c->n_finished = 0;
    c->last_T = 0;
    c->stop_reason = 0;
    c->info_valid = false;
    c->collated = false;
    c->arrived_set = false;
    c->begin_pending = false;
    c->offline = false;
    c->offline_perm = nullptr;
    c->d_lengths = nullptr;
    c->spec_used = false;
    return ODB_OK;
}

int odb_offline_plan(odb_ctx *c, const odb_offline_params *P, const int32_t *d_lengths, int64_t n_samples, void *stream) {
    if (!c || !P) return ODB_ERR_INVALID_ARG;
    if (c->world_ranks) return ODB_ERR_STATE;
    if (n_samples < 0 || n_samples > c->n_max || (n_samples > 0 && !d_lengths)) return ODB_ERR_INVALID_ARG;
    if (P->planner != ODB_PLANNER_GMT && P->planner != ODB_PLANNER_BMT && P->planner != ODB_PLANNER_HFG)
        return ODB_ERR_INVALID_ARG;
    if (P->planner != ODB_PLANNER_GMT && (P->size < 1 || (n_samples > 0 && !P->d_perm))) return ODB_ERR_INVALID_ARG;
    if (P->planner == ODB_PLANNER_BMT && n_samples > 0 && !P->d_shuffle_key) return ODB_ERR_INVALID_ARG;
    if (P->planner == ODB_PLANNER_HFG && P->batch_size < 1) return ODB_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    CU(c, cudaSetDevice(c->device));
    odb_reset(c);
    c->last_stream = st;
    c->offline = true;
    c->offline_planner = P->planner;
    c->offline_bs = P->batch_size;
    c->offline_perm = P->planner == ODB_PLANNER_GMT ? nullptr : P->d_perm;
    c->d_lengths = d_lengths;
    c->n_total = n_samples;
    c->max_nr = (int32_t)std::min<int64_t>(n_samples, 0x7fffffff);
    c->h_rank_ptr.assign((size_t)c->prm.n_ranks + 1, 0);
    c->dev_rank_ptr_valid = false;  // (the host copy no longer mirrors d_rank_ptr)
    CU(c, offline_build(c, P, d_lengths, n_samples, st));
    {  // bad lengths
        CU(c, cudaMemcpyAsync(c->h_rec, c->d_rec, sizeof(RoundRec), cudaMemcpyDeviceToHost, st));
        CU(c, cudaStreamSynchronize(st));
        if (c->h_rec->bad_length) {
            odb_reset(c);
            return ODB_ERR_BAD_LENGTH;
        }
    }
    const int64_t W = c->prm.n_ranks;
    int64_t n_steps;
    if (P->planner == ODB_PLANNER_HFG) {
        const int64_t n_per = (n_samples + W - 1) / W;
        n_steps = (n_per + P->batch_size - 1) / P->batch_size;
    } else {
        n_steps = (c->offline_G + W - 1) / W;
    }
    if (n_steps > 0x7fffffff / std::max<int64_t>(W, 1)) return ODB_ERR_INVALID_ARG;
    c->n_steps = (int32_t)n_steps;
    c->n_rounds = 1;
    c->round = 1;
    c->stop_reason = ODB_STOP_ALL_FINISHED;
    CU(c, offline_slots(c, st));
    c->state = 4;
    return ODB_OK;
}

int odb_set_option(odb_ctx *c, int option, int64_t value) {
    if (!c) return ODB_ERR_INVALID_ARG;
    switch (option) {
    case ODB_OPT_COLLATE_BULK_STORES: c->collate_bulk = value != 0; return ODB_OK;
    case ODB_OPT_ROUND_PARALLEL: c->round_parallel = value != 0; return ODB_OK;
    case ODB_OPT_HOST_DEVICE_ARENAS: c->host_device_arenas = value != 0; return ODB_OK;
    case ODB_OPT_HOST_STAGING_ELEMS:
        if (value < 1) return ODB_ERR_INVALID_ARG;
        c->host_staging_elems = value;
        return ODB_OK;
    default: return ODB_ERR_INVALID_ARG;
    }
}

int odb_set_timing(odb_ctx *c, int enable) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (enable && c->evring.empty()) {
        CU(c, cudaSetDevice(c->device));
        c->evring.assign((size_t)4 * kTimingRing, nullptr);
        for (cudaEvent_t &e : c->evring) CU(c, cudaEventCreate(&e));
    }
    c->timing = enable ? 1 : 0;
    c->ev_seq = 0;
    c->ev = c->evring.empty() ? nullptr : c->evring.data();
    c->ev_valid = false;
    return ODB_OK;
}

// the timed run `back` runs before the latest one (0 = the latest)
int odb_get_timing_at(odb_ctx *c, int back, float *ms3) {
    if (!c || !ms3 || back < 0) return ODB_ERR_INVALID_ARG;
    if (!c->timing || back >= kTimingRing || (int64_t)back >= c->ev_seq) return ODB_ERR_STATE;
    cudaEvent_t *ev = c->evring.data() + 4 * (size_t)((c->ev_seq - 1 - back) % kTimingRing);
    CU(c, cudaEventSynchronize(ev[3]));
    float plan = 0.f, col = 0.f, all = 0.f;
    CU(c, cudaEventElapsedTime(&plan, ev[0], ev[1]));
    CU(c, cudaEventElapsedTime(&col, ev[1], ev[2]));
    CU(c, cudaEventElapsedTime(&all, ev[2], ev[3]));
    ms3[0] = plan;
    ms3[1] = col;
    ms3[2] = all;
    return ODB_OK;
}

int odb_get_timing(odb_ctx *c, float *ms3) { return odb_get_timing_at(c, 0, ms3); }

// the quadruple a run that starts now records into; timing_done() closes it
static void timing_begin(odb_ctx *c) { c->ev = c->evring.data() + 4 * (size_t)(c->ev_seq % kTimingRing); }
static void timing_done(odb_ctx *c) {
    c->ev_seq++;
    c->ev_valid = true;
}

// first round after create / reset: bind inputs, clear the per-run device state
static int begin_run(odb_ctx *c, const int32_t *d_lengths, const int64_t *h_rank_ptr, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    if (!h_rank_ptr) return ODB_ERR_INVALID_ARG;
    if (h_rank_ptr[0] != 0) return ODB_ERR_INVALID_ARG;
    int64_t max_nr = 0;
    for (int r = 0; r < R; ++r) {
        int64_t n = h_rank_ptr[r + 1] - h_rank_ptr[r];
        if (n < 0) return ODB_ERR_INVALID_ARG;
        max_nr = std::max(max_nr, n);
    }
    if (h_rank_ptr[R] > c->n_max) return ODB_ERR_INVALID_ARG;
    if (h_rank_ptr[R] > 0 && !d_lengths) return ODB_ERR_INVALID_ARG;
    // the rank boundaries and the arrival counts go up only when they differ from what the device already holds
    // (a training job calls with the same partition step after step; every stream operation in front of the first
    // kernel costs a few microseconds of an otherwise 0.2 ms planning stage)
    if (c->dev_meta_stream != st) {  // (uploaded on another stream: no ordering with this one is assumed)
        c->dev_rank_ptr_valid = false;
        c->h_arrived_dev.clear();
    }
    c->dev_meta_stream = st;
    const bool same_ranks = c->dev_rank_ptr_valid && c->h_rank_ptr.size() == (size_t)R + 1 &&
                            std::equal(h_rank_ptr, h_rank_ptr + R + 1, c->h_rank_ptr.begin());
    c->h_rank_ptr.assign(h_rank_ptr, h_rank_ptr + R + 1);
    c->n_total = h_rank_ptr[R];
    c->max_nr = (int32_t)max_nr;
    c->d_lengths = d_lengths;
    CU(c, cudaSetDevice(c->device));
    if (!same_ranks) {
        c->dev_rank_ptr_valid = false;
        CU(c, cudaMemcpyAsync(c->d_rank_ptr, c->h_rank_ptr.data(), (R + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, st));
        c->dev_rank_ptr_valid = true;
    }
    if (!c->arrived_set) c->h_arrived.assign((size_t)R, 0x7fffffff);  // everything has arrived
    if (c->h_arrived != c->h_arrived_dev) {
        c->h_arrived_dev.clear();
        CU(c, cudaMemcpyAsync(c->d_arrived, c->h_arrived.data(), (size_t)R * sizeof(int32_t), cudaMemcpyHostToDevice, st));
        c->h_arrived_dev = c->h_arrived;
    }
    // rank state, emit positions, step totals, length validation: done by the first sort launch (or k_begin).
    // The status record: cleared by the slot scan of the previous complete plan when that ran on this stream.
    if (!(c->rec_clean && c->rec_clear_stream == st)) CU(c, cudaMemsetAsync(c->d_rec, 0, sizeof(RoundRec), st));
    c->rec_clean = false;
    c->begin_pending = true;
    c->n_finished = 0;
    for (int r = 0; r < R; ++r)
        if (h_rank_ptr[r + 1] == h_rank_ptr[r]) c->n_finished++;
    return ODB_OK;
}

// termination predicates, evaluated on the status shared by all ranks (Thm 3 proof P:341)
static bool check_terminated(odb_ctx *c) {
    const int R = c->prm.n_ranks;
    if (c->prm.join_mode && c->n_finished == R) {
        c->stop_reason = ODB_STOP_ALL_FINISHED;
        return true;
    }
    if (!c->prm.join_mode && c->n_finished > 0) {
        c->stop_reason = ODB_STOP_LOGICAL;
        return true;
    }
    return false;
}

int odb_form_groups(odb_ctx *c, const int32_t *d_lengths, const int64_t *h_rank_ptr, void *stream) {
    if (!c) return ODB_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    c->last_stream = st;
    if (c->state == 0) {
        int rc = begin_run(c, d_lengths, h_rank_ptr, st);
        if (rc != ODB_OK) return rc;
    } else if (c->state != 3) {
        return ODB_ERR_STATE;
    }
    CU(c, cudaSetDevice(c->device));
    // distributed mode: termination is decided on the device from the gathered world summary (k_align)
    if (!c->world_ranks && check_terminated(c)) {
        // the terminal check round: nothing to form; odb_align / odb_round_status report done
        CU(c, flush_begin(c, st));
        c->state = 1;
        c->last_T = 0;
        return ODB_OK;
    }
    const int R = c->prm.n_ranks;
    // make room for this round's steps: T <= the largest window, and <= slot_capacity
    int64_t bound = c->world_ranks ? std::max<int64_t>(c->max_nr, c->world_max_window) : c->max_nr;
    if (c->prm.buffer_size > 0) bound = std::min<int64_t>(bound, c->prm.buffer_size);
    if (c->prm.slot_capacity > 0) bound = std::min<int64_t>(bound, c->prm.slot_capacity);
    bound = std::max<int64_t>(bound, 1);
    const int64_t need = (int64_t)c->n_steps + bound;
    if (need > c->step_cap) {
        const int64_t want = need + need / 2 + 64;
        const size_t used = (size_t)c->n_steps * R;
        CU(c, grow_preserve(c->st_count, (size_t)want * R, used, st));
        CU(c, grow_preserve(c->st_width, (size_t)want * R, used, st));
        CU(c, grow_preserve(c->st_real, (size_t)want * R, used, st));
        CU(c, grow_preserve(c->st_round, (size_t)want * R, used, st));
        CU(c, grow_preserve(c->st_origin, (size_t)want * R, used, st));
        CU(c, grow_preserve(c->step_samples, (size_t)want, (size_t)c->n_steps, st));
        c->step_cap = want;
    }
    c->round_window = (int32_t)bound;
    CU(c, launch_round_form(c, st));
    if (c->world_ranks) CU(c, launch_pack_summary(c, st));
    c->state = 1;
    c->last_T = -1;
    return ODB_OK;
}

int odb_set_available(odb_ctx *c, const int64_t *h_arrived, void *stream) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (c->state != 0 && c->state != 3) return ODB_ERR_STATE;  // between rounds only
    const int R = c->prm.n_ranks;
    c->h_arrived.resize((size_t)R);
    for (int r = 0; r < R; ++r) {
        const int64_t a = h_arrived ? h_arrived[r] : 0x7fffffffll;
        c->h_arrived[r] = (int32_t)std::min<int64_t>(std::max<int64_t>(a, 0), 0x7fffffffll);
    }
    c->arrived_set = true;
    if (c->state == 3) {  // mid-run: the next odb_form_groups reads the device copy
        CU(c, cudaSetDevice(c->device));
        c->h_arrived_dev.clear();
        CU(c, cudaMemcpyAsync(c->d_arrived, c->h_arrived.data(), (size_t)R * sizeof(int32_t), cudaMemcpyHostToDevice,
                              (cudaStream_t)stream));
        c->h_arrived_dev = c->h_arrived;
        c->dev_meta_stream = (cudaStream_t)stream;
    }
    return ODB_OK;
}

int odb_emitted_counts(odb_ctx *c, int64_t *h_emitted) {
    if (!c || !h_emitted) return ODB_ERR_INVALID_ARG;
    if (c->state != 0 && c->state != 3 && c->state != 4 && c->state != 5) return ODB_ERR_STATE;  // not inside a round
    if (c->offline) return ODB_ERR_STATE;
    const int R = c->prm.n_ranks;
    if (c->state == 0) {  // nothing emitted yet (the cursors are cleared by the first round)
        for (int r = 0; r < R; ++r) h_emitted[r] = 0;
        return ODB_OK;
    }
    CU(c, cudaSetDevice(c->device));
    std::vector<int32_t> cur((size_t)R);
    // the rounds so far were enqueued on last_stream; the status of the last one has been read, so this waits for
    // nothing but the copy itself
    CU(c, cudaMemcpyAsync(cur.data(), c->emit_cur, (size_t)R * sizeof(int32_t), cudaMemcpyDeviceToHost, c->last_stream));
    CU(c, cudaStreamSynchronize(c->last_stream));
    for (int r = 0; r < R; ++r) h_emitted[r] = cur[(size_t)r];
    return ODB_OK;
}

int odb_fetch_quota(const odb_params *p, const int64_t *h_rank_ptr, int32_t prefetch_factor, int32_t num_workers,
                    const int64_t *h_emitted, int64_t *h_fetch_upto) {
    if (!p || !h_rank_ptr || !h_emitted || !h_fetch_upto || prefetch_factor < 0 || num_workers < 0 || p->n_ranks < 1 ||
        p->buffer_size < 0)
        return ODB_ERR_INVALID_ARG;
    // D = max(prefetch_factor * num_workers, buffer_size) (the clamp from below by buffer_size is App. P
    // P:767-771); buffer_size 0 = the window is the whole stream, so the envelope never binds
    const int64_t D = p->buffer_size > 0 ? std::max<int64_t>((int64_t)prefetch_factor * num_workers, p->buffer_size)
                                         : (int64_t)0x7fffffff;
    for (int r = 0; r < p->n_ranks; ++r) {
        const int64_t n_r = h_rank_ptr[r + 1] - h_rank_ptr[r];
        if (n_r < 0 || h_emitted[r] < 0 || h_emitted[r] > n_r) return ODB_ERR_INVALID_ARG;
        h_fetch_upto[r] = std::min<int64_t>(n_r, h_emitted[r] + D);  // |Q_r + B_r| = fetched - emitted <= D
    }
    return ODB_OK;
}

int odb_align(odb_ctx *c, void *stream) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (c->state != 1) return ODB_ERR_STATE;
    cudaStream_t st = (cudaStream_t)stream;
    CU(c, cudaSetDevice(c->device));
    if (c->last_T == 0) {  // terminal check round
        c->state = 2;
        return ODB_OK;
    }
    if (c->world_ranks) {  // the caller all_reduces the round's step_samples window, then odb_commit
        CU(c, launch_align_only(c, st));
        c->state = 6;
        return ODB_OK;
    }
    CU(c, launch_round_align(c, st));  // (single-process mode: k_commit's last CTA writes the status to the pinned h_rec)
    CU(c, cudaEventRecord(c->ev_status, st));
    c->state = 2;
    return ODB_OK;
}

int odb_commit(odb_ctx *c, void *stream) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (c->state != 6) return ODB_ERR_STATE;
    cudaStream_t st = (cudaStream_t)stream;
    CU(c, cudaSetDevice(c->device));
    CU(c, launch_commit_only(c, st));
    CU(c, cudaMemcpyAsync(c->h_rec, c->d_rec, sizeof(RoundRec), cudaMemcpyDeviceToHost, st));
    CU(c, cudaEventRecord(c->ev_status, st));
    c->state = 2;
    return ODB_OK;
}

int odb_dist_config(odb_ctx *c, int32_t world_ranks, int32_t rank_offset, int32_t world_max_window) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (c->state != 0 && c->state != 4 && c->state != 5) return ODB_ERR_STATE;  // not in the middle of a run
    const int R = c->prm.n_ranks;
    if (world_ranks == 0) {  // back to single-process mode
        c->world_ranks = 0;
        c->rank_offset = 0;
        c->world_max_window = 0;
        return ODB_OK;
    }
    if (world_ranks < R || world_ranks > 65535 || rank_offset < 0 || rank_offset + R > world_ranks || world_max_window < 0)
        return ODB_ERR_INVALID_ARG;
    CU(c, cudaSetDevice(c->device));
    if (!c->gs_local) CU(c, dev_alloc(&c->gs_local, 2 * (size_t)R));
    if (c->gs_world_cap < world_ranks) {
        if (c->gs_world) cudaFree(c->gs_world);
        c->gs_world = nullptr;
        CU(c, dev_alloc(&c->gs_world, 2 * (size_t)world_ranks));
        c->gs_world_cap = world_ranks;
    }
    c->world_ranks = world_ranks;
    c->rank_offset = rank_offset;
    c->world_max_window = world_max_window;
    odb_reset(c);
    return ODB_OK;
}

int odb_dist_buffers(odb_ctx *c, odb_dist_bufs *out) {
    if (!c || !out) return ODB_ERR_INVALID_ARG;
    if (!c->world_ranks) return ODB_ERR_STATE;
    memset(out, 0, sizeof(*out));
    out->d_summary_local = c->gs_local;
    out->d_summary_world = c->gs_world;
    out->summary_local_count = 2 * c->prm.n_ranks;
    out->summary_world_count = 2 * c->world_ranks;
    if (c->state == 1 || c->state == 6) {  // inside a round: the window of step totals this round may touch
        out->d_step_samples_round = c->step_samples.p + c->n_steps;
        out->step_window = c->round_window;
    }
    if (c->state == 7 || c->state == 8) {  // batched exchange: the local G table; the step totals of the whole run so far
        out->d_spec_G_local = c->dist_spec_G;
        out->spec_G_count = c->dist_spec_rounds * c->prm.n_ranks;
        out->d_step_samples_round = c->step_samples.p;
        out->step_window = (int32_t)std::min<int64_t>(c->step_cap, 0x7fffffff);
    }
    return ODB_OK;
}

// ---- distributed mode, batched exchange (the round-parallel planner over several processes) ----
int odb_dist_spec_form(odb_ctx *c, const int32_t *d_lengths, const int64_t *h_rank_ptr, int32_t n_rounds,
                       int64_t world_max_stream, void *stream) {
    if (!c || !h_rank_ptr) return ODB_ERR_INVALID_ARG;
    if (!c->world_ranks || c->state != 0 || c->arrived_set) return ODB_ERR_STATE;
    if (c->prm.buffer_size < kSpecMinWindow || c->prm.buffer_size > kSortChunk || n_rounds < 1 || n_rounds > kSpecMaxRounds ||
        (!c->prm.join_mode && c->prm.sample_quota > 0) || world_max_stream < 0)
        return ODB_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int R = c->prm.n_ranks;
    c->last_stream = st;
    int rc = begin_run(c, d_lengths, h_rank_ptr, st);
    if (rc != ODB_OK) return rc;
    // room for every step the job can have: n_steps <= the longest stream of the job, plus one round's window
    const int64_t steps_bound = std::max<int64_t>(world_max_stream, c->max_nr) + c->prm.buffer_size + 64;
    if (steps_bound > c->step_cap) {
        CU(c, grow_preserve(c->st_count, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->st_width, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->st_real, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->st_round, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->st_origin, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->step_samples, (size_t)steps_bound, 0, st));
        c->step_cap = steps_bound;
    }
    CU(c, launch_dist_spec_form(c, n_rounds, &c->dist_spec_G, st));
    c->begin_pending = false;
    c->dist_spec_rounds = n_rounds;
    c->state = 7;
    return ODB_OK;
}

int odb_dist_spec_commit(odb_ctx *c, const int32_t *d_G_world, const int32_t *d_n_world, int32_t n_procs, void *stream) {
    if (!c || !d_G_world || !d_n_world) return ODB_ERR_INVALID_ARG;
    if (c->state != 7) return ODB_ERR_STATE;
    if (n_procs < 1 || (int64_t)n_procs * c->prm.n_ranks != c->world_ranks) return ODB_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    CU(c, cudaSetDevice(c->device));
    CU(c, launch_dist_spec_commit(c, c->dist_spec_rounds, d_G_world, d_n_world, n_procs, st));
    if (!c->h_spec) CU(c, cudaMallocHost((void **)&c->h_spec, (4 + (size_t)kSpecMaxRounds + 1) * sizeof(int32_t)));
    // SpecRec, the bad-length flag and the rounds' T go back together (status read by odb_dist_spec_status)
    const size_t tab_fixed = 4 + (size_t)kSpecMaxRounds + 1;
    CU(c, cudaMemcpyAsync(c->h_spec, c->spec_tab.p, 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CU(c, cudaMemcpyAsync(c->h_spec + 4, c->spec_tab.p + tab_fixed, (size_t)c->dist_spec_rounds * sizeof(int32_t),
                          cudaMemcpyDeviceToHost, st));
    CU(c, cudaMemcpyAsync(c->h_rec, c->d_rec, sizeof(RoundRec), cudaMemcpyDeviceToHost, st));
    CU(c, cudaEventRecord(c->ev_status, st));
    c->state = 8;
    return ODB_OK;
}

int odb_dist_spec_status(odb_ctx *c, int32_t *h_rounds, int32_t *h_steps, int32_t *h_T, int32_t T_capacity, int32_t *h_done) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (c->state != 8) return ODB_ERR_STATE;
    CU(c, cudaEventSynchronize(c->ev_status));
    if (c->h_rec->bad_length) {
        c->state = 0;
        return ODB_ERR_BAD_LENGTH;
    }
    const int32_t js = c->h_spec[0], n_steps = c->h_spec[1];
    if (js < 0 || js > c->dist_spec_rounds || n_steps < 0 || n_steps > c->step_cap) return ODB_ERR_STATE;
    if (h_T && T_capacity < js) return ODB_ERR_CAPACITY;
    for (int j = 0; h_T && j < js; ++j) h_T[j] = c->h_spec[4 + j];
    c->round = js;
    c->n_steps = n_steps;
    c->last_T = js > 0 ? c->h_spec[4 + js - 1] : 0;
    c->spec_used = true;
    if (h_rounds) *h_rounds = js;
    if (h_steps) *h_steps = n_steps;
    if (c->h_spec[2]) {
        // every data round has been committed: round js is the terminal check (join: every stream is drained; non-join:
        // one is).  Every process reads this from the same gathered data (Lemma 3), so the round needs no exchange.
        c->stop_reason = c->prm.join_mode ? ODB_STOP_ALL_FINISHED : ODB_STOP_LOGICAL;
        c->n_rounds = js + 1;
        c->last_T = 0;
        c->state = 4;
        if (h_done) *h_done = 1;
        return ODB_OK;
    }
    if (h_done) *h_done = 0;
    c->state = 3;  // between rounds: odb_form_groups continues with round js
    return ODB_OK;
}

int odb_round_status(odb_ctx *c, int32_t *h_done, int32_t *h_T) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (c->state != 2) return ODB_ERR_STATE;
    if (c->last_T == 0) {  // the terminal check round
        if (c->round == 0 && c->n_total > 0) {  // no emitting round ran: still report bad lengths
            CU(c, cudaMemcpyAsync(c->h_rec, c->d_rec, sizeof(RoundRec), cudaMemcpyDeviceToHost, c->last_stream));
            CU(c, cudaStreamSynchronize(c->last_stream));
            if (c->h_rec->bad_length) {
                c->state = 0;
                return ODB_ERR_BAD_LENGTH;
            }
        }
        c->n_rounds = c->round + 1;
        c->state = 4;
        if (h_done) *h_done = 1;
        if (h_T) *h_T = 0;
        return ODB_OK;
    }
    CU(c, cudaEventSynchronize(c->ev_status));
    const RoundRec rec = *c->h_rec;
    if (rec.bad_length) {
        c->state = 0;
        return ODB_ERR_BAD_LENGTH;
    }
    if (rec.done) {  // distributed mode: the gathered status said "terminated"; nothing was emitted
        c->stop_reason = c->prm.join_mode ? ODB_STOP_ALL_FINISHED : ODB_STOP_LOGICAL;
        c->n_rounds = c->round + 1;
        c->last_T = 0;
        c->state = 4;
        if (h_done) *h_done = 1;
        if (h_T) *h_T = 0;
        return ODB_OK;
    }
    c->last_T = rec.T;
    c->n_steps += rec.T_emit;
    c->samples_emitted += rec.emitted_round;
    c->n_finished = rec.n_finished;
    c->round += 1;
    if (h_T) *h_T = rec.T;
    if (rec.quota_hit) {
        c->stop_reason = ODB_STOP_QUOTA;
        c->n_rounds = c->round;
        c->state = 4;
        if (h_done) *h_done = 1;
        return ODB_OK;
    }
    c->state = 3;
    if (h_done) *h_done = 0;
    return ODB_OK;
}

// internal rank-major tables for a plan of at most n_slots slots / n_steps steps
static int ensure_plan_tables(odb_ctx *c, size_t n_slots, size_t n_steps) {
    const size_t R = (size_t)c->prm.n_ranks;
    if (c->sub_mode) {  // a step range: no leftover tables
        CU(c, c->left_out.ensure(1));
        CU(c, c->left_ptr.ensure(R + 1));
    }
    CU(c, c->grp_count.ensure(n_slots + 1));
    CU(c, c->grp_width.ensure(n_slots + 1));
    CU(c, c->grp_round.ensure(n_slots + 1));
    CU(c, c->grp_valid.ensure(n_slots + 1));
    CU(c, c->grp_real.ensure(n_slots + 1));
    CU(c, c->grp_origin.ensure(n_slots + 1));
    CU(c, c->grp_offset.ensure(n_slots + 1));
    CU(c, c->grp_sample_ptr.ensure(n_slots + 1));
    CU(c, c->grp_sample_ids.ensure((size_t)c->n_total + 1));
    if (!c->sub_mode) {
        CU(c, c->left_out.ensure((size_t)c->n_total + 1));
        CU(c, c->left_ptr.ensure(R + 1));
    }
    CU(c, c->step_valid.ensure(n_steps + 1));
    return ODB_OK;
}

static void fill_info(odb_ctx *c) {
    odb_plan_info &I = c->info;
    const PlanDims &D = *c->h_dims;
    c->rec_clean = D.complete && !c->offline;  // (the slot scan that produced these sizes cleared the status record)
    I.n_rounds = c->n_rounds;
    I.n_steps = c->n_steps;
    I.stop_reason = c->stop_reason;
    I.reserved = 0;
    I.n_slots = (int64_t)c->prm.n_ranks * c->n_steps;
    I.total_elems = D.total_elems;
    I.samples_emitted = D.samples_emitted;
    I.samples_left = D.samples_left;  // Lemma 1: emitted + un-emitted = all (0 for an offline plan)
    I.real_tokens = (int64_t)D.real_tokens;
    I.padded_elems = D.padded_elems;
    c->info_valid = true;
}

int odb_plan_query(odb_ctx *c, odb_plan_info *h_out) {
    if (!c || !h_out) return ODB_ERR_INVALID_ARG;
    if (c->state == 5 && c->info_valid) {
        *h_out = c->info;
        return ODB_OK;
    }
    if (c->state != 4) return ODB_ERR_STATE;
    CU(c, cudaSetDevice(c->device));
    cudaStream_t st = c->last_stream;  // the stream of the last odb_form_groups / odb_align
    const int R = c->prm.n_ranks;
    const size_t n_slots = (size_t)R * (size_t)c->n_steps;
    {
        int rc = ensure_plan_tables(c, n_slots, (size_t)c->n_steps);
        if (rc != ODB_OK) return rc;
    }
    // the host has followed the rounds: its sizes go up, every later kernel reads them on the device
    PlanDims *U = c->h_dims_up;
    memset(U, 0, sizeof(*U));
    U->n_steps = c->n_steps;
    U->n_rounds = c->n_rounds;
    U->stop_reason = c->stop_reason;
    U->complete = 1;
    CU(c, cudaMemcpyAsync(c->d_dims, U, sizeof(PlanDims), cudaMemcpyHostToDevice, st));
    CapCheck cap = {-1, -1, -1, -1, -1, -1};
    CU(c, launch_finalize(c, (int64_t)n_slots, cap, c->h_rank_off, st));
    CU(c, cudaStreamSynchronize(st));
    fill_info(c);
    if (c->offline) {  // the slot CSR's (global) ids: wrap-around repetition can emit a sample twice
        CU(c, c->grp_sample_ids.ensure((size_t)c->info.samples_emitted + 1));
        CU(c, launch_offline_ids(c, st));
        CU(c, cudaMemsetAsync(c->left_ptr.p, 0, ((size_t)R + 1) * sizeof(int64_t), st));
    }
    c->state = 5;
    *h_out = c->info;
    return ODB_OK;
}

static int check_capacity(const odb_ctx *c, const odb_outputs *o) {
    const odb_plan_info &I = c->info;
    if (I.total_elems > 0) {
        if (!o->d_input_ids || !o->d_labels || !o->d_position_ids || !o->d_attention_mask) return ODB_ERR_INVALID_ARG;
        if (o->arena_capacity < I.total_elems) return ODB_ERR_CAPACITY;
    }
    const bool any_slot_tab = o->d_grp_count || o->d_grp_width || o->d_grp_round || o->d_grp_valid_tokens ||
                              o->d_grp_real_tokens || o->d_grp_origin || o->d_grp_offset || o->d_grp_sample_ptr;
    if (any_slot_tab && o->slot_capacity_alloc < I.n_slots) return ODB_ERR_CAPACITY;
    if (o->d_grp_sample_ids && o->ids_capacity < I.samples_emitted) return ODB_ERR_CAPACITY;
    if ((o->d_step_samples || o->d_step_valid_tokens) && o->step_capacity_alloc < I.n_steps) return ODB_ERR_CAPACITY;
    if (o->d_left_ids && o->left_capacity < I.samples_left) return ODB_ERR_CAPACITY;
    return ODB_OK;
}

// One collate launch.  whole = false: the arena elements [elem_lo, elem_hi) (both multiples of 16: slot
// offsets; tiles are arena-aligned, a tile that straddles elem_lo / elem_hi is visited by both neighbouring
// launches, each writing only its own elements); `counter` is this launch's zeroed work counter.
// whole = true: the whole arena, its extent read on the device from PlanDims (tile_bound = the most tiles
// it can have, for the grid), with the fused epilogue (step totals, the caller's valid-token tables).
static int collate_launch(odb_ctx *c, const int32_t *d_tokens, const int32_t *d_span_lo, const int32_t *d_span_hi,
                          const odb_outputs *o, bool whole, int64_t elem_lo, int64_t elem_hi, int64_t tile_bound,
                          unsigned long long *counter, cudaStream_t st) {
    CollateArgs A;
    memset(&A, 0, sizeof(A));
    A.tokens = d_tokens;
    A.rows = c->rows.p;
    A.row_sp = c->row_sp.p;
    A.span_lo = d_span_lo;
    A.span_hi = d_span_hi;
    A.grp_offset = c->grp_offset.p;
    A.grp_sample_ptr = c->grp_sample_ptr.p;
    A.grp_count = c->grp_count.p;
    A.grp_width = c->grp_width.p;
    A.tiles = c->tiles.p;
    A.dims = c->d_dims;
    A.ids = o->d_input_ids;
    A.labels = o->d_labels;
    A.pos = o->d_position_ids;
    A.mask = o->d_attention_mask;
    A.grp_valid = c->grp_valid.p;
    A.tile_counter = counter;
    A.pad_id = c->prm.pad_id;
    A.ignore_index = c->prm.ignore_index;
    A.shift_labels = c->prm.shift_labels;
    if (whole) {
        A.total_elems = 0;  // read on the device
        A.elem_lo = 0;
        A.tile_lo = 0;
        A.tile_hi = tile_bound;
        A.whole = 1;
    } else {
        A.total_elems = elem_hi;
        A.elem_lo = elem_lo;
        A.tile_lo = elem_lo / kColTile;
        A.tile_hi = (elem_hi + kColTile - 1) / kColTile;
    }
    CU(c, launch_collate(c, A, st));
    return ODB_OK;
}

static int check_pointers(const int32_t *d_tokens, const odb_outputs *o) {
    if (((uintptr_t)d_tokens & 15u) != 0) return ODB_ERR_INVALID_ARG;
    if (((uintptr_t)o->d_input_ids & 15u) || ((uintptr_t)o->d_labels & 15u) || ((uintptr_t)o->d_position_ids & 15u) ||
        ((uintptr_t)o->d_attention_mask & 15u))
        return ODB_ERR_INVALID_ARG;
    return ODB_OK;
}

// Everything behind the slot scan: collate preparation (one launch), the collate kernel over the whole
// arena (with the step totals fused into its last CTA).  Nothing here needs a size from the host: the
// kernels read PlanDims.  rows_bound / tile_bound size the library's row and tile tables.
static int enqueue_collate(odb_ctx *c, const int32_t *d_tokens, const int64_t *d_sample_ptr, const int64_t *d_span_ptr,
                           const int32_t *d_span_lo, const int32_t *d_span_hi, const odb_outputs *o, int64_t rows_bound,
                           int64_t tile_bound, cudaStream_t st) {
    CU(c, c->rows.ensure((size_t)rows_bound + 1));
    CU(c, c->row_sp.ensure((size_t)rows_bound + 1));
    CU(c, c->tiles.ensure((size_t)tile_bound + 2));
    CU(c, launch_prep(c, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, o, st));
    // ev[1]..ev[2] brackets the collate kernel alone; what precedes it is ev[0]..ev[1]
    if (c->timing) CU(c, cudaEventRecord(c->ev[1], st));
    {
        int rc = collate_launch(c, d_tokens, d_span_lo, d_span_hi, o, true, 0, 0, tile_bound, c->d_tile_counter, st);
        if (rc != ODB_OK) return rc;
    }
    if (c->timing) CU(c, cudaEventRecord(c->ev[2], st));
    {  // step totals (Eq. 2's T_tok per step) + the caller's valid-token tables
        PostArgs P;
        memset(&P, 0, sizeof(P));
        P.R = c->prm.n_ranks;
        P.dims = c->d_dims;
        P.grp_valid = c->grp_valid.p;
        P.step_valid = c->step_valid.p;
        P.user_step_valid = o->d_step_valid_tokens;
        P.user_grp_valid = o->d_grp_valid_tokens;
        CU(c, launch_post(c, P, st));
    }
    if (c->timing) CU(c, cudaEventRecord(c->ev[3], st));
    return ODB_OK;
}

static int collate_impl(odb_ctx *c, const int32_t *d_tokens, const int64_t *d_sample_ptr, const int64_t *d_span_ptr,
                        const int32_t *d_span_lo, const int32_t *d_span_hi, const odb_outputs *o, cudaStream_t st) {
    const odb_plan_info &I = c->info;
    if (I.samples_emitted > 0 && (!d_tokens || !d_sample_ptr)) return ODB_ERR_INVALID_ARG;
    {
        int rc = check_pointers(d_tokens, o);
        if (rc != ODB_OK) return rc;
    }
    const int64_t n_tiles = (I.total_elems + kColTile - 1) / kColTile;
    int rc = enqueue_collate(c, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, o, I.samples_emitted, n_tiles, st);
    if (rc != ODB_OK) return rc;
    if (c->timing) timing_done(c);
    c->collated = true;
    return ODB_OK;
}

int odb_collate(odb_ctx *c, const int32_t *d_tokens, const int64_t *d_sample_ptr, const int64_t *d_span_ptr,
                const int32_t *d_span_lo, const int32_t *d_span_hi, const odb_outputs *o, void *stream) {
    if (!c || !o) return ODB_ERR_INVALID_ARG;
    if (c->state != 5) return ODB_ERR_STATE;
    CU(c, cudaSetDevice(c->device));
    int rc = check_capacity(c, o);
    if (rc != ODB_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (c->timing) {
        timing_begin(c);
        CU(c, cudaEventRecord(c->ev[0], st));
    }
    return collate_impl(c, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, o, st);
}

static int run_rounds(odb_ctx *c, const int32_t *d_lengths, const int64_t *h_rank_ptr, odb_plan_info *h_out,
                      cudaStream_t st) {
    odb_reset(c);
    if (c->timing) {
        timing_begin(c);
        CU(c, cudaEventRecord(c->ev[0], st));
    }
    int32_t done = 0, T = 0;
    while (!done) {
        int rc = odb_form_groups(c, d_lengths, h_rank_ptr, st);
        if (rc != ODB_OK) return rc;
        rc = odb_align(c, st);
        if (rc != ODB_OK) return rc;
        rc = odb_round_status(c, &done, &T);
        if (rc != ODB_OK) return rc;
    }
    return odb_plan_query(c, h_out);
}

// Everything behind the round loop, enqueued BEFORE the host knows the plan: the slot scan (which checks the
// caller's capacities on the device), the read-back of the plan sizes with an event behind it, the collate
// preparation, the collate kernel and the step totals.  Every kernel reads PlanDims and does nothing unless
// the plan is complete and fits.  steps_bound >= the number of steps the plan can have.
static int enqueue_tail(odb_ctx *c, int64_t steps_bound, const int32_t *d_tokens, const int64_t *d_sample_ptr,
                        const int64_t *d_span_ptr, const int32_t *d_span_lo, const int32_t *d_span_hi,
                        const odb_outputs *o, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    const int64_t slots_bound = (int64_t)R * steps_bound;
    int rc = ensure_plan_tables(c, (size_t)slots_bound, (size_t)steps_bound);
    if (rc != ODB_OK) return rc;
    const int64_t tile_bound = (std::max<int64_t>(o->arena_capacity, 0) + kColTile - 1) / kColTile;
    CU(c, c->tiles.ensure((size_t)tile_bound + 2));
    const bool any_slot_tab = o->d_grp_count || o->d_grp_width || o->d_grp_round || o->d_grp_valid_tokens ||
                              o->d_grp_real_tokens || o->d_grp_origin || o->d_grp_offset || o->d_grp_sample_ptr;
    CapCheck cap;
    cap.arena = std::max<int64_t>(o->arena_capacity, 0);
    cap.slots = any_slot_tab ? o->slot_capacity_alloc : -1;
    cap.ids = o->d_grp_sample_ids ? o->ids_capacity : -1;
    cap.steps = (o->d_step_samples || o->d_step_valid_tokens) ? o->step_capacity_alloc : -1;
    cap.left = o->d_left_ids ? o->left_capacity : -1;
    cap.tiles = tile_bound;
    CU(c, launch_finalize(c, slots_bound, cap, c->h_rank_off, st));
    CU(c, cudaEventRecord(c->ev_plan, st));
    return enqueue_collate(c, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, o, c->n_total, tile_bound, st);
}

// Regime (A) of odb_run / odb_plan: every protocol round on the device (the round-parallel planner where it
// applies, then the persistent round loop).  *le = cudaSuccess: enqueued; otherwise the cooperative launch is not
// possible here (too many ranks for the device), the context has been reset and the caller drives the rounds
// from the host.  *steps_bound >= the steps the run can have.
static int fused_rounds(odb_ctx *c, const int32_t *d_lengths, const int64_t *h_rank_ptr, int64_t max_nr, int64_t window,
                        cudaStream_t st, int64_t *steps_bound_out, cudaError_t *le_out) {
    const int R = c->prm.n_ranks;
    c->last_stream = st;
    int rc = begin_run(c, d_lengths, h_rank_ptr, st);
    if (rc != ODB_OK) return rc;
    // room for every step the run can have: n_steps <= the longest stream (a rank that is active in every
    // emitting round emits at least T samples per round), plus one round's window
    const int64_t steps_bound = max_nr + window + 64;
    *steps_bound_out = steps_bound;
    if (steps_bound > c->step_cap) {
        CU(c, grow_preserve(c->st_count, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->st_width, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->st_real, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->st_round, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->st_origin, (size_t)steps_bound * R, 0, st));
        CU(c, grow_preserve(c->step_samples, (size_t)steps_bound, 0, st));
        c->step_cap = steps_bound;
    }
    // rounds that are certainly not the terminal check (join: some stream still holds views; non-join: every
    // stream does): formed and committed round-parallel as long as no round overflows (odb_plan.cu)
    int64_t spec_rounds = 0;
    bool spec_terminal = true;
    if (c->round_parallel && c->prm.buffer_size >= kSpecMinWindow) {
        const int64_t B = c->prm.buffer_size;
        int64_t min_nr = max_nr;
        for (int r = 0; r < R; ++r) min_nr = std::min(min_nr, h_rank_ptr[r + 1] - h_rank_ptr[r]);
        spec_rounds = ((c->prm.join_mode ? max_nr : min_nr) + B - 1) / B;
        if (!c->prm.join_mode && c->prm.sample_quota > 0) {
            // non-join with a sample quota (Thm 2 / P:347): a round-parallel round emits its whole windows, so the
            // rounds whose cumulative emission stays below the quota cannot contain the cut; the round that reaches
            // it -- and the cut inside it -- belongs to the sequential loop.  (the emission after j rounds is
            // monotone in j: bisection for the first j whose round reaches the quota)
            auto emitted_after = [&](int64_t rounds) {
                long long cum = (long long)c->prm.emitted_so_far;
                for (int r = 0; r < R; ++r) cum += std::min<int64_t>(rounds * B, h_rank_ptr[r + 1] - h_rank_ptr[r]);
                return cum;
            };
            int64_t lo = 0, hi = spec_rounds;  // the first j in [0, spec_rounds] with emitted_after(j + 1) >= quota
            while (lo < hi) {
                const int64_t mid = (lo + hi) / 2;
                if (emitted_after(mid + 1) >= (long long)c->prm.sample_quota) hi = mid;
                else lo = mid + 1;
            }
            if (lo < spec_rounds) {
                spec_rounds = lo;
                spec_terminal = false;
            }
        }
        if (spec_rounds < 2 || spec_rounds > kSpecMaxRounds) spec_rounds = 0;
    }
    const cudaError_t le = launch_rounds(c, (int)spec_rounds, spec_terminal, st);
    *le_out = le;
    if (le == cudaSuccess) {
        c->spec_used = spec_rounds > 0;
        c->begin_pending = false;
        return ODB_OK;
    }
    (void)cudaGetLastError();
    if (le != cudaErrorNotSupported) c->no_rounds_kernel = true;
    odb_reset(c);
    return ODB_OK;
}

// ... and the host's side of it: wait for the plan sizes (an event behind the slot scan) and take them over
static int fused_sizes(odb_ctx *c, odb_plan_info *h_out) {
    CU(c, cudaEventSynchronize(c->ev_plan));
    const PlanDims &D = *c->h_dims;
    if (D.bad_length) {
        c->state = 0;
        return ODB_ERR_BAD_LENGTH;
    }
    if (!D.complete) return D.err ? D.err : ODB_ERR_STATE;
    c->n_steps = D.n_steps;
    c->n_rounds = D.n_rounds;
    c->round = D.n_rounds;
    c->stop_reason = D.stop_reason;
    c->samples_emitted = D.samples_emitted;
    fill_info(c);
    c->state = 5;
    *h_out = c->info;
    return D.err;  // ODB_ERR_CAPACITY: the kernels behind the slot scan wrote nothing
}

static bool fused_applies(const odb_ctx *c, int64_t max_nr, int64_t window) {
    return max_nr > 0 && window <= kSortChunk && !c->no_rounds_kernel &&
           (int64_t)c->prm.n_ranks * (max_nr + window + 64) <= (1ll << 27);
}

// the whole plan: every round on the device where that applies, else host-driven rounds; ends in state 5
static int plan_impl(odb_ctx *c, const int32_t *d_lengths, const int64_t *h_rank_ptr, odb_plan_info *h_out, cudaStream_t st) {
    const int R = c->prm.n_ranks;
    int64_t max_nr = 0;
    for (int r = 0; r < R; ++r) max_nr = std::max(max_nr, h_rank_ptr[r + 1] - h_rank_ptr[r]);
    const int64_t window = c->prm.buffer_size > 0 ? std::min<int64_t>(max_nr, c->prm.buffer_size) : max_nr;
    odb_reset(c);
    CU(c, cudaSetDevice(c->device));
    if (c->timing) {  // (odb_run_host closes the quadruple)
        timing_begin(c);
        CU(c, cudaEventRecord(c->ev[0], st));
    }
    if (fused_applies(c, max_nr, window)) {
        int64_t steps_bound = 0;
        cudaError_t le = cudaSuccess;
        int rc = fused_rounds(c, d_lengths, h_rank_ptr, max_nr, window, st, &steps_bound, &le);
        if (rc != ODB_OK) return rc;
        if (le == cudaSuccess) {
            const int64_t slots_bound = (int64_t)R * steps_bound;
            rc = ensure_plan_tables(c, (size_t)slots_bound, (size_t)steps_bound);
            if (rc != ODB_OK) return rc;
            const CapCheck cap = {-1, -1, -1, -1, -1, -1};
            CU(c, launch_finalize(c, slots_bound, cap, c->h_rank_off, st));
            CU(c, cudaEventRecord(c->ev_plan, st));
            return fused_sizes(c, h_out);
        }
    }
    return run_rounds(c, d_lengths, h_rank_ptr, h_out, st);
}

int odb_plan(odb_ctx *c, const int32_t *d_lengths, const int64_t *h_rank_ptr, odb_plan_info *h_out, void *stream) {
    if (!c || !h_out || !h_rank_ptr) return ODB_ERR_INVALID_ARG;
    if (c->world_ranks) return ODB_ERR_STATE;
    return plan_impl(c, d_lengths, h_rank_ptr, h_out, (cudaStream_t)stream);
}

int odb_collate_steps(odb_ctx *c, int32_t step_lo, int32_t step_hi, const int32_t *d_tokens, const int64_t *d_sample_ptr,
                      const int64_t *d_span_ptr, const int32_t *d_span_lo, const int32_t *d_span_hi, const odb_outputs *o,
                      odb_plan_info *h_out, void *stream) {
    if (!c || !o || !h_out) return ODB_ERR_INVALID_ARG;
    if ((c->state != 3 && c->state != 4 && c->state != 5) || c->offline || c->world_ranks) return ODB_ERR_STATE;
    if (step_lo < 0 || step_hi < step_lo || step_hi > c->n_steps) return ODB_ERR_INVALID_ARG;
    const bool arenas = o->d_input_ids && o->d_labels && o->d_position_ids && o->d_attention_mask;
    if (arenas && (!d_tokens || !d_sample_ptr || check_pointers(d_tokens, o) != ODB_OK)) return ODB_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    CU(c, cudaSetDevice(c->device));
    const int R = c->prm.n_ranks;
    const int n = step_hi - step_lo;
    SubTabs &T = c->sub[c->sub_seq & 1];
    if (!T.ready) {
        CU(c, dev_alloc(&T.d_dims, 1));
        CU(c, cudaMemset(T.d_dims, 0, sizeof(PlanDims)));
        CU(c, dev_alloc(&T.d_tile_counter, (size_t)R + 1));
        CU(c, cudaMallocHost((void **)&T.h_dims, sizeof(PlanDims)));
        CU(c, cudaEventCreateWithFlags(&T.ev_plan, cudaEventDisableTiming));
        T.ready = true;
    }
    // the full plan's slot CSR (state 5) tells where a rank's rows of the range start in its emit region
    const int64_t *full_sp = (c->state == 5 && c->info_valid && c->n_steps > 0) ? c->grp_sample_ptr.p : nullptr;
    const int full_K = c->n_steps;
    // (a set is reused by every second call: its previous plan sizes have been read, its kernels are ordered by
    //  the caller's streams -- at most two step ranges in flight)
    swap_tabs(c, T);
    c->sub_mode = true;
    c->sub_step_lo = step_lo;
    const int timing = c->timing;
    c->timing = 0;
    int rc = [&]() -> int {
        const int64_t slots = (int64_t)R * n;
        // Table sizes: growing a table is cudaFree + cudaMalloc, both device-wide synchronisations that would stall the
        // range in flight on the other stream.  Once the whole plan is known (odb_plan) every table of a set is
        // therefore sized for the WHOLE plan the first time the set is used -- a few bytes per slot, 12 per tile --
        // and no later range (a longer chunk, a larger arena) grows it.  While rounds are still being added (state 3)
        // the plan's size is open and a range larger than any before it does grow the set.
        const bool whole = c->state == 5 && c->info_valid;
        const int64_t slots_alloc = whole ? std::max<int64_t>(slots, (int64_t)R * c->n_steps) : slots;
        const int64_t steps_alloc = whole ? std::max<int64_t>(n, c->n_steps) : n;
        int rc2 = ensure_plan_tables(c, (size_t)slots_alloc, (size_t)steps_alloc);
        if (rc2 != ODB_OK) return rc2;
        int64_t tile_bound = (std::max<int64_t>(o->arena_capacity, 0) + kColTile - 1) / kColTile;
        if (whole) {  // (a range holds a subset of the plan's blocks: never more tiles than the plan)
            const int64_t plan_tiles = (c->info.total_elems + kColTile - 1) / kColTile;
            tile_bound = std::min(tile_bound, plan_tiles);
            CU(c, c->tiles.ensure((size_t)plan_tiles + 2));
        }
        const bool any_slot_tab = o->d_grp_count || o->d_grp_width || o->d_grp_round || o->d_grp_valid_tokens ||
                                  o->d_grp_real_tokens || o->d_grp_origin || o->d_grp_offset || o->d_grp_sample_ptr;
        CapCheck cap;
        cap.arena = arenas ? std::max<int64_t>(o->arena_capacity, 0) : 0;
        cap.slots = any_slot_tab ? o->slot_capacity_alloc : -1;
        cap.ids = o->d_grp_sample_ids ? o->ids_capacity : -1;
        cap.steps = (o->d_step_samples || o->d_step_valid_tokens) ? o->step_capacity_alloc : -1;
        cap.left = -1;
        cap.tiles = tile_bound;
        CU(c, launch_sub_dims(c, n, st));
        CU(c, launch_finalize(c, slots, cap, nullptr, st, step_lo, slots_alloc));
        CU(c, cudaEventRecord(c->ev_plan, st));
        CU(c, launch_sub_ids(c, step_lo, o->d_grp_sample_ids, full_sp, full_K, st));
        if (!arenas) return ODB_OK;  // a sizing call
        return enqueue_collate(c, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, o, c->n_total, tile_bound, st);
    }();
    c->timing = timing;
    c->sub_mode = false;
    swap_tabs(c, T);
    // a sizing call (no arenas) enqueues no collate kernel: the real call that follows it takes the SAME table set, on
    // the same stream, so that "sizing call, then the range" still leaves the other set to the other range in flight
    if (arenas) c->sub_seq++;
    if (rc != ODB_OK) return rc;
    CU(c, cudaEventSynchronize(T.ev_plan));  // the range's sizes; its collate kernel is running
    const PlanDims &D = *T.h_dims;
    memset(h_out, 0, sizeof(*h_out));
    h_out->n_rounds = c->state == 3 ? c->round : c->n_rounds;
    h_out->n_steps = n;
    h_out->stop_reason = c->state == 3 ? 0 : c->stop_reason;
    h_out->n_slots = D.n_slots;
    h_out->total_elems = D.total_elems;
    h_out->samples_emitted = D.samples_emitted;
    h_out->samples_left = 0;
    h_out->real_tokens = (int64_t)D.real_tokens;
    h_out->padded_elems = D.padded_elems;
    if (D.err) return D.err;
    if (!arenas && D.total_elems > 0) return ODB_ERR_CAPACITY;
    return ODB_OK;
}

int odb_run(odb_ctx *c, const int32_t *d_lengths, const int64_t *h_rank_ptr, const int32_t *d_tokens,
            const int64_t *d_sample_ptr, const int64_t *d_span_ptr, const int32_t *d_span_lo, const int32_t *d_span_hi,
            const odb_outputs *o, odb_plan_info *h_out, void *stream) {
    if (!c || !o || !h_out || !h_rank_ptr) return ODB_ERR_INVALID_ARG;
    if (c->world_ranks) return ODB_ERR_STATE;  // the caller drives the rounds and their collectives
    cudaStream_t st = (cudaStream_t)stream;
    const int R = c->prm.n_ranks;
    // NOTHING needs the host between the first kernel and the last when
    //  (A) the windows are small (<= 4096 samples: the paper's regime) and the R ranks fit the device:
    //      ONE persistent kernel runs every protocol round (k_rounds), or
    //  (B) every rank's whole stream fits its window and the output slots are unlimited: the protocol
    //      normally ends with the first round (unequal group counts are levelled by splitting; only unequal
    //      windows overflow), and k_commit closes the round on the device.
    // The slot scan, the collate preparation and the collate kernel are enqueued behind the rounds; they read
    // the plan sizes from PlanDims and check the caller's capacities on the device.  The host waits only for
    // the sizes (an event behind the slot scan) while the collate kernel is already running.  If (B)'s first
    // round does not end the protocol, those launches were no-ops and the staged loop below takes over.
    int64_t max_nr = 0;
    for (int r = 0; r < R; ++r) max_nr = std::max(max_nr, h_rank_ptr[r + 1] - h_rank_ptr[r]);
    const int64_t window = c->prm.buffer_size > 0 ? std::min<int64_t>(max_nr, c->prm.buffer_size) : max_nr;
    const bool arenas = o->d_input_ids && o->d_labels && o->d_position_ids && o->d_attention_mask;
    const bool async_ok = arenas && d_tokens && d_sample_ptr && check_pointers(d_tokens, o) == ODB_OK && max_nr > 0;
    const bool fused = async_ok && fused_applies(c, max_nr, window);
    const bool speculate = async_ok && !fused && window >= max_nr && c->prm.slot_capacity == 0;
    odb_reset(c);
    CU(c, cudaSetDevice(c->device));
    if (c->timing) {
        timing_begin(c);
        CU(c, cudaEventRecord(c->ev[0], st));
    }
    int32_t done = 0, T = 0;
    int rc;
    if (fused) {
        int64_t steps_bound = 0;
        cudaError_t le = cudaSuccess;
        rc = fused_rounds(c, d_lengths, h_rank_ptr, max_nr, window, st, &steps_bound, &le);
        if (rc != ODB_OK) return rc;
        if (le == cudaSuccess) {
            rc = enqueue_tail(c, steps_bound, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, o, st);
            if (rc != ODB_OK) return rc;
            rc = fused_sizes(c, h_out);  // the sizes are here; the collate kernel is running
            if (rc != ODB_OK) return rc;
            if (c->timing) timing_done(c);
            c->collated = true;
            return ODB_OK;
        }
    }
    rc = odb_form_groups(c, d_lengths, h_rank_ptr, st);
    if (rc != ODB_OK) return rc;
    bool collate_enqueued = false;
    if (speculate && c->last_T != 0) {  // an emitting round was formed
        rc = odb_align(c, st);
        if (rc != ODB_OK) return rc;
        rc = enqueue_tail(c, c->round_window /* T_grp <= the largest window */, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo,
                          d_span_hi, o, st);
        if (rc != ODB_OK) return rc;
        CU(c, cudaEventSynchronize(c->ev_plan));  // the sizes are here; the collate kernel is running
        collate_enqueued = c->h_dims->complete != 0;
        rc = odb_round_status(c, &done, &T);
        if (rc != ODB_OK) return rc;
    } else {
        rc = odb_align(c, st);
        if (rc != ODB_OK) return rc;
        rc = odb_round_status(c, &done, &T);
        if (rc != ODB_OK) return rc;
    }
    while (!done) {  // (after a speculated round that ended the protocol: the terminal check, no launch)
        rc = odb_form_groups(c, d_lengths, h_rank_ptr, st);
        if (rc != ODB_OK) return rc;
        rc = odb_align(c, st);
        if (rc != ODB_OK) return rc;
        rc = odb_round_status(c, &done, &T);
        if (rc != ODB_OK) return rc;
    }
    if (collate_enqueued) {
        const PlanDims &D = *c->h_dims;
        // the device closed the round with the predicates the host state machine has just applied
        if (D.n_steps != c->n_steps || D.n_rounds != c->n_rounds || D.stop_reason != c->stop_reason) return ODB_ERR_STATE;
        fill_info(c);
        c->state = 5;
        *h_out = c->info;
        if (D.err) return D.err;  // ODB_ERR_CAPACITY: the kernels behind the slot scan wrote nothing
        if (c->timing) timing_done(c);
        c->collated = true;
        return ODB_OK;
    }
    rc = odb_plan_query(c, h_out);
    if (rc != ODB_OK) return rc;
    rc = check_capacity(c, o);
    if (rc != ODB_OK) return rc;
    return collate_impl(c, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, o, st);
}

// a pool of timing-less events (odb_run_host orders its three streams with one event per token load and two
// per output piece)
static cudaError_t pool_event(odb_ctx *c, size_t i, cudaEvent_t *out) {
    while (c->ev_pool.size() <= i) {
        cudaEvent_t e = nullptr;
        cudaError_t rc = cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
        if (rc != cudaSuccess) return rc;
        c->ev_pool.push_back(e);
    }
    *out = c->ev_pool[i];
    return cudaSuccess;
}

// Device memory of odb_run_host does NOT grow with the job: the tokens go through a ring of three rank-sized
// buffers, the four arenas through a ring of three fixed-size pieces (host_staging_elems elements each), so a job
// whose inputs and outputs exceed the device memory still runs.  Three streams: lengths go up first on the compute
// stream (planning needs nothing else); the CSR arrays and then the tokens go up RANK BY RANK on the copy stream
// (a ring slot is reused once the rank that held it has been collated); a rank's slots are collated piece by piece
// as soon as its tokens have landed (a piece = a tile-aligned range of arena elements inside the rank's range; a
// tile that straddles a rank boundary is visited by both neighbouring launches, each writing only its own
// elements), and every piece goes down on the third stream while later pieces are collated and later ranks
// uploaded: both directions of the host link are busy at once.
static int run_host_impl(odb_ctx *c, const int32_t *h_lengths, const int64_t *h_rank_ptr, const int32_t *h_tokens,
                 const int64_t *h_sample_ptr, const int64_t *h_span_ptr, const int32_t *h_span_lo,
                 const int32_t *h_span_hi, const odb_outputs *ho, odb_plan_info *h_out, void *stream) {
    if (!c || !ho || !h_out || !h_rank_ptr) return ODB_ERR_INVALID_ARG;
    if (c->world_ranks) return ODB_ERR_STATE;
    cudaStream_t st = (cudaStream_t)stream;
    CU(c, cudaSetDevice(c->device));
    const int R = c->prm.n_ranks;
    const int64_t N = h_rank_ptr[R];
    if (N < 0 || N > c->n_max) return ODB_ERR_INVALID_ARG;
    if (N > 0 && (!h_lengths || !h_sample_ptr || !h_tokens)) return ODB_ERR_INVALID_ARG;
    const int64_t n_span = (h_span_ptr && N > 0) ? h_span_ptr[N] : 0;
    int64_t max_rank_tok = 0;
    for (int r = 0; r < R && N > 0; ++r)
        max_rank_tok = std::max(max_rank_tok, h_sample_ptr[h_rank_ptr[r + 1]] - h_sample_ptr[h_rank_ptr[r]]);
    constexpr int kRing = 3;
    const size_t tok_slot = ((size_t)max_rank_tok + 8 + 3) & ~(size_t)3;  // ints per ring slot (16-byte multiples)
    const int64_t piece = std::max<int64_t>(kColTile, (c->host_staging_elems / kColTile) * kColTile);
    CU(c, c->hs_lengths.ensure((size_t)N + 1));
    CU(c, c->hs_sample_ptr.ensure((size_t)N + 1));
    CU(c, c->hs_span_ptr.ensure((size_t)N + 1));
    CU(c, c->hs_span_lo.ensure((size_t)n_span + 1));
    CU(c, c->hs_span_hi.ensure((size_t)n_span + 1));
    CU(c, c->hs_tokens.ensure(kRing * tok_slot + 16));
    if (!c->host_device_arenas) {
        CU(c, c->hs_ids.ensure(kRing * (size_t)piece + 16));
        CU(c, c->hs_labels.ensure(kRing * (size_t)piece + 16));
        CU(c, c->hs_pos.ensure(kRing * (size_t)piece + 16));
        CU(c, c->hs_mask.ensure(kRing * (size_t)piece + 16));
    }
    if (!c->copy_stream) {
        CU(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        CU(c, cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking));
        CU(c, cudaEventCreateWithFlags(&c->copy_ev, cudaEventDisableTiming));
    }
    // events: [0, R) tokens of rank r landed; [R, 2R) rank r collated; then two per piece (collated, copied back)
    auto drain = [&]() {
        cudaStreamSynchronize(c->copy_stream);
        cudaStreamSynchronize(c->d2h_stream);
        cudaStreamSynchronize(st);
    };
    if (N > 0) CU(c, cudaMemcpyAsync(c->hs_lengths.p, h_lengths, (size_t)N * 4, cudaMemcpyHostToDevice, st));
    CU(c, cudaEventRecord(c->copy_ev, st));
    CU(c, cudaStreamWaitEvent(c->copy_stream, c->copy_ev, 0));  // orders this call after the previous one's reads
    CU(c, cudaStreamWaitEvent(c->d2h_stream, c->copy_ev, 0));
    if (N > 0) {
        CU(c, cudaMemcpyAsync(c->hs_sample_ptr.p, h_sample_ptr, (size_t)(N + 1) * 8, cudaMemcpyHostToDevice, c->copy_stream));
        if (h_span_ptr) {
            CU(c, cudaMemcpyAsync(c->hs_span_ptr.p, h_span_ptr, (size_t)(N + 1) * 8, cudaMemcpyHostToDevice, c->copy_stream));
            if (n_span) {
                CU(c, cudaMemcpyAsync(c->hs_span_lo.p, h_span_lo, (size_t)n_span * 4, cudaMemcpyHostToDevice, c->copy_stream));
                CU(c, cudaMemcpyAsync(c->hs_span_hi.p, h_span_hi, (size_t)n_span * 4, cudaMemcpyHostToDevice, c->copy_stream));
            }
        }
    }
    CU(c, cudaEventRecord(c->copy_ev, c->copy_stream));  // CSR arrays landed
    // the first ring's worth of tokens can go up while the plan is being made
    auto upload_rank = [&](int r) -> int {
        cudaEvent_t ev;
        if (r >= kRing) {  // the slot is free once the rank that held it has been collated
            CU(c, pool_event(c, (size_t)R + (size_t)(r - kRing), &ev));
            CU(c, cudaStreamWaitEvent(c->copy_stream, ev, 0));
        }
        if (N > 0) {
            const int64_t t0 = h_sample_ptr[h_rank_ptr[r]], t1 = h_sample_ptr[h_rank_ptr[r + 1]];
            // placed so that (slot + (t0 & 3)) - t0 is 16-byte aligned: the kernel's aligned vector loads see the same
            // skew as in the caller's buffer
            int32_t *dst = c->hs_tokens.p + (size_t)(r % kRing) * tok_slot + (size_t)(t0 & 3);
            if (t1 > t0)
                CU(c, cudaMemcpyAsync(dst, h_tokens + t0, (size_t)(t1 - t0) * 4, cudaMemcpyHostToDevice, c->copy_stream));
        }
        CU(c, pool_event(c, (size_t)r, &ev));
        CU(c, cudaEventRecord(ev, c->copy_stream));
        return ODB_OK;
    };
    int uploaded = 0;
    for (; uploaded < std::min(R, kRing); ++uploaded) {
        int urc = upload_rank(uploaded);
        if (urc != ODB_OK) {
            drain();
            return urc;
        }
    }
    int rc = plan_impl(c, c->hs_lengths.p, h_rank_ptr, h_out, st);
    if (rc != ODB_OK) {
        drain();
        return rc;
    }
    const odb_plan_info I = *h_out;
    {  // host capacities
        const bool any_slot_tab = ho->d_grp_count || ho->d_grp_width || ho->d_grp_round || ho->d_grp_valid_tokens ||
                                  ho->d_grp_real_tokens || ho->d_grp_origin || ho->d_grp_offset || ho->d_grp_sample_ptr;
        if (I.total_elems > 0 && (!ho->d_input_ids || !ho->d_labels || !ho->d_position_ids || !ho->d_attention_mask))
            rc = ODB_ERR_INVALID_ARG;
        else if (I.total_elems > ho->arena_capacity)
            rc = ODB_ERR_CAPACITY;
        if (rc == ODB_OK && any_slot_tab && ho->slot_capacity_alloc < I.n_slots) rc = ODB_ERR_CAPACITY;
        if (rc == ODB_OK && ho->d_grp_sample_ids && ho->ids_capacity < I.samples_emitted) rc = ODB_ERR_CAPACITY;
        if (rc == ODB_OK && (ho->d_step_samples || ho->d_step_valid_tokens) && ho->step_capacity_alloc < I.n_steps)
            rc = ODB_ERR_CAPACITY;
        if (rc == ODB_OK && ho->d_left_ids && ho->left_capacity < I.samples_left) rc = ODB_ERR_CAPACITY;
        if (rc == ODB_OK && c->host_device_arenas && check_pointers(nullptr, ho) != ODB_OK) rc = ODB_ERR_INVALID_ARG;
    }
    if (rc != ODB_OK) {
        drain();
        return rc;
    }
    const size_t n_slots = (size_t)I.n_slots;
    CU(c, c->rows.ensure((size_t)I.samples_emitted + 1));
    CU(c, c->row_sp.ensure((size_t)I.samples_emitted + 1));
    CU(c, c->tiles.ensure((size_t)((I.total_elems + kColTile - 1) / kColTile) + 2));
    // pieces: every rank's arena range [lo, hi) cut at tile-aligned positions, at most `piece` elements each
    // (device arenas: a rank's range is one piece, written in place)
    const bool dev_arenas = c->host_device_arenas;
    int64_t n_pieces = 0;
    for (int r = 0; r < R; ++r) {
        const int64_t lo = c->h_rank_off[r], hi = c->h_rank_off[r + 1];
        if (dev_arenas) n_pieces += hi > lo ? 1 : 0;
        else
            for (int64_t cur = lo; cur < hi; ++n_pieces) cur = std::min(hi, (cur / kColTile) * kColTile + piece);
    }
    CU(c, c->piece_ctr.ensure((size_t)n_pieces + 1));
    CU(c, cudaMemsetAsync(c->piece_ctr.p, 0, ((size_t)n_pieces + 1) * sizeof(unsigned long long), st));
    CU(c, cudaStreamWaitEvent(st, c->copy_ev, 0));  // sample_ptr / spans have landed
    // row descriptors, tile table, id / leftover tables: one launch
    CU(c, launch_prep(c, c->hs_sample_ptr.p, h_span_ptr ? c->hs_span_ptr.p : nullptr, c->hs_span_lo.p, c->hs_span_hi.p,
                      nullptr, st));
    if (c->timing) CU(c, cudaEventRecord(c->ev[1], st));
    int64_t pi = 0;
    const size_t ev_piece0 = 2 * (size_t)R;
    for (int r = 0; r < R; ++r) {
        const int64_t lo = c->h_rank_off[r], hi = c->h_rank_off[r + 1];
        cudaEvent_t ev;
        if (hi > lo) {
            CU(c, pool_event(c, (size_t)r, &ev));
            CU(c, cudaStreamWaitEvent(st, ev, 0));  // the rank's tokens have landed
            const int64_t t0 = N > 0 ? h_sample_ptr[h_rank_ptr[r]] : 0;
            const int32_t *tok_base = c->hs_tokens.p + (size_t)(r % kRing) * tok_slot + (size_t)(t0 & 3) - t0;
            if (dev_arenas) {  // the arenas are device memory: the rank's slots are collated in place, nothing comes back
                rc = collate_launch(c, tok_base, c->hs_span_lo.p, c->hs_span_hi.p, ho, false, lo, hi, 0, c->piece_ctr.p + pi, st);
                if (rc != ODB_OK) {
                    drain();
                    return rc;
                }
                ++pi;
            }
            for (int64_t cur = lo; cur < hi && !dev_arenas;) {
                const int64_t end = std::min(hi, (cur / kColTile) * kColTile + piece);
                const size_t slot = (size_t)(pi % kRing) * (size_t)piece;
                if (pi >= kRing) {  // the staging piece is free once its previous contents have been copied back
                    CU(c, pool_event(c, ev_piece0 + 2 * (size_t)(pi - kRing) + 1, &ev));
                    CU(c, cudaStreamWaitEvent(st, ev, 0));
                }
                odb_outputs dev;
                memset(&dev, 0, sizeof(dev));
                // arena element a of this piece lives at staging element a - cur (cur is a multiple of 16)
                dev.d_input_ids = c->hs_ids.p + slot - cur;
                dev.d_labels = c->hs_labels.p + slot - cur;
                dev.d_position_ids = c->hs_pos.p + slot - cur;
                dev.d_attention_mask = c->hs_mask.p + slot - cur;
                rc = collate_launch(c, tok_base, c->hs_span_lo.p, c->hs_span_hi.p, &dev, false, cur, end, 0, c->piece_ctr.p + pi, st);
                if (rc != ODB_OK) {
                    drain();
                    return rc;
                }
                CU(c, pool_event(c, ev_piece0 + 2 * (size_t)pi, &ev));
                CU(c, cudaEventRecord(ev, st));
                CU(c, cudaStreamWaitEvent(c->d2h_stream, ev, 0));
                const size_t n = (size_t)(end - cur);
                CU(c, cudaMemcpyAsync(ho->d_input_ids + cur, c->hs_ids.p + slot, n * 4, cudaMemcpyDeviceToHost, c->d2h_stream));
                CU(c, cudaMemcpyAsync(ho->d_labels + cur, c->hs_labels.p + slot, n * 4, cudaMemcpyDeviceToHost, c->d2h_stream));
                CU(c, cudaMemcpyAsync(ho->d_position_ids + cur, c->hs_pos.p + slot, n * 4, cudaMemcpyDeviceToHost, c->d2h_stream));
                CU(c, cudaMemcpyAsync(ho->d_attention_mask + cur, c->hs_mask.p + slot, n, cudaMemcpyDeviceToHost, c->d2h_stream));
                CU(c, pool_event(c, ev_piece0 + 2 * (size_t)pi + 1, &ev));
                CU(c, cudaEventRecord(ev, c->d2h_stream));
                cur = end;
                ++pi;
            }
        }
        CU(c, pool_event(c, (size_t)R + (size_t)r, &ev));
        CU(c, cudaEventRecord(ev, st));  // rank r is collated: its token slot may be reused
        if (uploaded < R) {
            int urc = upload_rank(uploaded++);
            if (urc != ODB_OK) {
                drain();
                return urc;
            }
        }
    }
    if (c->timing) CU(c, cudaEventRecord(c->ev[2], st));
    {  // step totals (Eq. 2's T_tok per step)
        PostArgs P;
        memset(&P, 0, sizeof(P));
        P.R = R;
        P.dims = c->d_dims;
        P.grp_valid = c->grp_valid.p;
        P.step_valid = c->step_valid.p;
        CU(c, launch_post(c, P, st));
    }
    if (c->timing) {
        CU(c, cudaEventRecord(c->ev[3], st));
        timing_done(c);
    }
    c->collated = true;
    // tables device -> host (small) on the compute stream
    auto d2h = [&](void *dst, const void *src, size_t bytes) -> cudaError_t {
        if (!dst || bytes == 0) return cudaSuccess;
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st);
    };
    CU(c, d2h(ho->d_grp_count, c->grp_count.p, n_slots * 4));
    CU(c, d2h(ho->d_grp_width, c->grp_width.p, n_slots * 4));
    CU(c, d2h(ho->d_grp_round, c->grp_round.p, n_slots * 4));
    CU(c, d2h(ho->d_grp_valid_tokens, c->grp_valid.p, n_slots * 4));
    CU(c, d2h(ho->d_grp_real_tokens, c->grp_real.p, n_slots * 4));
    CU(c, d2h(ho->d_grp_origin, c->grp_origin.p, n_slots * 4));
    CU(c, d2h(ho->d_grp_offset, c->grp_offset.p, n_slots * 8));
    CU(c, d2h(ho->d_grp_sample_ptr, c->grp_sample_ptr.p, (n_slots + 1) * 8));
    CU(c, d2h(ho->d_grp_sample_ids, c->grp_sample_ids.p, (size_t)I.samples_emitted * 4));
    CU(c, d2h(ho->d_step_samples, c->step_samples.p, (size_t)I.n_steps * 4));
    CU(c, d2h(ho->d_step_valid_tokens, c->step_valid.p, (size_t)I.n_steps * 8));
    CU(c, d2h(ho->d_left_ptr, c->left_ptr.p, (size_t)(R + 1) * 8));
    CU(c, d2h(ho->d_left_ids, c->left_out.p, (size_t)I.samples_left * 4));
    CU(c, cudaStreamSynchronize(st));
    CU(c, cudaStreamSynchronize(c->d2h_stream));
    CU(c, cudaStreamSynchronize(c->copy_stream));
    return ODB_OK;
}

int odb_run_host(odb_ctx *c, const int32_t *h_lengths, const int64_t *h_rank_ptr, const int32_t *h_tokens,
                 const int64_t *h_sample_ptr, const int64_t *h_span_ptr, const int32_t *h_span_lo,
                 const int32_t *h_span_hi, const odb_outputs *ho, odb_plan_info *h_out, void *stream) {
    const int rc = run_host_impl(c, h_lengths, h_rank_ptr, h_tokens, h_sample_ptr, h_span_ptr, h_span_lo, h_span_hi, ho,
                                 h_out, stream);
    if (rc != ODB_OK && c) {
        // whatever failed, no copy may still be running on the caller's host buffers when we return
        if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);
        if (c->d2h_stream) cudaStreamSynchronize(c->d2h_stream);
        cudaStreamSynchronize((cudaStream_t)stream);
        (void)cudaGetLastError();
    }
    return rc;
}

int odb_loss_weights(odb_ctx *c, int mode, double *d_weights, void *stream) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (mode != ODB_SCALE_SAMPLE && mode != ODB_SCALE_TOKEN_APPROX && mode != ODB_SCALE_TOKEN_EXACT)
        return ODB_ERR_INVALID_ARG;
    if (c->state != 5 || !c->collated) return ODB_ERR_STATE;
    if (c->info.n_slots > 0 && !d_weights) return ODB_ERR_INVALID_ARG;
    CU(c, cudaSetDevice(c->device));
    CU(c, launch_loss_weights(c, mode, d_weights, (cudaStream_t)stream));
    return ODB_OK;
}

int odb_loss_numerators(odb_ctx *c, int mode, double *d_num, void *stream) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (mode != ODB_SCALE_SAMPLE && mode != ODB_SCALE_TOKEN_APPROX && mode != ODB_SCALE_TOKEN_EXACT)
        return ODB_ERR_INVALID_ARG;
    if (c->state != 5 || !c->collated) return ODB_ERR_STATE;
    if (c->info.n_slots > 0 && !d_num) return ODB_ERR_INVALID_ARG;
    CU(c, cudaSetDevice(c->device));
    CU(c, launch_loss_numerators(c, mode, d_num, (cudaStream_t)stream));
    return ODB_OK;
}

int odb_loss_normalize(odb_ctx *c, const double *d_num_world, int32_t world_ranks, int32_t rank_offset, double *d_weights,
                       void *stream) {
    if (!c) return ODB_ERR_INVALID_ARG;
    if (c->state != 5 || !c->collated) return ODB_ERR_STATE;
    if (world_ranks < c->prm.n_ranks || rank_offset < 0 || rank_offset + c->prm.n_ranks > world_ranks)
        return ODB_ERR_INVALID_ARG;
    if (c->info.n_slots > 0 && (!d_num_world || !d_weights)) return ODB_ERR_INVALID_ARG;
    CU(c, cudaSetDevice(c->device));
    CU(c, launch_loss_normalize(c, d_num_world, world_ranks, rank_offset, d_weights, (cudaStream_t)stream));
    return ODB_OK;
}

int64_t odb_debug_read(odb_ctx *c, int what, void *h_dst, int64_t max_bytes) {
    if (!c || !h_dst) return -1;
    if (what == 5) {  // a host-side counter: no device access
        if (max_bytes < 8) return -1;
        const long long v = odb::g_table_allocs.load(std::memory_order_relaxed);
        memcpy(h_dst, &v, 8);
        return 8;
    }
    const void *src = nullptr;
    int64_t bytes = 0;
    const int R = c->prm.n_ranks;
    switch (what) {
    case 0: src = c->G; bytes = (int64_t)R * 4; break;
    case 1: src = c->S; bytes = (int64_t)R * 4; break;
    case 2: src = c->sorted; bytes = c->n_total * 8; break;
    case 3: src = c->emit_cur; bytes = (int64_t)R * 4; break;
    case 4: src = c->spec_used ? c->spec_tab.p : nullptr; bytes = 16; break;
    default: return -1;
    }
    if (!src) return -1;
    bytes = std::min(bytes, max_bytes);
    if (cudaSetDevice(c->device) != cudaSuccess) return -1;
    if (cudaDeviceSynchronize() != cudaSuccess) return -1;
    if (bytes > 0 && cudaMemcpy(h_dst, src, (size_t)bytes, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return bytes;
}

}  // extern "C"
