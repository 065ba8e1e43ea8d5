"""Thin ctypes binding of ``libodb.so`` (the C ABI declared in ``include/odb.h``).

Argument marshalling only: every step of the path (sort, grouping, alignment, collation) runs in
the CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams, nothing else.
There is NO CPU fallback: if the library is missing and cannot be built, importing the entry points
raises ``OdbLibraryError``; without a CUDA device ``odb_create`` raises ``OdbError(ODB_ERR_CUDA)``.

Function names and argument order follow ``include/odb.h`` one to one.  Tensor arguments may be
``torch.Tensor`` (device or host, as the header says), raw integer addresses, or ``None``.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

# ---- enums (include/odb.h) -------------------------------------------------------------------
ODB_OK, ODB_ERR_INVALID_ARG, ODB_ERR_BAD_LENGTH, ODB_ERR_CAPACITY, ODB_ERR_CUDA, ODB_ERR_STATE = range(6)
ODB_RULE_THRESHOLD, ODB_RULE_MAXFIT_ASC = 0, 1
ODB_STOP_ALL_FINISHED, ODB_STOP_LOGICAL, ODB_STOP_QUOTA = 0, 1, 2

_i32, _i64, _u8, _vp = ctypes.c_int32, ctypes.c_int64, ctypes.c_uint8, ctypes.c_void_p


class odb_params(ctypes.Structure):
    _fields_ = [("n_ranks", _i32), ("rule", _i32), ("join_mode", _i32), ("buffer_size", _i32),
                ("slot_capacity", _i32), ("pad_id", _i32), ("ignore_index", _i32), ("shift_labels", _i32),
                ("budget", _i64), ("sample_quota", _i64), ("emitted_so_far", _i64)]


class odb_plan_info(ctypes.Structure):
    _fields_ = [("n_rounds", _i32), ("n_steps", _i32), ("stop_reason", _i32), ("reserved", _i32),
                ("n_slots", _i64), ("total_elems", _i64), ("samples_emitted", _i64), ("samples_left", _i64),
                ("real_tokens", _i64), ("padded_elems", _i64)]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_ if k != "reserved"}


class odb_outputs(ctypes.Structure):
    _fields_ = [("d_input_ids", _vp), ("d_labels", _vp), ("d_position_ids", _vp), ("d_attention_mask", _vp),
                ("arena_capacity", _i64),
                ("d_grp_count", _vp), ("d_grp_width", _vp), ("d_grp_round", _vp), ("d_grp_valid_tokens", _vp),
                ("d_grp_real_tokens", _vp), ("d_grp_origin", _vp), ("d_grp_offset", _vp), ("d_grp_sample_ptr", _vp),
                ("slot_capacity_alloc", _i64),
                ("d_grp_sample_ids", _vp), ("ids_capacity", _i64),
                ("d_step_samples", _vp), ("d_step_valid_tokens", _vp), ("step_capacity_alloc", _i64),
                ("d_left_ptr", _vp), ("d_left_ids", _vp), ("left_capacity", _i64)]


class odb_dist_bufs(ctypes.Structure):
    _fields_ = [("d_summary_local", _vp), ("d_summary_world", _vp), ("summary_local_count", _i32),
                ("summary_world_count", _i32), ("d_step_samples_round", _vp), ("step_window", _i32),
                ("spec_G_count", _i32), ("d_spec_G_local", _vp)]


class odb_offline_params(ctypes.Structure):
    _fields_ = [("planner", _i32), ("size", _i32), ("batch_size", _i32), ("reserved", _i32), ("d_perm", _vp),
                ("d_shuffle_key", _vp)]


ODB_PLANNER_GMT, ODB_PLANNER_BMT, ODB_PLANNER_HFG = 0, 1, 2


class OdbLibraryError(RuntimeError):
    """libodb.so is missing / unloadable.  There is no fallback path."""


class OdbError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        msg = "%s: %s (status %d)" % (where, status_string(status), status)
        if cuda_error:
            msg += " [cudaError %d]" % cuda_error
        super().__init__(msg)


_lib = None

# every symbol include/odb.h declares: name -> (restype, argtypes)
_P = ctypes.POINTER
SYMBOLS = {
    "odb_create": (_i32, [_P(odb_params), _i32, _i64, _P(_vp)]),
    "odb_destroy": (_i32, [_vp]),
    "odb_reset": (_i32, [_vp]),
    "odb_form_groups": (_i32, [_vp, _vp, _P(_i64), _vp]),
    "odb_align": (_i32, [_vp, _vp]),
    "odb_set_available": (_i32, [_vp, _P(_i64), _vp]),
    "odb_round_status": (_i32, [_vp, _P(_i32), _P(_i32)]),
    "odb_plan_query": (_i32, [_vp, _P(odb_plan_info)]),
    "odb_collate": (_i32, [_vp, _vp, _vp, _vp, _vp, _vp, _P(odb_outputs), _vp]),
    "odb_run": (_i32, [_vp, _vp, _P(_i64), _vp, _vp, _vp, _vp, _vp, _P(odb_outputs), _P(odb_plan_info), _vp]),
    "odb_plan": (_i32, [_vp, _vp, _P(_i64), _P(odb_plan_info), _vp]),
    "odb_collate_steps": (_i32, [_vp, _i32, _i32, _vp, _vp, _vp, _vp, _vp, _P(odb_outputs), _P(odb_plan_info), _vp]),
    "odb_run_host": (_i32, [_vp, _vp, _P(_i64), _vp, _vp, _vp, _vp, _vp, _P(odb_outputs), _P(odb_plan_info), _vp]),
    "odb_loss_weights": (_i32, [_vp, _i32, _vp, _vp]),
    "odb_loss_numerators": (_i32, [_vp, _i32, _vp, _vp]),
    "odb_loss_normalize": (_i32, [_vp, _vp, _i32, _i32, _vp, _vp]),
    "odb_dist_config": (_i32, [_vp, _i32, _i32, _i32]),
    "odb_dist_spec_form": (_i32, [_vp, _vp, _P(_i64), _i32, _i64, _vp]),
    "odb_dist_spec_commit": (_i32, [_vp, _vp, _vp, _i32, _vp]),
    "odb_dist_spec_status": (_i32, [_vp, _P(_i32), _P(_i32), _P(_i32), _i32, _P(_i32)]),
    "odb_dist_buffers": (_i32, [_vp, _P(odb_dist_bufs)]),
    "odb_commit": (_i32, [_vp, _vp]),
    "odb_emitted_counts": (_i32, [_vp, _P(_i64)]),
    "odb_fetch_quota": (_i32, [_P(odb_params), _P(_i64), _i32, _i32, _P(_i64), _P(_i64)]),
    "odb_set_timing": (_i32, [_vp, _i32]),
    "odb_get_timing": (_i32, [_vp, _P(ctypes.c_float)]),
    "odb_get_timing_at": (_i32, [_vp, _i32, _P(ctypes.c_float)]),
    "odb_offline_plan": (_i32, [_vp, _P(odb_offline_params), _vp, _i64, _vp]),
    "odb_slot_offsets_static": (_i32, [_vp, _vp, _i64, _vp, _vp]),
    "odb_static_max_slots": (_i64, []),
    "odb_static_last_cuda_error": (_i32, []),
    "odb_set_option": (_i32, [_vp, _i32, _i64]),
    "odb_probe_bandwidth": (_i32, [_i32, _vp, _vp, _vp, _vp, _vp, _i64, _i32, _vp, _P(ctypes.c_float)]),
    "odb_kernel_launches": (_i64, [_vp]),
    "odb_debug_read": (_i64, [_vp, _i32, _vp, _i64]),
    "odb_synth_tokens": (_i32, [_vp, _i64, _i64, ctypes.c_uint64, _i32, _vp]),
    "odb_last_cuda_error": (_i32, [_vp]),
    "odb_status_string": (ctypes.c_char_p, [_i32]),
}


def library_path() -> str:
    return _build.LIB


def load():
    """Load libodb.so (building it in-tree with nvcc when the sources are newer).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        if _build.needs_build():
            _build.build()
    except Exception as e:  # no nvcc on this machine, or a compile error
        if not os.path.exists(_build.LIB):
            raise OdbLibraryError("libodb.so is not built and building it failed: %r" % (e,)) from e
    try:
        L = ctypes.CDLL(_build.LIB)
    except OSError as e:
        raise OdbLibraryError("cannot load %s: %s" % (_build.LIB, e)) from e
    for name, (res, args) in SYMBOLS.items():
        try:
            fn = getattr(L, name)
        except AttributeError as e:
            raise OdbLibraryError("%s does not export %s" % (_build.LIB, name)) from e
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


# ---- marshalling helpers ---------------------------------------------------------------------
def _ptr(x) -> Optional[int]:
    """Address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x or None
    if isinstance(x, np.ndarray):
        return x.ctypes.data or None
    dp = getattr(x, "data_ptr", None)
    if dp is not None:
        return dp() or None
    raise TypeError("cannot take the address of %r" % type(x))


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream or None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


def _host_i64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int64)


def _check(rc: int, where: str, ctx=None):
    if rc != ODB_OK:
        ce = load().odb_last_cuda_error(ctx) if ctx else 0
        raise OdbError(rc, where, ce)


def status_string(status: int) -> str:
    return load().odb_status_string(int(status)).decode()


def make_params(n_ranks: int, budget: int, *, rule=ODB_RULE_THRESHOLD, join_mode=1, sample_quota=0,
                emitted_so_far=0, buffer_size=0, slot_capacity=0, pad_id=0, ignore_index=-100,
                shift_labels=1) -> odb_params:
    return odb_params(n_ranks=n_ranks, rule=rule, join_mode=join_mode, buffer_size=buffer_size,
                      slot_capacity=slot_capacity, pad_id=pad_id, ignore_index=ignore_index,
                      shift_labels=shift_labels, budget=budget, sample_quota=sample_quota,
                      emitted_so_far=emitted_so_far)


# ---- the C ABI, one Python function per entry point ------------------------------------------
def odb_create(params: odb_params, device: int, max_samples_total: int) -> int:
    h = _vp()
    _check(load().odb_create(ctypes.byref(params), int(device), int(max_samples_total), ctypes.byref(h)), "odb_create")
    return h.value


def odb_destroy(ctx: int) -> None:
    _check(load().odb_destroy(ctx), "odb_destroy")


def odb_reset(ctx: int) -> None:
    _check(load().odb_reset(ctx), "odb_reset", ctx)


def odb_form_groups(ctx: int, d_lengths, h_rank_ptr, stream=None) -> None:
    rp = _host_i64(h_rank_ptr)
    _check(load().odb_form_groups(ctx, _ptr(d_lengths), rp.ctypes.data_as(_P(_i64)), _stream(stream)),
           "odb_form_groups", ctx)


def odb_set_available(ctx: int, h_arrived, stream=None) -> None:
    """Views of each rank's stream that have arrived so far (None = everything)."""
    if h_arrived is None:
        rc = load().odb_set_available(ctx, None, _stream(stream))
    else:
        a = _host_i64(h_arrived)
        rc = load().odb_set_available(ctx, a.ctypes.data_as(_P(_i64)), _stream(stream))
    _check(rc, "odb_set_available", ctx)


def odb_emitted_counts(ctx: int, n_ranks: int) -> np.ndarray:
    """Views of each rank's stream emitted so far (int64[n_ranks]); between rounds only (include/odb.h)."""
    out = np.zeros(int(n_ranks), dtype=np.int64)
    _check(load().odb_emitted_counts(ctx, out.ctypes.data_as(_P(_i64))), "odb_emitted_counts", ctx)
    return out


def odb_fetch_quota(params: odb_params, h_rank_ptr, prefetch_factor: int, num_workers: int, h_emitted) -> np.ndarray:
    """How far into each rank's stream the workers may have fetched under the outstanding-depth envelope
    D = max(prefetch_factor * num_workers, buffer_size) (App. P): int64[n_ranks], computed by the library
    (host arithmetic: no context, no device)."""
    rp, em = _host_i64(h_rank_ptr), _host_i64(h_emitted)
    if len(em) != int(params.n_ranks) or len(rp) != len(em) + 1:
        raise ValueError("h_emitted needs n_ranks entries, h_rank_ptr n_ranks + 1")
    out = np.zeros(len(em), dtype=np.int64)
    rc = load().odb_fetch_quota(ctypes.byref(params), rp.ctypes.data_as(_P(_i64)), int(prefetch_factor), int(num_workers),
                                em.ctypes.data_as(_P(_i64)), out.ctypes.data_as(_P(_i64)))
    _check(rc, "odb_fetch_quota")
    return out


def odb_align(ctx: int, stream=None) -> None:
    _check(load().odb_align(ctx, _stream(stream)), "odb_align", ctx)


def odb_round_status(ctx: int):
    """Returns (done, T_grp)."""
    done, T = _i32(0), _i32(0)
    _check(load().odb_round_status(ctx, ctypes.byref(done), ctypes.byref(T)), "odb_round_status", ctx)
    return int(done.value), int(T.value)


def odb_plan_query(ctx: int) -> odb_plan_info:
    info = odb_plan_info()
    _check(load().odb_plan_query(ctx, ctypes.byref(info)), "odb_plan_query", ctx)
    return info


def odb_collate(ctx: int, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, out: odb_outputs,
                stream=None) -> None:
    _check(load().odb_collate(ctx, _ptr(d_tokens), _ptr(d_sample_ptr), _ptr(d_span_ptr), _ptr(d_span_lo),
                              _ptr(d_span_hi), ctypes.byref(out), _stream(stream)), "odb_collate", ctx)


def odb_run(ctx: int, d_lengths, h_rank_ptr, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi,
            out: odb_outputs, stream=None, *, allow_capacity_error: bool = False) -> odb_plan_info:
    """Whole path.  With ``allow_capacity_error`` an ODB_ERR_CAPACITY is not raised: the returned
    info (with ``.status`` set) tells the caller how much to allocate."""
    rp = _host_i64(h_rank_ptr)
    info = odb_plan_info()
    rc = load().odb_run(ctx, _ptr(d_lengths), rp.ctypes.data_as(_P(_i64)), _ptr(d_tokens), _ptr(d_sample_ptr),
                        _ptr(d_span_ptr), _ptr(d_span_lo), _ptr(d_span_hi), ctypes.byref(out), ctypes.byref(info),
                        _stream(stream))
    info.status = rc
    if rc == ODB_ERR_CAPACITY and allow_capacity_error:
        return info
    _check(rc, "odb_run", ctx)
    return info


def odb_plan(ctx: int, d_lengths, h_rank_ptr, stream=None) -> odb_plan_info:
    """The whole plan (every protocol round + the slot scan), no collation."""
    rp = _host_i64(h_rank_ptr)
    info = odb_plan_info()
    _check(load().odb_plan(ctx, _ptr(d_lengths), rp.ctypes.data_as(_P(_i64)), ctypes.byref(info), _stream(stream)),
           "odb_plan", ctx)
    info.status = ODB_OK
    return info


def odb_collate_steps(ctx: int, step_lo: int, step_hi: int, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi,
                      out: odb_outputs, stream=None, *, allow_capacity_error: bool = False) -> odb_plan_info:
    """Steps [step_lo, step_hi) of the plan so far as a self-contained plan in ``out`` (include/odb.h)."""
    info = odb_plan_info()
    rc = load().odb_collate_steps(ctx, int(step_lo), int(step_hi), _ptr(d_tokens), _ptr(d_sample_ptr), _ptr(d_span_ptr),
                                  _ptr(d_span_lo), _ptr(d_span_hi), ctypes.byref(out), ctypes.byref(info),
                                  _stream(stream))
    info.status = rc
    if rc == ODB_ERR_CAPACITY and allow_capacity_error:
        return info
    _check(rc, "odb_collate_steps", ctx)
    return info


def odb_run_host(ctx: int, h_lengths, h_rank_ptr, h_tokens, h_sample_ptr, h_span_ptr, h_span_lo, h_span_hi,
                 h_out: odb_outputs, stream=None, *, allow_capacity_error: bool = False) -> odb_plan_info:
    rp = _host_i64(h_rank_ptr)
    info = odb_plan_info()
    rc = load().odb_run_host(ctx, _ptr(h_lengths), rp.ctypes.data_as(_P(_i64)), _ptr(h_tokens), _ptr(h_sample_ptr),
                             _ptr(h_span_ptr), _ptr(h_span_lo), _ptr(h_span_hi), ctypes.byref(h_out),
                             ctypes.byref(info), _stream(stream))
    info.status = rc
    if rc == ODB_ERR_CAPACITY and allow_capacity_error:
        return info
    _check(rc, "odb_run_host", ctx)
    return info


ODB_SCALE_SAMPLE, ODB_SCALE_TOKEN_APPROX, ODB_SCALE_TOKEN_EXACT = 1, 2, 3


def odb_loss_weights(ctx: int, mode: int, d_weights, stream=None) -> None:
    """w[r * n_steps + k] (fp64, device) of loss-scaling ``mode`` for the plan last collated on ``ctx``."""
    _check(load().odb_loss_weights(ctx, int(mode), _ptr(d_weights), _stream(stream)), "odb_loss_weights", ctx)


def odb_loss_numerators(ctx: int, mode: int, d_num, stream=None) -> None:
    _check(load().odb_loss_numerators(ctx, int(mode), _ptr(d_num), _stream(stream)), "odb_loss_numerators", ctx)


def odb_loss_normalize(ctx: int, d_num_world, world_ranks: int, rank_offset: int, d_weights, stream=None) -> None:
    _check(load().odb_loss_normalize(ctx, _ptr(d_num_world), int(world_ranks), int(rank_offset), _ptr(d_weights),
                                     _stream(stream)), "odb_loss_normalize", ctx)


def odb_dist_config(ctx: int, world_ranks: int, rank_offset: int, world_max_window: int) -> None:
    _check(load().odb_dist_config(ctx, int(world_ranks), int(rank_offset), int(world_max_window)), "odb_dist_config", ctx)


def odb_dist_buffers(ctx: int) -> odb_dist_bufs:
    b = odb_dist_bufs()
    _check(load().odb_dist_buffers(ctx, ctypes.byref(b)), "odb_dist_buffers", ctx)
    return b


def odb_dist_spec_form(ctx: int, d_lengths, h_rank_ptr, n_rounds: int, world_max_stream: int, stream=None) -> None:
    rp = _host_i64(h_rank_ptr)
    _check(load().odb_dist_spec_form(ctx, _ptr(d_lengths), rp.ctypes.data_as(_P(_i64)), int(n_rounds), int(world_max_stream),
                                     _stream(stream)), "odb_dist_spec_form", ctx)


def odb_dist_spec_commit(ctx: int, d_G_world, d_n_world, n_procs: int, stream=None) -> None:
    _check(load().odb_dist_spec_commit(ctx, _ptr(d_G_world), _ptr(d_n_world), int(n_procs), _stream(stream)),
           "odb_dist_spec_commit", ctx)


def odb_dist_spec_status(ctx: int, max_rounds: int):
    """(rounds committed, their steps, [T_grp of each], done)."""
    r, k, d = _i32(0), _i32(0), _i32(0)
    T = (ctypes.c_int32 * max(int(max_rounds), 1))()
    _check(load().odb_dist_spec_status(ctx, ctypes.byref(r), ctypes.byref(k), T, int(max_rounds), ctypes.byref(d)),
           "odb_dist_spec_status", ctx)
    return int(r.value), int(k.value), [int(T[j]) for j in range(r.value)], int(d.value)


def odb_commit(ctx: int, stream=None) -> None:
    _check(load().odb_commit(ctx, _stream(stream)), "odb_commit", ctx)


def odb_set_timing(ctx: int, enable: bool) -> None:
    _check(load().odb_set_timing(ctx, 1 if enable else 0), "odb_set_timing", ctx)


def odb_get_timing(ctx: int):
    """(planning ms, collate-kernel ms, post ms) of the last odb_run / odb_collate."""
    ms = (ctypes.c_float * 3)()
    _check(load().odb_get_timing(ctx, ms), "odb_get_timing", ctx)
    return float(ms[0]), float(ms[1]), float(ms[2])


def odb_get_timing_at(ctx: int, back: int):
    """The same for the timed run ``back`` runs before the latest one (the last 64 runs are kept)."""
    ms = (ctypes.c_float * 3)()
    _check(load().odb_get_timing_at(ctx, int(back), ms), "odb_get_timing_at", ctx)
    return float(ms[0]), float(ms[1]), float(ms[2])


def odb_offline_plan(ctx: int, planner: int, d_lengths, n_samples: int, *, d_perm=None, d_shuffle_key=None, size: int = 0,
                     batch_size: int = 0, stream=None) -> None:
    """Plan with one of the paper's offline comparators (GMT / BMT / HFG; include/odb.h); then odb_plan_query /
    odb_collate as usual.  The caller keeps d_perm / d_shuffle_key alive until the collate call."""
    prm = odb_offline_params(planner=int(planner), size=int(size), batch_size=int(batch_size), reserved=0,
                             d_perm=_ptr(d_perm), d_shuffle_key=_ptr(d_shuffle_key))
    _check(load().odb_offline_plan(ctx, ctypes.byref(prm), _ptr(d_lengths), int(n_samples), _stream(stream)),
           "odb_offline_plan", ctx)


ODB_OPT_COLLATE_BULK_STORES = 1
ODB_OPT_HOST_STAGING_ELEMS = 2
ODB_OPT_ROUND_PARALLEL = 3
ODB_OPT_HOST_DEVICE_ARENAS = 4


def odb_set_option(ctx: int, option: int, value: int) -> None:
    _check(load().odb_set_option(ctx, int(option), int(value)), "odb_set_option", ctx)


def odb_static_max_slots() -> int:
    """Largest ``n_slots`` ``odb_slot_offsets_static`` accepts (ODB_STATIC_MAX_SLOTS)."""
    return int(load().odb_static_max_slots())


def odb_slot_offsets_static(d_grp_count, d_grp_width, n_slots: int, d_grp_offset, stream=None) -> None:
    """The plan's output offsets without a context and without any device allocation, for callers that are not
    allowed to allocate on the GPU they run on (a loader living inside a trainer that owns all of HBM; code in the
    middle of a step, where cudaMalloc / cudaFree stall the device).  ``d_grp_offset[s]`` (int64, ``n_slots + 1``
    entries) = sum over s' < s of round_up(count * width, 16).  The tile records of the scan live in a fixed array
    inside libodb.so, shared by every call on the device: keep calls on one stream (or order them), make the first
    call on a device outside stream capture, and stay within ``odb_static_max_slots()`` -- beyond it the call raises
    ``OdbError(ODB_ERR_CAPACITY)`` and touches nothing.  Details: include/odb.h."""
    L = load()
    rc = L.odb_slot_offsets_static(_ptr(d_grp_count), _ptr(d_grp_width), int(n_slots), _ptr(d_grp_offset),
                                   _stream(stream))
    if rc == ODB_ERR_CAPACITY:
        raise OdbError(rc, "odb_slot_offsets_static: n_slots %d is above the fixed scratch's limit of %d slots"
                       % (int(n_slots), int(L.odb_static_max_slots())))
    if rc != ODB_OK:
        raise OdbError(rc, "odb_slot_offsets_static", L.odb_static_last_cuda_error() if rc == ODB_ERR_CUDA else 0)


def odb_probe_bandwidth(kind: int, d_in, d_out0, d_out1, d_out2, d_out3, n_elems: int, reps: int = 5, stream=None) -> float:
    """Average milliseconds per launch of bandwidth probe ``kind`` (include/odb.h)."""
    ms = ctypes.c_float(0.0)
    _check(load().odb_probe_bandwidth(int(kind), _ptr(d_in), _ptr(d_out0), _ptr(d_out1), _ptr(d_out2), _ptr(d_out3),
                                      int(n_elems), int(reps), _stream(stream), ctypes.byref(ms)), "odb_probe_bandwidth")
    return float(ms.value)


def odb_kernel_launches(ctx: int) -> int:
    return int(load().odb_kernel_launches(ctx))


def odb_debug_read(ctx: int, what: int, dst: np.ndarray) -> int:
    return int(load().odb_debug_read(ctx, what, dst.ctypes.data, dst.nbytes))


def odb_synth_tokens(d_tokens, start: int, count: int, seed: int, vocab: int, stream=None) -> None:
    _check(load().odb_synth_tokens(_ptr(d_tokens), int(start), int(count), int(seed), int(vocab), _stream(stream)),
           "odb_synth_tokens")


def odb_last_cuda_error(ctx: int) -> int:
    return int(load().odb_last_cuda_error(ctx))


odb_status_string = status_string


# ---- memory plumbing (torch allocations only; no arithmetic) ---------------------------------
_TABLES = (  # name, torch dtype name, size key
    ("grp_count", "int32", "slots"), ("grp_width", "int32", "slots"), ("grp_round", "int32", "slots"),
    ("grp_valid_tokens", "int32", "slots"), ("grp_real_tokens", "int32", "slots"), ("grp_origin", "int32", "slots"),
    ("grp_offset", "int64", "slots"),
    ("grp_sample_ptr", "int64", "slots1"), ("grp_sample_ids", "int32", "ids"),
    ("step_samples", "int32", "steps"), ("step_valid_tokens", "int64", "steps"),
    ("left_ptr", "int64", "ranks1"), ("left_ids", "int32", "left"),
)


class OutputBuffers:
    """Caller-owned output arenas and tables (torch tensors) plus the ``odb_outputs`` view of them.

    ``device`` = a CUDA device for odb_run / odb_collate, or ``"cpu"`` (pinned) for odb_run_host.
    ``fill`` pre-fills the four arenas with a byte pattern (tests prove no stray writes with it).
    """

    def __init__(self, n_ranks: int, total_elems: int, n_slots: int, samples_emitted: int, n_steps: int,
                 samples_left: int, device, *, pinned: bool = True, fill: Optional[int] = None, tables: bool = True):
        import torch
        host = str(device) == "cpu"
        kw = dict(device="cpu", pin_memory=pinned) if host else dict(device=device)
        E = int(total_elems)
        cap = E + 16

        def arena(dt):
            t = torch.empty(cap, dtype=dt, **kw)
            if fill is not None:
                t.view(torch.uint8).fill_(fill)
            return t

        self.input_ids = arena(torch.int32)
        self.labels = arena(torch.int32)
        self.position_ids = arena(torch.int32)
        self.attention_mask = arena(torch.uint8)
        sizes = dict(slots=int(n_slots), slots1=int(n_slots) + 1, ids=int(samples_emitted), steps=int(n_steps),
                     ranks1=int(n_ranks) + 1, left=int(samples_left))
        self.sizes = sizes
        s = odb_outputs()
        s.d_input_ids, s.d_labels = _ptr(self.input_ids), _ptr(self.labels)
        s.d_position_ids, s.d_attention_mask = _ptr(self.position_ids), _ptr(self.attention_mask)
        s.arena_capacity = E
        if tables:
            for name, dt, key in _TABLES:
                t = torch.zeros(max(sizes[key], 1), dtype=getattr(torch, dt), **kw)
                setattr(self, name, t)
                setattr(s, "d_" + name, _ptr(t))
        s.slot_capacity_alloc = sizes["slots"]
        s.ids_capacity = sizes["ids"]
        s.step_capacity_alloc = sizes["steps"]
        s.left_capacity = sizes["left"]
        self.struct = s
        self.total_elems = E

    @classmethod
    def for_plan(cls, n_ranks: int, info: odb_plan_info, device, **kw) -> "OutputBuffers":
        return cls(n_ranks, info.total_elems, info.n_slots, info.samples_emitted, info.n_steps, info.samples_left,
                   device, **kw)

    def table(self, name: str):
        """Table trimmed to its logical size."""
        key = dict((n, k) for n, _, k in _TABLES)[name]
        return getattr(self, name)[: self.sizes[key]]

    def nbytes_arenas(self) -> int:
        return self.total_elems * 13


class Odb:
    """Context holder: ``with Odb(params, max_samples) as ctx: ...`` (handle in ``.h``)."""

    def __init__(self, params: odb_params, max_samples_total: int, device: int = 0):
        self.params = params
        self.h = odb_create(params, device, max_samples_total)

    def close(self):
        if self.h:
            odb_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def plan(self, d_lengths, h_rank_ptr, stream=None, avail_schedule=None) -> odb_plan_info:
        """The round loop (odb_form_groups / odb_align / odb_round_status until done) + odb_plan_query.
        ``avail_schedule[j][r]`` (optional) = views of rank r that have arrived by round j; after the
        schedule everything has (odb_set_available)."""
        odb_reset(self.h)
        done = 0
        self.round_T = []
        j = 0
        while not done:
            if avail_schedule is not None:
                odb_set_available(self.h, avail_schedule[j] if j < len(avail_schedule) else None, stream)
                j += 1
            odb_form_groups(self.h, d_lengths, h_rank_ptr, stream)
            odb_align(self.h, stream)
            done, T = odb_round_status(self.h)
            if T > 0:
                self.round_T.append(T)
        return odb_plan_query(self.h)
