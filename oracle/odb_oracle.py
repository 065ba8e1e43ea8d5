"""ctypes front end of the CPU oracle (``odb_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this module.  It shares
nothing with ``paper_2606_19989_b200`` (the CUDA path) and never imports it.

The arithmetic lives in the C file; this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "odb_oracle.c")
_LIB = os.path.join(_HERE, "libodb_oracle.so")

RULE_THRESHOLD = 0
RULE_MAXFIT_ASC = 1
STOP_ALL_FINISHED = 0
STOP_LOGICAL = 1
STOP_QUOTA = 2


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, single-threaded).  Returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-std=c99", "-shared", "-fPIC", "-Wall", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _p(a: Optional[np.ndarray], ctype):
    if a is None:
        return ctypes.POINTER(ctype)()
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i32, i64 = ctypes.c_int32, ctypes.c_int64
        pi32, pi64, pu8 = ctypes.POINTER(i32), ctypes.POINTER(i64), ctypes.POINTER(ctypes.c_uint8)
        vp = ctypes.c_void_p
        L.oracle_group_window.restype = i64
        L.oracle_group_window.argtypes = [i32, i64, pi32, pi32, i32, pi32, pi64]
        L.oracle_align_list.restype = i64
        L.oracle_align_list.argtypes = [pi32, pi64, i64, i64, pi32, pi64, pi32, pi64]
        L.oracle_target_groups.restype = i64
        L.oracle_target_groups.argtypes = [pi64, pi64, i32, i64]
        L.oracle_target_group_size.restype = i64
        L.oracle_target_group_size.argtypes = [i64, i64]
        L.oracle_plan_run.restype = vp
        L.oracle_plan_run.argtypes = [i32, i64, i32, i32, i64, i64, i32, i32, pi32, pi64, pi32]
        L.oracle_plan_run_sched.restype = vp
        L.oracle_plan_run_sched.argtypes = [i32, i64, i32, i32, i64, i64, i32, i32, pi32, pi64, pi64, i32, pi32]
        L.oracle_offline_plan.restype = vp
        L.oracle_offline_plan.argtypes = [i32, i32, i64, pi32, i64, pi32, pi32, i32, i32, pi32]
        L.oracle_plan_free.restype = None
        L.oracle_plan_free.argtypes = [vp]
        L.oracle_plan_scalar.restype = i64
        L.oracle_plan_scalar.argtypes = [vp, i32]
        L.oracle_plan_tables.restype = None
        L.oracle_plan_tables.argtypes = [vp, pi32, pi32, pi32, pi64, pi32, pi64, pi32, pi32, pi64, pi32, pi32]
        L.oracle_collate_slot.restype = i64
        L.oracle_collate_slot.argtypes = [vp, i64, pi32, pi64, pi64, pi32, pi32, i32, i32, i32, pi32, pu8, pi32, pi32]
        L.oracle_collate_all.restype = None
        L.oracle_collate_all.argtypes = [vp, pi32, pi64, pi64, pi32, pi32, i32, i32, i32, pi32, pu8, pi32, pi32,
                                         pi32, pi64]
        L.oracle_collate_range.restype = None
        L.oracle_collate_range.argtypes = [vp, i64, i64, i64, pi32, pi64, pi64, pi32, pi32, i32, i32, i32, pi32, pu8,
                                           pi32, pi32, pi32]
        L.oracle_plan_origin.restype = None
        L.oracle_plan_origin.argtypes = [vp, pi32]
        L.oracle_loss_weights.restype = None
        L.oracle_loss_weights.argtypes = [i32, i32, i64, pi32, pi32, pi32, ctypes.POINTER(ctypes.c_double)]
        _lib = L
    return _lib


# ---------------------------------------------------------------------------------------
# pieces, exposed so that each can be pinned on its own
# ---------------------------------------------------------------------------------------
def group_window(rule: int, budget: int, lengths, ids=None):
    """Group one window.  Returns a list of groups (lists of local ids), list order short->long."""
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    if ids is None:
        ids = np.arange(len(lengths), dtype=np.int32)
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    S = len(ids)
    order = np.zeros(max(S, 1), dtype=np.int32)
    gptr = np.zeros(S + 1, dtype=np.int64)
    G = lib().oracle_group_window(rule, budget, _p(lengths, ctypes.c_int32), _p(ids, ctypes.c_int32), S,
                                  _p(order, ctypes.c_int32), _p(gptr, ctypes.c_int64))
    return [order[gptr[j]:gptr[j + 1]].tolist() for j in range(G)]


def align_list(groups, T: int):
    """Alg. 1 on one rank's candidate list.  Returns (aligned groups, samples returned to the buffer)."""
    rows = np.ascontiguousarray([x for g in groups for x in g], dtype=np.int32)
    gptr = np.zeros(len(groups) + 1, dtype=np.int64)
    for j, g in enumerate(groups):
        gptr[j + 1] = gptr[j] + len(g)
    n = max(len(rows), 1)
    rows_out = np.zeros(n, dtype=np.int32)
    gptr_out = np.zeros(max(len(groups), T, len(rows)) + 2, dtype=np.int64)
    back = np.zeros(n, dtype=np.int32)
    n_back = ctypes.c_int64(0)
    rows_in = rows if len(rows) else np.zeros(1, dtype=np.int32)
    G = lib().oracle_align_list(_p(rows_in, ctypes.c_int32), _p(gptr, ctypes.c_int64), len(groups), T,
                                _p(rows_out, ctypes.c_int32), _p(gptr_out, ctypes.c_int64),
                                _p(back, ctypes.c_int32), ctypes.byref(n_back))
    out = [rows_out[gptr_out[j]:gptr_out[j + 1]].tolist() for j in range(G)]
    return out, back[:n_back.value].tolist()


def target_groups(G, S, C: int) -> int:
    G = np.ascontiguousarray(G, dtype=np.int64)
    S = np.ascontiguousarray(S, dtype=np.int64)
    return int(lib().oracle_target_groups(_p(G, ctypes.c_int64), _p(S, ctypes.c_int64), len(G), C))


def target_group_size(budget: int, l: int) -> int:
    """Eq. 1: B(l) = max(floor(L_max / l), 1)."""
    return int(lib().oracle_target_group_size(int(budget), int(l)))


SCALE_SAMPLE = 1
SCALE_TOKEN_APPROX = 2
SCALE_TOKEN_EXACT = 3


def loss_weights(mode: int, R: int, n_steps: int, count, valid, origin) -> np.ndarray:
    """w[r, k] (fp64) of the three loss-scaling modes; tables are rank-major."""
    count = np.ascontiguousarray(count, dtype=np.int32)
    valid = np.ascontiguousarray(valid, dtype=np.int32)
    origin = np.ascontiguousarray(origin, dtype=np.int32)
    w = np.zeros(max(R * n_steps, 1), dtype=np.float64)
    lib().oracle_loss_weights(int(mode), int(R), int(n_steps), _p(count, ctypes.c_int32), _p(valid, ctypes.c_int32),
                              _p(origin, ctypes.c_int32), w.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return w[:R * n_steps].reshape(R, n_steps)


# ---------------------------------------------------------------------------------------
# whole plan / collation
# ---------------------------------------------------------------------------------------
class OraclePlan:
    """Result of the round loop (grouping + alignment) for R ranks; owns the C object."""

    def __init__(self, lengths, rank_ptr, *, budget, rule=0, join_mode=1, sample_quota=0, emitted_so_far=0,
                 buffer_size=0, slot_capacity=0, avail_schedule=None, **_ignored):
        self.lengths = np.ascontiguousarray(lengths, dtype=np.int32)
        self.rank_ptr = np.ascontiguousarray(rank_ptr, dtype=np.int64)
        self.R = len(self.rank_ptr) - 1
        err = ctypes.c_int32(0)
        lens = self.lengths if len(self.lengths) else np.zeros(1, dtype=np.int32)
        if avail_schedule is None:
            self._h = lib().oracle_plan_run(self.R, int(budget), int(rule), int(join_mode), int(sample_quota),
                                            int(emitted_so_far), int(buffer_size), int(slot_capacity),
                                            _p(lens, ctypes.c_int32), _p(self.rank_ptr, ctypes.c_int64),
                                            ctypes.byref(err))
        else:  # [n_sched, R]: views of each rank that have arrived by round j (see oracle_plan_run_sched)
            sched = np.ascontiguousarray(avail_schedule, dtype=np.int64).reshape(-1, self.R)
            sp = sched if sched.size else np.zeros(1, np.int64)
            self._h = lib().oracle_plan_run_sched(self.R, int(budget), int(rule), int(join_mode), int(sample_quota),
                                                  int(emitted_so_far), int(buffer_size), int(slot_capacity),
                                                  _p(lens, ctypes.c_int32), _p(self.rank_ptr, ctypes.c_int64),
                                                  _p(sp, ctypes.c_int64), int(sched.shape[0]), ctypes.byref(err))
        self.err = err.value
        self._load()

    PLANNER_GMT, PLANNER_BMT, PLANNER_HFG = 0, 1, 2

    @classmethod
    def offline(cls, planner: int, lengths, n_ranks: int, *, budget: int = 1, perm=None, shuffle_key=None, size: int = 0,
                batch_size: int = 0) -> "OraclePlan":
        """The paper's offline comparators as planners (App. I; App. J): GMT (0), BMT (1), HFG (2) over a
        GLOBAL length array; slot ids are global sample ids.  ``perm`` / ``shuffle_key``: the random draws, as inputs."""
        self = cls.__new__(cls)
        self.lengths = np.ascontiguousarray(lengths, dtype=np.int32)
        self.R = int(n_ranks)
        self.rank_ptr = np.zeros(self.R + 1, dtype=np.int64)
        err = ctypes.c_int32(0)
        lens = self.lengths if len(self.lengths) else np.zeros(1, dtype=np.int32)
        pm = None if perm is None else np.ascontiguousarray(perm, dtype=np.int32)
        sk = None if shuffle_key is None else np.ascontiguousarray(shuffle_key, dtype=np.int32)
        self._h = lib().oracle_offline_plan(int(planner), self.R, int(budget), _p(lens, ctypes.c_int32), len(self.lengths),
                                            _p(pm, ctypes.c_int32), _p(sk, ctypes.c_int32), int(size), int(batch_size),
                                            ctypes.byref(err))
        self.err = err.value
        self._load()
        return self

    def _load(self):
        if not self._h:
            raise ValueError("the oracle planner failed with status %d" % self.err)
        if self.err:
            raise AssertionError("oracle: ranks hold different slot counts")
        sc = lambda w: int(lib().oracle_plan_scalar(self._h, w))
        self.n_rounds, self.n_steps, self.stop_reason = sc(0), sc(1), sc(2)
        self.n_slots, self.total_elems = sc(3), sc(4)
        self.samples_emitted, self.samples_left = sc(5), sc(6)
        self.real_tokens, self.padded_elems = sc(7), sc(8)
        n_emit_rounds = sc(9)
        ns = max(self.n_slots, 1)
        self.grp_count = np.zeros(ns, np.int32)
        self.grp_width = np.zeros(ns, np.int32)
        self.grp_round = np.zeros(ns, np.int32)
        self.grp_offset = np.zeros(ns, np.int64)
        self.grp_real_tokens = np.zeros(ns, np.int32)
        self.grp_sample_ptr = np.zeros(self.n_slots + 1, np.int64)
        self.grp_sample_ids = np.zeros(max(self.samples_emitted, 1), np.int32)
        self.step_samples = np.zeros(max(self.n_steps, 1), np.int32)
        self.left_ptr = np.zeros(self.R + 1, np.int64)
        self.left_ids = np.zeros(max(self.samples_left, 1), np.int32)
        self.round_T = np.zeros(max(n_emit_rounds, 1), np.int32)
        self.grp_origin = np.zeros(ns, np.int32)
        lib().oracle_plan_origin(self._h, _p(self.grp_origin, ctypes.c_int32))
        i32, i64 = ctypes.c_int32, ctypes.c_int64
        lib().oracle_plan_tables(self._h, _p(self.grp_count, i32), _p(self.grp_width, i32), _p(self.grp_round, i32),
                                 _p(self.grp_offset, i64), _p(self.grp_real_tokens, i32),
                                 _p(self.grp_sample_ptr, i64), _p(self.grp_sample_ids, i32),
                                 _p(self.step_samples, i32), _p(self.left_ptr, i64), _p(self.left_ids, i32),
                                 _p(self.round_T, i32))
        for name in ("grp_count", "grp_width", "grp_round", "grp_offset", "grp_real_tokens", "grp_origin"):
            setattr(self, name, getattr(self, name)[:self.n_slots])
        self.grp_sample_ids = self.grp_sample_ids[:self.samples_emitted]
        self.step_samples = self.step_samples[:self.n_steps]
        self.left_ids = self.left_ids[:self.samples_left]
        self.round_T = self.round_T[:n_emit_rounds]

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            try:
                lib().oracle_plan_free(h)
            except Exception:  # interpreter shutdown: module globals are already gone
                pass
            self._h = None

    def slot_ids(self, r: int, k: int):
        s = r * self.n_steps + k
        return self.grp_sample_ids[self.grp_sample_ptr[s]:self.grp_sample_ptr[s + 1]]

    def groups_of_rank(self, r: int):
        return [self.slot_ids(r, k).tolist() for k in range(self.n_steps)]

    # -- collation ---------------------------------------------------------------------
    def collate_slot(self, slot: int, tokens, tok_start, span_ptr, span_lo, span_hi, *, pad_id=0,
                     ignore_index=-100, shift_labels=1) -> Dict[str, np.ndarray]:
        """Collate one slot into dense [count, width] arrays (C.4)."""
        count, width = int(self.grp_count[slot]), int(self.grp_width[slot])
        n = max(count * width, 1)
        ids = np.zeros(n, np.int32)
        mask = np.zeros(n, np.uint8)
        pos = np.zeros(n, np.int32)
        lab = np.zeros(n, np.int32)
        tokens = np.ascontiguousarray(tokens, dtype=np.int32)
        tok_start = np.ascontiguousarray(tok_start, dtype=np.int64)
        span_ptr = np.ascontiguousarray(span_ptr, dtype=np.int64)
        span_lo = np.ascontiguousarray(span_lo, dtype=np.int32)
        span_hi = np.ascontiguousarray(span_hi, dtype=np.int32)
        i32, i64 = ctypes.c_int32, ctypes.c_int64
        valid = lib().oracle_collate_slot(self._h, slot, _p(tokens, i32), _p(tok_start, i64), _p(span_ptr, i64),
                                          _p(span_lo, i32), _p(span_hi, i32), pad_id, ignore_index, shift_labels,
                                          _p(ids, i32), _p(mask, ctypes.c_uint8), _p(pos, i32), _p(lab, i32))
        sh = (count, width)
        n = count * width
        return dict(input_ids=ids[:n].reshape(sh), attention_mask=mask[:n].reshape(sh),
                    position_ids=pos[:n].reshape(sh), labels=lab[:n].reshape(sh), valid=int(valid))

    def collate_all(self, tokens, tok_start, span_ptr, span_lo, span_hi, *, pad_id=0, ignore_index=-100,
                    shift_labels=1, sentinel: int = 0x5A, outputs: bool = True) -> Dict[str, np.ndarray]:
        """All slots into flat arenas laid out at grp_offset; gaps keep the sentinel fill."""
        n = max(self.total_elems, 1)
        i32, i64 = ctypes.c_int32, ctypes.c_int64
        if outputs:
            s32 = np.int32(sentinel | (sentinel << 8) | (sentinel << 16) | (sentinel << 24))
            ids = np.full(n, s32, np.int32)
            pos = np.full(n, s32, np.int32)
            lab = np.full(n, s32, np.int32)
            mask = np.full(n, sentinel, np.uint8)
        else:
            ids = pos = lab = mask = None
        gv = np.zeros(max(self.n_slots, 1), np.int32)
        sv = np.zeros(max(self.n_steps, 1), np.int64)
        tokens = np.ascontiguousarray(tokens, dtype=np.int32)
        tok_start = np.ascontiguousarray(tok_start, dtype=np.int64)
        span_ptr = np.ascontiguousarray(span_ptr, dtype=np.int64)
        span_lo = np.ascontiguousarray(span_lo, dtype=np.int32)
        span_hi = np.ascontiguousarray(span_hi, dtype=np.int32)
        lib().oracle_collate_all(self._h, _p(tokens, i32), _p(tok_start, i64), _p(span_ptr, i64), _p(span_lo, i32),
                                 _p(span_hi, i32), pad_id, ignore_index, shift_labels, _p(ids, i32),
                                 _p(mask, ctypes.c_uint8), _p(pos, i32), _p(lab, i32), _p(gv, i32), _p(sv, i64))
        return dict(input_ids=ids, attention_mask=mask, position_ids=pos, labels=lab,
                    grp_valid_tokens=gv[:self.n_slots], step_valid_tokens=sv[:self.n_steps])


def collate_rank(plan: "OraclePlan", r: int, tokens, tok_start, span_ptr, span_lo, span_hi, *, pad_id=0,
                 ignore_index=-100, shift_labels=1, sentinel: int = 0x5A) -> Dict[str, np.ndarray]:
    """Rank r's slots into flat buffers that start at the rank's first arena element (gaps keep the sentinel).
    ``tokens`` / ``tok_start`` need to cover rank r's samples only (tok_start is indexed by global sample id).
    Thread-safe (the collation routines only read the plan)."""
    K = plan.n_steps
    s0, s1 = r * K, (r + 1) * K
    e0 = int(plan.grp_offset[s0]) if s0 < plan.n_slots else plan.total_elems
    e1 = int(plan.grp_offset[s1]) if s1 < plan.n_slots else plan.total_elems
    n = max(e1 - e0, 1)
    s32 = np.int32(sentinel | (sentinel << 8) | (sentinel << 16) | (sentinel << 24))
    ids, pos, lab = np.full(n, s32, np.int32), np.full(n, s32, np.int32), np.full(n, s32, np.int32)
    mask = np.full(n, sentinel, np.uint8)
    gv = np.zeros(max(K, 1), np.int32)
    i32, i64 = ctypes.c_int32, ctypes.c_int64
    tokens = np.ascontiguousarray(tokens, dtype=np.int32)
    tok_start = np.ascontiguousarray(tok_start, dtype=np.int64)
    lib().oracle_collate_range(plan._h, s0, s1, e0, _p(tokens, i32), _p(tok_start, i64),
                               _p(np.ascontiguousarray(span_ptr, dtype=np.int64), i64),
                               _p(np.ascontiguousarray(span_lo, dtype=np.int32), i32),
                               _p(np.ascontiguousarray(span_hi, dtype=np.int32), i32), pad_id, ignore_index,
                               shift_labels, _p(ids, i32), _p(mask, ctypes.c_uint8), _p(pos, i32), _p(lab, i32),
                               _p(gv, i32))
    m = e1 - e0
    return dict(elem_lo=e0, elem_hi=e1, input_ids=ids[:m], attention_mask=mask[:m], position_ids=pos[:m],
                labels=lab[:m], grp_valid_tokens=gv[:K])


def run_workload(wl, tokens=None, *, collate: bool = True, avail_schedule=None):
    """Plan (and optionally collate) an ``odb_inputs.Workload``.  Returns (plan, outputs-or-None)."""
    p = wl.params
    plan = OraclePlan(wl.lengths, wl.rank_ptr, avail_schedule=avail_schedule, **p)
    if not collate:
        return plan, None
    if tokens is None:
        tokens = wl.tokens()
    out = plan.collate_all(tokens, wl.sample_ptr[:-1], wl.span_ptr, wl.span_lo, wl.span_hi, pad_id=p["pad_id"],
                           ignore_index=p["ignore_index"], shift_labels=p["shift_labels"])
    return plan, out
