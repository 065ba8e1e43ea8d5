"""Ranks spread over several processes / GPUs: the host-side protocol driver.

The paper runs one rank per process and exchanges, once per round, every rank's status and group counts
with ONE unconditional all_gather on a dedicated channel (section 2.3; message layout
P:250; deadlock-freedom Lemma 3), then evaluates Eq. 3 and the termination predicates
on the shared tensor.  Here every process holds ``n_ranks`` consecutive virtual ranks of the job on its
own GPU; per round it runs

    odb_form_groups -> all_gather (G_r, S_r) -> odb_align -> all_reduce step totals -> odb_commit

with the collectives issued by THIS module through ``torch.distributed`` (NCCL over NVLink on GPUs) on
device buffers the library exposes (``odb_dist_buffers``).  Every step of the method itself runs in the
kernels of libodb; this module only sequences calls and collectives (plumbing).

The protocol is written as a generator that yields one request per collective, so that the same code
is driven (a) by ``torch.distributed`` (``run``), one process per GPU, and (b) in lock step for several
engines inside one process (``run_lockstep``), which is how a single GPU checks the multi-process path
bit for bit against the oracle without ranks ever waiting on one another.

Every process issues the same collectives in the same order whatever its data (no data-dependent early
exit before a collective): the deadlock-freedom argument of Lemma 3.
"""
from __future__ import annotations

from typing import Generator, List, Sequence, Tuple

import numpy as np

from . import binding as B


# ---- collective requests yielded by the protocol ----------------------------------------------
#   ("max_int", value)                 -> the driver sends back max over processes (int)
#   ("all_gather", out, inp)           -> out = concatenation over processes of inp (tensors)
#   ("all_reduce_sum", t)              -> t = elementwise sum over processes, in place (tensor)
Request = Tuple


class _DevArray:
    """A raw device pointer as something ``torch.as_tensor`` can wrap (no copy)."""

    def __init__(self, ptr: int, count: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (int(count),), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 3, "strides": None}


def _wrap(ptr: int, count: int, typestr: str, device):
    import torch
    if count <= 0 or not ptr:
        return torch.zeros(0, dtype=torch.int32 if typestr == "<i4" else torch.int64, device=device)
    return torch.as_tensor(_DevArray(ptr, count, typestr), device=device)


class CudaEngine:
    """The local half of the protocol on one GPU: a thin holder of an ``Odb`` context in distributed
    mode plus torch views of the buffers the collectives work on."""

    def __init__(self, params: B.odb_params, max_samples_total: int, d_lengths, h_rank_ptr, device: int = 0,
                 stream=None):
        self.ctx = B.Odb(params, max_samples_total, device)
        self.params = params
        self.d_lengths = d_lengths
        self.h_rank_ptr = np.ascontiguousarray(h_rank_ptr, dtype=np.int64)
        self.device = "cuda:%d" % device
        self.stream = stream
        self.n_ranks = int(params.n_ranks)

    def close(self):
        self.ctx.close()

    # window bound of the local ranks: max_r min(n_r, buffer_size or n_r)
    def local_max_window(self) -> int:
        n = np.diff(self.h_rank_ptr)
        m = int(n.max()) if len(n) else 0
        bs = int(self.params.buffer_size)
        return min(m, bs) if bs > 0 else m

    def dist_config(self, world_ranks: int, rank_offset: int, world_max_window: int):
        B.odb_dist_config(self.ctx.h, world_ranks, rank_offset, world_max_window)

    def set_available(self, h_arrived):
        B.odb_set_available(self.ctx.h, h_arrived, self.stream)

    def form_groups(self):
        B.odb_form_groups(self.ctx.h, self.d_lengths, self.h_rank_ptr, self.stream)

    def summary(self):
        b = B.odb_dist_buffers(self.ctx.h)
        return (_wrap(b.d_summary_world, b.summary_world_count, "<i4", self.device),
                _wrap(b.d_summary_local, b.summary_local_count, "<i4", self.device))

    def align(self):
        B.odb_align(self.ctx.h, self.stream)

    def step_samples_window(self):
        b = B.odb_dist_buffers(self.ctx.h)
        return _wrap(b.d_step_samples_round, b.step_window, "<i4", self.device)

    def commit(self):
        B.odb_commit(self.ctx.h, self.stream)

    # ---- batched exchange (the round-parallel planner over several processes; include/odb.h) ----
    def stream_lengths(self):
        """n_r of the local ranks as an int32 tensor on the engine's device (the all_gather's input)."""
        import torch
        return torch.from_numpy(np.diff(self.h_rank_ptr).astype(np.int32)).to(self.device)

    def spec_form(self, n_rounds: int, world_max_stream: int):
        B.odb_dist_spec_form(self.ctx.h, self.d_lengths, self.h_rank_ptr, n_rounds, world_max_stream, self.stream)

    def spec_table(self):
        b = B.odb_dist_buffers(self.ctx.h)
        return _wrap(b.d_spec_G_local, b.spec_G_count, "<i4", self.device)

    def spec_commit(self, g_world, n_world, n_procs: int):
        B.odb_dist_spec_commit(self.ctx.h, g_world, n_world, n_procs, self.stream)

    def spec_step_window(self, n: int):
        b = B.odb_dist_buffers(self.ctx.h)
        return _wrap(b.d_step_samples_round, min(int(n), int(b.step_window)), "<i4", self.device)

    def spec_status(self, max_rounds: int):
        return B.odb_dist_spec_status(self.ctx.h, max_rounds)

    def round_status(self):
        return B.odb_round_status(self.ctx.h)

    def plan_query(self):
        return B.odb_plan_query(self.ctx.h)

    def collate(self, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, out: B.OutputBuffers):
        B.odb_collate(self.ctx.h, d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi, out.struct, self.stream)

    def loss_numerators(self, mode: int, d_num):
        B.odb_loss_numerators(self.ctx.h, mode, d_num, self.stream)

    def loss_normalize(self, d_num_world, world_ranks: int, rank_offset: int, d_weights):
        B.odb_loss_normalize(self.ctx.h, d_num_world, world_ranks, rank_offset, d_weights, self.stream)


# ---- the protocol ------------------------------------------------------------------------------
SPEC_MIN_WINDOW, SPEC_MAX_WINDOW, SPEC_MAX_ROUNDS = 8, 4096, 65535


def batched_rounds(n_world: np.ndarray, params) -> int:
    """Rounds that are certainly not the terminal check and can be exchanged at once (0 = the batched exchange does
    not apply): join -- some stream still holds views; non-join -- every stream does.  Host logic shared by every
    process: the same gathered stream lengths and the same parameters give the same answer everywhere."""
    B_ = int(getattr(params, "buffer_size", 0) or 0)
    join = int(getattr(params, "join_mode", 1))
    quota = int(getattr(params, "sample_quota", 0) or 0)
    if B_ < SPEC_MIN_WINDOW or B_ > SPEC_MAX_WINDOW or (not join and quota > 0) or len(n_world) == 0:
        return 0
    n = int(n_world.max()) if join else int(n_world.min())
    J = (n + B_ - 1) // B_
    return J if 2 <= J <= SPEC_MAX_ROUNDS and J * len(n_world) <= (1 << 22) else 0


def plan_protocol(engine, world_ranks: int, rank_offset: int, avail_schedule=None,
                  batched: bool = True) -> Generator[Request, object, tuple]:
    """Round loop of one process.  Returns (plan info of the local ranks, [T_grp of every emitting round]).
    ``avail_schedule[j]`` (optional): arrived views of the LOCAL ranks at round j (odb_set_available).

    A process whose engine reports an error (a bad length, an invalid argument, a CUDA error) does NOT leave the
    protocol on its own -- its peers would wait for ever in the next collective.  It stops calling its engine,
    keeps issuing the round's collectives with buffers of the agreed sizes, and every round ends with a MAX
    exchange of the error status: all processes then raise together (Lemma 3's "same collectives in the same
    order whatever the data", extended to failures)."""
    import torch
    err = [0]
    exc = [None]

    def call(fn, *a):
        if err[0]:
            return None
        try:
            return fn(*a)
        except B.OdbError as e:
            err[0] = int(e.status) or B.ODB_ERR_STATE
            exc[0] = e
            return None

    # one MAX exchange carries the largest window of the job and, as (n, -n), the largest and the smallest number of
    # ranks any process holds: what decides the protocol's shape below is then the same data in every process
    wmax, r_hi, r_lo = yield ("max_int", [int(engine.local_max_window()), int(engine.n_ranks), -int(engine.n_ranks)])
    even_split = r_hi == -r_lo and r_hi > 0 and world_ranks % r_hi == 0
    call(engine.dist_config, world_ranks, rank_offset, int(wmax))
    # the step-total window of a round has the same size in every process: T_grp <= the largest window of the job
    cap = int(getattr(engine.params, "slot_capacity", 0) or 0)
    window = max(1, min(int(wmax), cap) if cap > 0 else int(wmax))
    dev = getattr(engine, "device", "cpu")
    round_T: List[int] = []
    # ---- batched exchange: every round that starts without leftovers, 3 collectives for all of them ----
    # (a round depends on its predecessors only through the leftovers; Eq. 3 and the no-overflow check of every
    #  round are evaluated by every process on the same gathered tables, so all take the same decisions: Lemma 3)
    # (its [process][round][local rank] layout needs the same number of ranks in every process: with 2 + 6 ranks of 8
    #  every process takes the per-round exchange below -- decided from the exchanged counts, never from the local one)
    if batched and avail_schedule is None and hasattr(engine, "spec_form") and even_split:
        n_local = call(engine.stream_lengths)
        if n_local is None:
            n_local = torch.zeros(engine.n_ranks, dtype=torch.int32, device=dev)
        n_world = torch.zeros(world_ranks, dtype=torch.int32, device=dev)
        yield ("all_gather", n_world, n_local)              # every rank's stream length, once per run
        nw = n_world.cpu().numpy()
        J = batched_rounds(nw, engine.params)
        if J:
            n_max = int(nw.max())
            call(engine.spec_form, J, n_max)
            g_local = call(engine.spec_table)
            if g_local is None or g_local.numel() != J * engine.n_ranks:
                g_local = torch.zeros(J * engine.n_ranks, dtype=torch.int32, device=dev)
            g_world = torch.zeros(J * world_ranks, dtype=torch.int32, device=dev)
            yield ("all_gather", g_world, g_local)          # the G tables of all those rounds (batched)
            call(engine.spec_commit, g_world, n_world, world_ranks // engine.n_ranks)
            win = call(engine.spec_step_window, n_max)
            if win is None or win.numel() != n_max:
                win = torch.zeros(n_max, dtype=torch.int32, device=dev)
            yield ("all_reduce_sum", win)                   # global e_k of the committed rounds' steps
            st = call(engine.spec_status, J)
            worst = yield ("max_int", int(err[0]))
            if worst:
                raise exc[0] if exc[0] is not None else B.OdbError(int(worst), "plan_protocol (a peer process failed)")
            round_T.extend(st[2])
            if st[3]:  # every data round was committed: the terminal check needs no exchange (same data everywhere)
                return engine.plan_query(), round_T
    j = 0
    while True:
        if avail_schedule is not None:
            call(engine.set_available, avail_schedule[j] if j < len(avail_schedule) else None)
            j += 1
        call(engine.form_groups)
        bufs = call(engine.summary)
        if bufs is None:  # (the engine failed: stand-ins of the agreed sizes keep the collective well-formed)
            bufs = (torch.zeros(2 * world_ranks, dtype=torch.int32, device=dev),
                    torch.zeros(2 * engine.n_ranks, dtype=torch.int32, device=dev))
        yield ("all_gather", bufs[0], bufs[1])              # the per-round metadata exchange
        call(engine.align)                                  # Eq. 3 + termination predicates on the shared tensor
        win = call(engine.step_samples_window)
        if win is None or win.numel() != window:
            win = torch.zeros(window, dtype=torch.int32, device=dev) if err[0] else win
        yield ("all_reduce_sum", win)                       # global e_k (trainer-side count)
        call(engine.commit)
        st = call(engine.round_status)
        worst = yield ("max_int", int(err[0]))              # does every process still stand?
        if worst:
            raise exc[0] if exc[0] is not None else B.OdbError(int(worst), "plan_protocol (a peer process failed)")
        done, T = st
        if T > 0:
            round_T.append(T)
        if done:
            break
    return engine.plan_query(), round_T


def step_valid_protocol(step_valid_tokens) -> Generator[Request, object, None]:
    """After the local collate: T_tok per step over ALL ranks (Eq. 2)."""
    yield ("all_reduce_sum", step_valid_tokens)


def loss_weights_protocol(engine, mode: int, world_ranks: int, rank_offset: int, num_local, num_world,
                          weights) -> Generator[Request, object, None]:
    """w_{r,k} of the local slots; denominators run over all ranks of the job in rank order, so the
    result is bit-identical to a single-process evaluation (see odb_loss_normalize)."""
    engine.loss_numerators(mode, num_local)
    yield ("all_gather", num_world, num_local)
    engine.loss_normalize(num_world, world_ranks, rank_offset, weights)


# ---- drivers -----------------------------------------------------------------------------------
class TorchCollectives:
    """``torch.distributed`` (NCCL for CUDA tensors, gloo for CPU tensors)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist = dist
        self.group = group
        self.world_size = dist.get_world_size(group)
        self.rank = dist.get_rank(group)

    def max_int(self, v, device="cpu"):
        """Element-wise MAX over the processes of an int or of a short list of ints (one collective either way)."""
        import torch
        many = isinstance(v, (list, tuple))
        t = torch.tensor([int(x) for x in (v if many else [v])], dtype=torch.int64, device=device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX, group=self.group)
        return [int(x) for x in t.tolist()] if many else int(t.item())

    def all_gather(self, out, inp):
        if inp.numel() == 0:
            return
        self.dist.all_gather_into_tensor(out, inp, group=self.group)

    def all_reduce_sum(self, t):
        if t.numel() == 0:
            return
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)


def run(gen: Generator, coll: TorchCollectives, device="cpu"):
    """Drive one protocol generator with real collectives.  Returns the generator's return value."""
    reply = None
    try:
        while True:
            req = gen.send(reply)
            reply = None
            if req[0] == "max_int":
                reply = coll.max_int(req[1], device)
            elif req[0] == "all_gather":
                coll.all_gather(req[1], req[2])
            elif req[0] == "all_reduce_sum":
                coll.all_reduce_sum(req[1])
            else:
                raise ValueError("unknown request %r" % (req[0],))
    except StopIteration as e:
        return e.value


def run_lockstep(gens: Sequence[Generator]):
    """Drive the generators of several processes-in-one in lock step: all are advanced to their next
    collective, the collective is performed among their tensors by plain copies / sums, then all are
    resumed.  Nothing ever waits on a kernel of another engine.  Returns the list of return values."""
    import torch
    n = len(gens)
    replies = [None] * n
    results = [None] * n
    live = [True] * n
    while any(live):
        reqs = [None] * n
        for i, g in enumerate(gens):
            if not live[i]:
                continue
            try:
                reqs[i] = g.send(replies[i])
            except StopIteration as e:
                results[i] = e.value
                live[i] = False
        active = [r for r in reqs if r is not None]
        if not active:
            break
        if len(active) != n or len({r[0] for r in active}) != 1:
            raise RuntimeError("processes diverged: %r" % ([r and r[0] for r in reqs],))  # Lemma 3 would be violated
        kind = active[0][0]
        replies = [None] * n
        if kind == "max_int":
            if isinstance(reqs[0][1], (list, tuple)):
                m = [max(col) for col in zip(*(r[1] for r in reqs))]
                replies = [list(m) for _ in range(n)]
            else:
                m = max(r[1] for r in reqs)
                replies = [m] * n
        elif kind == "all_gather":
            cat = torch.cat([r[2].reshape(-1) for r in reqs]) if reqs[0][2].numel() else None
            for r in reqs:
                if cat is not None:
                    r[1].reshape(-1)[:cat.numel()].copy_(cat)
        elif kind == "all_reduce_sum":
            if reqs[0][1].numel():
                tot = reqs[0][1].clone()
                for r in reqs[1:]:
                    tot += r[1]
                for r in reqs:
                    r[1].copy_(tot)
        else:
            raise ValueError(kind)
    return results
