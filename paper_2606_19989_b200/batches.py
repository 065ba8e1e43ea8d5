"""Step-wise view of a collated plan: what a training loop iterates over (adapter).

The paper's main-process iterator "pops batches from the output queue and transparently skips
IDLE_DATA sentinels" (section 2.1); every rank sees the same number of steps (P:40,
reading U26: step k = slot k of every rank).  Here a collated plan already sits in four flat arenas;
this module only builds zero-copy ``[count, width]`` tensor VIEWS of them, per step and rank, and
leaves out IDLE slots.  No arithmetic of the method happens here (plumbing).
"""
from __future__ import annotations

from typing import Dict, Iterator, List, Optional


class StepBatches:
    """``for step in StepBatches(out, info, n_ranks): step[r] -> batch dict or None (IDLE)``.

    ``out`` is an ``OutputBuffers`` filled by odb_collate / odb_run (device or pinned host).  The
    per-slot tables are read back once (a few KB).  ``weights`` (optional) is the fp64 tensor written
    by odb_loss_weights: each batch then carries its ``loss_weight`` w_{r,k} (Eq. 2).
    """

    def __init__(self, out, info, n_ranks: int, weights=None):
        self.out = out
        self.n_ranks = int(n_ranks)
        self.n_steps = int(info.n_steps)
        tab = lambda name: out.table(name).cpu().tolist()
        self._count = tab("grp_count")
        self._width = tab("grp_width")
        self._offset = tab("grp_offset")
        self._valid = tab("grp_valid_tokens")
        self._round = tab("grp_round")
        self._sptr = tab("grp_sample_ptr")
        self._step_valid = tab("step_valid_tokens")
        self._step_samples = tab("step_samples")
        self._weights = weights

    def __len__(self) -> int:
        return self.n_steps

    def batch(self, rank: int, step: int) -> Optional[Dict]:
        """The batch rank ``rank`` trains on at step ``step``; None for an IDLE slot."""
        s = rank * self.n_steps + step
        c, w = self._count[s], self._width[s]
        if c == 0:
            return None
        o = self._offset[s]
        view = lambda t: t[o:o + c * w].view(c, w)
        b = dict(input_ids=view(self.out.input_ids), attention_mask=view(self.out.attention_mask),
                 position_ids=view(self.out.position_ids), labels=view(self.out.labels),
                 sample_ids=self.out.grp_sample_ids[self._sptr[s]:self._sptr[s + 1]], valid_tokens=self._valid[s],
                 step_valid_tokens=self._step_valid[step], step_samples=self._step_samples[step],
                 round=self._round[s], rank=rank, step=step)
        if self._weights is not None:
            b["loss_weight"] = self._weights[s]
        return b

    def __iter__(self) -> Iterator[List[Optional[Dict]]]:
        for k in range(self.n_steps):
            yield [self.batch(r, k) for r in range(self.n_ranks)]

    def rank_iter(self, rank: int) -> Iterator[Dict]:
        """What one rank's training loop sees: its real batches in step order, IDLE slots skipped."""
        for k in range(self.n_steps):
            b = self.batch(rank, k)
            if b is not None:
                yield b


class StepStream:
    """A terminated plan pulled through TWO output buffers of bounded size, ``steps_per_chunk`` steps at a time
    (odb_collate_steps): ``for chunk in StepStream(...): for step in chunk: ...`` where ``chunk`` is a
    ``StepBatches`` over the chunk's steps (``chunk.step_lo`` = its first plan-wide step).  While the consumer
    works on chunk i, chunk i + 1 is being collated on the other stream into the other buffer (double buffering,
    SURVEY.md 8(f) F3; "output queue").  The views of a chunk are valid until the NEXT chunk is requested:
    asking for chunk i hands the buffer of chunk i - 1 back, and chunk i + 1 is enqueued into it at once.  That
    overwrite is ordered behind whatever the consumer had enqueued, up to the moment of the request, on the stream
    that is current when it asks (an event recorded there, waited on by the collating stream); work on any other
    stream must be joined to that stream (``wait_stream``) before asking.  ``slot_elems`` bounds one slot's block
    (max(budget, longest sample) is enough); plumbing only.
    """

    def __init__(self, ctx, n_ranks: int, n_steps: int, n_samples: int, inputs, steps_per_chunk: int, slot_elems: int,
                 device, fill: Optional[int] = None):
        import torch
        from . import binding as B
        self._B = B
        self.ctx = ctx
        self.n_ranks, self.n_steps = int(n_ranks), int(n_steps)
        self.inputs = inputs  # (d_tokens, d_sample_ptr, d_span_ptr, d_span_lo, d_span_hi)
        self.chunk = max(1, int(steps_per_chunk))
        slots = self.n_ranks * self.chunk
        elems = slots * ((int(slot_elems) + 15) // 16 * 16)
        ids = min(slots * int(slot_elems), int(n_samples))  # (a sample has at least one token)
        self.bufs = [B.OutputBuffers(self.n_ranks, elems, slots, ids, self.chunk, 0, device, fill=fill) for _ in range(2)]
        self.streams = [torch.cuda.Stream(device=device) for _ in range(2)]
        self.device = device
        self._torch = torch

    def __len__(self) -> int:
        return (self.n_steps + self.chunk - 1) // self.chunk

    def _issue(self, i: int):
        lo = i * self.chunk
        hi = min(self.n_steps, lo + self.chunk)
        b = i & 1
        # buffer b last held chunk i - 2, which the consumer gave up with this request: its reads come first
        released = self._torch.cuda.Event()
        released.record(self._torch.cuda.current_stream(self.device))
        self.streams[b].wait_event(released)
        info = self._B.odb_collate_steps(self.ctx, lo, hi, *self.inputs, self.bufs[b].struct,
                                         stream=self.streams[b].cuda_stream)
        return b, info, lo

    def __iter__(self) -> Iterator[StepBatches]:
        n = len(self)
        pending = self._issue(0) if n else None
        for i in range(n):
            nxt = self._issue(i + 1) if i + 1 < n else None  # enqueued before chunk i is handed out
            b, info, lo = pending
            self.streams[b].synchronize()
            sb = StepBatches(self.bufs[b], info, self.n_ranks)
            sb.step_lo = lo
            yield sb
            pending = nxt
