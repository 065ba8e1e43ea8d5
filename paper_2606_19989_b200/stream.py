"""Online operation: a model of the asynchronous side of the paper's per-rank state machine
(App. C.1) that drives the library's arrival interface.

In the paper a sampler view travels  R_r (sampler-pending) -> Q_r (worker queue) -> B_r (collate buffer) -> E_r
(emitted); the iterator schedules Fetch so that the fetched-but-not-emitted set Q_r + B_r stays within the
OUTSTANDING-DEPTH ENVELOPE  D = max(prefetch_factor * num_workers, buffer_size)  (the clamp to
buffer_size is App. P).  The library itself is synchronous: it is told, before every round, how many
views of each rank's stream have ARRIVED (``odb_set_available``); a rank whose window is empty while views are
pending advertises status 0 "insufficient data", and a round in which nobody has a group is a skip round (
Lemma 2 P:323-329 is why such rounds are finite: the envelope lets the workers make progress).

``WorkerPool`` is that missing asynchronous side as a small deterministic model: per round it fetches as many
views as the envelope allows and delivers them ``latency`` rounds later, at most ``rate`` per round and rank.
``plan_online`` runs the protocol rounds against it.  No arithmetic of the method lives here: grouping, alignment
and termination run in the kernels behind the C ABI, the envelope and its clamp are ``odb_fetch_quota``, the emit
cursors ``odb_emitted_counts``; this module only decides WHEN a fetched view becomes visible (latency, rate).
"""
from __future__ import annotations

from collections import deque
from typing import List, Optional, Sequence

import numpy as np

from . import binding as B


class WorkerPool:
    """Deterministic model of a rank's DataLoader workers under the outstanding-depth envelope."""

    def __init__(self, n_per_rank: Sequence[int], quota, depth: int, latency: int = 1, rate: Optional[int] = None):
        """``quota(emitted) -> fetch_upto`` is the envelope rule (``from_loader``: the library's odb_fetch_quota);
        ``depth`` is D as the library reports it, kept for the caller's checks and logs."""
        if latency < 0:
            raise ValueError("latency >= 0")
        self.n = np.asarray(n_per_rank, dtype=np.int64)
        self.quota = quota
        self.depth = int(depth)
        self.latency = int(latency)
        self.rate = None if rate is None else int(rate)
        self.fetched = np.zeros_like(self.n)
        self.arrived = np.zeros_like(self.n)
        self._in_flight = deque([np.zeros_like(self.n) for _ in range(self.latency)])

    @classmethod
    def from_loader(cls, n_per_rank, prefetch_factor: int, num_workers: int, buffer_size: int, **kw) -> "WorkerPool":
        """A pool whose Fetch follows the library's envelope, odb_fetch_quota: D = max(prefetch_factor * num_workers,
        buffer_size) with its clamp (App. P) is computed behind the C ABI, not here."""
        n = np.asarray(n_per_rank, dtype=np.int64)
        rp = np.concatenate([[0], np.cumsum(n)]).astype(np.int64)
        prm = B.make_params(len(n), 1, buffer_size=int(buffer_size))
        quota = lambda emitted: B.odb_fetch_quota(prm, rp, prefetch_factor, num_workers, emitted)
        # D itself, for reporting: what one rank with an endless stream and nothing emitted may fetch
        one = B.make_params(1, 1, buffer_size=int(buffer_size))
        depth = int(B.odb_fetch_quota(one, [0, 1 << 40], prefetch_factor, num_workers, [0])[0])
        return cls(n, quota, depth, **kw)

    def step(self, emitted: Sequence[int]) -> np.ndarray:
        """One protocol round: Fetch up to the envelope, Drain what the workers have finished.  ``emitted[r]`` =
        views of rank r emitted so far.  Returns the arrived counts to hand to odb_set_available."""
        emitted = np.asarray(emitted, dtype=np.int64)
        # Fetch: |Q + B| = fetched - emitted <= D
        self.fetched = np.maximum(self.fetched, self.quota(emitted))
        self._in_flight.append(self.fetched.copy())
        ready = self._in_flight.popleft()          # what was fetched `latency` rounds ago has been processed ...
        if self.rate is not None:                  # ... unless the workers' throughput caps it
            ready = np.minimum(ready, self.arrived + self.rate)
        self.arrived = np.maximum(self.arrived, ready)
        return self.arrived.copy()

    def outstanding(self, emitted: Sequence[int]) -> np.ndarray:
        return self.fetched - np.asarray(emitted, dtype=np.int64)


def plan_online(ctx: "B.Odb", d_lengths, h_rank_ptr, pool: WorkerPool, stream=None, max_rounds: int = 1 << 22):
    """The round loop against a worker model.  Returns (plan info, log) where log[j] = dict(arrived, emitted, T) of
    round j (``arrived`` is the schedule the run actually saw: replaying it through an oracle gives the same plan)."""
    R = int(ctx.params.n_ranks)
    B.odb_reset(ctx.h)
    emitted = np.zeros(R, dtype=np.int64)
    log: List[dict] = []
    done = 0
    while not done:
        if len(log) >= max_rounds:
            raise RuntimeError("plan_online: no termination after %d rounds (a worker model that never delivers?)" % max_rounds)
        arrived = pool.step(emitted)
        B.odb_set_available(ctx.h, arrived, stream)
        B.odb_form_groups(ctx.h, d_lengths, h_rank_ptr, stream)
        B.odb_align(ctx.h, stream)
        done, T = B.odb_round_status(ctx.h)
        emitted = B.odb_emitted_counts(ctx.h, R)
        log.append(dict(arrived=arrived, emitted=emitted.copy(), T=int(T), outstanding=pool.outstanding(emitted)))
    return B.odb_plan_query(ctx.h), log
