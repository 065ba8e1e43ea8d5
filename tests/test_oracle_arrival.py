"""Pins of the oracle's arrival-schedule mode (status code 0 "insufficient data" and skip rounds,
PAPER.md:52; App. C.1; Lemma 1, Lemma 2, Thm 1): hand-worked fixture e8,
reduction to the synchronous plan, and the theorems' invariants under random schedules."""
import numpy as np
import pytest

import odb_inputs as I
from tests import _golden as G


@pytest.fixture(scope="module")
def oracle():
    from oracle import odb_oracle
    odb_oracle.build()
    return odb_oracle


def _e8(oracle, **kw):
    g = G.load("e8_arrival.txt")
    per_rank = [G.ints(x) for x in g["rank_lengths"].split("|")]
    lens = np.array([x for r in per_rank for x in r], np.int32)
    return g, oracle.OraclePlan(lens, np.array([0, 4, 8], np.int64), budget=int(g["budget"]), **kw)


def test_e8_case1_status0_rank_gets_idle_slots(oracle):
    g, p = _e8(oracle, avail_schedule=[G.ints(G.load("e8_arrival.txt")["case1_schedule"])])
    assert p.groups_of_rank(0) == G.groups(g["case1_groups_a"])
    assert p.groups_of_rank(1) == G.groups(g["case1_groups_b"])
    assert p.grp_round.reshape(2, -1).tolist() == [G.ints(g["case1_rounds_of_slots"])] * 2
    assert p.n_rounds == int(g["case1_n_rounds"]) and p.round_T.tolist() == G.ints(g["case1_round_T"])
    assert p.stop_reason == oracle.STOP_ALL_FINISHED and p.samples_emitted == 8


def test_e8_case2_nonjoin_stops_when_a_rank_finishes(oracle):
    g, p = _e8(oracle, join_mode=0, avail_schedule=[G.ints(G.load("e8_arrival.txt")["case1_schedule"])])
    assert p.groups_of_rank(0) == G.groups(g["case2_groups_a"])
    assert p.groups_of_rank(1) == G.groups(g["case2_groups_b"])
    assert p.n_rounds == int(g["case2_n_rounds"]) and p.stop_reason == int(g["case2_stop"])
    assert p.left_ids[p.left_ptr[1]:p.left_ptr[2]].tolist() == G.ints(g["case2_left_b"])


def test_e8_case3_skip_round(oracle):
    g, p = _e8(oracle, avail_schedule=[G.ints(G.load("e8_arrival.txt")["case3_schedule"])])
    assert p.groups_of_rank(0) == G.groups(g["case3_groups_a"])
    assert p.groups_of_rank(1) == G.groups(g["case3_groups_b"])
    assert p.grp_round.reshape(2, -1).tolist() == [G.ints(g["case3_rounds_of_slots"])] * 2
    assert p.n_rounds == int(g["case3_n_rounds"]) and p.round_T.tolist() == G.ints(g["case3_round_T"])


def _random_schedule(rng, wl, n_rounds):
    """Non-decreasing arrivals per rank, some ranks starved for a while, some rounds with no arrival at all."""
    n = np.diff(wl.rank_ptr)
    sched = np.zeros((n_rounds, wl.n_ranks), np.int64)
    cur = np.zeros(wl.n_ranks, np.int64)
    for j in range(n_rounds):
        step = rng.integers(0, np.maximum(n // 3, 2) + 1)
        step[rng.random(wl.n_ranks) < 0.4] = 0
        cur = np.minimum(cur + step, n)
        sched[j] = cur
    return sched


def test_full_availability_schedule_is_the_synchronous_plan(oracle):
    for kind in ("overflow_multiround", "unequal", "empty_rank"):
        wl = I.protocol_workload(kind, 1)
        a, _ = oracle.run_workload(wl, collate=False)
        big = np.tile(np.diff(wl.rank_ptr), (3, 1))
        b, _ = oracle.run_workload(wl, collate=False, avail_schedule=big)
        for name in ("grp_count", "grp_width", "grp_round", "grp_offset", "grp_sample_ids", "step_samples", "round_T"):
            assert np.array_equal(getattr(a, name), getattr(b, name)), (kind, name)
        assert (a.n_rounds, a.n_steps, a.stop_reason) == (b.n_rounds, b.n_steps, b.stop_reason)


@pytest.mark.parametrize("seed", range(40))
def test_invariants_under_random_schedules(oracle, seed):
    """Lemma 1 (no leak): emitted + left = all; Thm 1 (join): every id exactly once per rank; every rank
    holds the same number of slots; every group within budget or a singleton (U10); slot rounds
    non-decreasing; the number of rounds is bounded by schedule length + the synchronous bound (Thm 4
    P:331 with the skip rounds of Lemma 2 counted: at most one per schedule entry)."""
    rng = np.random.default_rng(seed)
    wl = I.protocol_workload("fuzz", seed)
    join = wl.params["join_mode"]
    sched = _random_schedule(rng, wl, int(rng.integers(1, 12)))
    plan, _ = oracle.run_workload(wl, collate=False, avail_schedule=sched)
    R, K = wl.n_ranks, plan.n_steps
    n = np.diff(wl.rank_ptr)
    assert plan.samples_emitted + plan.samples_left == wl.n_samples
    assert len(plan.grp_count) == R * K
    L = wl.params["budget"]
    for r in range(R):
        ids = [i for k in range(K) for i in plan.slot_ids(r, k)]
        assert len(ids) == len(set(ids))
        left = plan.left_ids[plan.left_ptr[r]:plan.left_ptr[r + 1]].tolist()
        assert sorted(ids + left) == list(range(int(n[r])))
        if join:
            assert not left
        lens_r = wl.lengths[wl.rank_ptr[r]:wl.rank_ptr[r + 1]]
        for k in range(K):
            g = plan.slot_ids(r, k)
            if len(g) > 1:
                assert len(g) * int(lens_r[g].max()) <= L
        rr = plan.grp_round.reshape(R, K)[r]
        assert (np.diff(rr) >= 0).all()
    assert plan.n_rounds <= len(sched) + int(n.max()) + 1
    if join:
        assert plan.stop_reason == oracle.STOP_ALL_FINISHED
