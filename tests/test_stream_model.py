"""The worker-pool model of paper_2606_19989_b200/stream.py (the asynchronous side of App. C.1):
host logic only, checked on CPU -- the outstanding-depth envelope D = max(pf * nw, buffer_size), its clamp
(App. P), progress (Lemma 2: skip rounds are finite because the envelope lets the workers
deliver), and that a run against the model is the oracle's run under the arrival schedule the model produced."""
import numpy as np
import pytest

import odb_inputs as I
from paper_2606_19989_b200.stream import WorkerPool


def test_envelope_and_clamp():
    p = WorkerPool.from_loader([100, 40, 0], prefetch_factor=2, num_workers=4, buffer_size=32, latency=2)
    assert p.depth == 32                                    # pf * nw = 8 < buffer_size: clamped up to the buffer (App. P)
    assert WorkerPool.from_loader([5], 256, 4, 1024).depth == 1024
    emitted = np.zeros(3, np.int64)
    seen = []
    for k in range(12):
        a = p.step(emitted)
        assert (p.outstanding(emitted) <= p.depth).all() and (a <= p.fetched).all() and (a <= p.n).all()
        seen.append(a.copy())
        emitted = np.minimum(a, emitted + 10)               # the protocol emits at most 10 views per round here
    assert (seen[0] == 0).all() and (seen[1] == 0).all()     # nothing arrives before the latency has passed
    assert seen[2].tolist() == [32, 32, 0]                   # the first envelope's worth
    assert np.all(np.diff(np.array(seen), axis=0) >= 0)      # arrivals never decrease
    assert seen[-1].tolist() == [100, 40, 0]                 # everything is delivered in the end


def test_fetch_quota_hand_values():
    """odb_fetch_quota (include/odb.h; App. P) against values worked by hand: D = max(pf * nw,
    buffer_size); fetch_upto = min(n_r, emitted + D); buffer_size 0 = no bound; bad arguments are refused."""
    import paper_2606_19989_b200 as P
    rp = [0, 100, 140, 140, 1140]                        # n = 100, 40, 0, 1000
    prm = P.make_params(4, 1, buffer_size=32)
    assert P.odb_fetch_quota(prm, rp, 2, 4, [0, 0, 0, 0]).tolist() == [32, 32, 0, 32]          # 8 < 32: D = 32 (clamp)
    assert P.odb_fetch_quota(prm, rp, 16, 4, [0, 0, 0, 0]).tolist() == [64, 40, 0, 64]         # 64 > 32: D = 64
    assert P.odb_fetch_quota(prm, rp, 16, 4, [50, 40, 0, 990]).tolist() == [100, 40, 0, 1000]  # capped by n_r
    assert P.odb_fetch_quota(prm, rp, 0, 0, [10, 1, 0, 500]).tolist() == [42, 33, 0, 532]      # no workers: D = 32
    whole = P.make_params(4, 1, buffer_size=0)
    assert P.odb_fetch_quota(whole, rp, 2, 4, [0, 0, 0, 0]).tolist() == [100, 40, 0, 1000]
    for bad in ([101, 0, 0, 0], [-1, 0, 0, 0]):
        with pytest.raises(P.OdbError):
            P.odb_fetch_quota(prm, rp, 2, 4, bad)
    with pytest.raises(P.OdbError):
        P.odb_fetch_quota(prm, rp, -1, 4, [0, 0, 0, 0])


def _oracle_online(oracle, wl, pool):
    """The protocol rounds of a whole job with the oracle-backed engine of the gloo tests (single process), the
    arrivals coming from the worker model: returns the arrival schedule the run saw and its result."""
    from tests._oracle_engine import OracleEngine
    eng = OracleEngine(oracle, wl)
    eng.dist_config(wl.n_ranks, 0, eng.local_max_window())
    sched, n_skip = [], 0
    emitted = np.zeros(wl.n_ranks, np.int64)
    for _ in range(100000):
        a = pool.step(emitted)
        sched.append(a.copy())
        eng.set_available(a)
        eng.form_groups()
        eng.world[:] = eng.local
        eng.align()
        eng.commit()
        done, T = eng.round_status()
        emitted = np.array([sum(len(g) for g in s) for s in eng.slots], np.int64)
        assert (pool.outstanding(emitted) <= pool.depth).all()
        n_skip += (T == 0 and not done)
        if done:
            break
    return np.array(sched), eng.plan_query(), n_skip


@pytest.mark.parametrize("kind", ["overflow_multiround", "unequal", "empty_rank", "audit:longtail"])
@pytest.mark.parametrize("latency,rate", [(0, None), (1, None), (3, 7)])
def test_online_run_is_the_oracle_run_under_the_models_schedule(oracle, kind, latency, rate):
    wl = I.protocol_workload(kind, 4)
    n = np.diff(wl.rank_ptr)
    bs = wl.params["buffer_size"] or int(n.max())
    pool = WorkerPool.from_loader(n, prefetch_factor=2, num_workers=2, buffer_size=bs, latency=latency, rate=rate)
    sched, res, n_skip = _oracle_online(oracle, wl, pool)
    plan, _ = oracle.run_workload(wl, collate=False, avail_schedule=sched)
    assert (res.n_rounds, res.n_steps, res.stop_reason) == (plan.n_rounds, plan.n_steps, plan.stop_reason)
    for r in range(wl.n_ranks):
        assert res.slots[r] == plan.groups_of_rank(r)
        assert sorted(i for g in res.slots[r] for i in g) == list(range(int(n[r])))      # Thm 1: every view once
    if latency == 0:
        # views arrive in the round they are fetched: the run is the synchronous one
        sync, _ = oracle.run_workload(wl, collate=False)
        assert res.n_steps == sync.n_steps and n_skip == 0
    else:
        assert n_skip >= latency                            # the first rounds find nothing delivered: skip rounds ...
    assert len(sched) <= 2 * (int(n.max()) + latency + 2)    # ... and they are finite (Lemma 2 / Thm 4)
