"""world_size-2 gloo test of the multi-process protocol driver (paper_2606_19989_b200/dist.py) on CPU:
two real processes, real torch.distributed collectives; the local engine is the oracle-backed stand-in
of tests/_oracle_engine.py (the CUDA engine needs a GPU: tests/test_gpu_dist.py).  Each process must
end with the slots the whole-job oracle gives to its ranks, the global step totals, and the same
termination as everyone else (Lemma 3: predicates computed from the same gathered tensor)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


CASES = ["tiny", "unequal", "empty_rank", "overflow_multiround", "overflow_nonjoin_quota", "nonjoin_logical",
         "one_process_idle", "batched_equal", "batched_ragged", "batched_nonjoin", "batched_maxfit",
         "batched_idle_process"]


def _case(name):
    import odb_inputs as I
    if name == "tiny":
        return I.make_workload(0)
    if name == "overflow_nonjoin_quota":
        wl = I.protocol_workload("overflow_multiround", 3, join_mode=0)
        wl.params["sample_quota"] = int(0.6 * wl.n_samples)
        return wl
    if name == "nonjoin_logical":
        return I.protocol_workload("unequal", 5, join_mode=0, buffer_size=32)
    if name == "one_process_idle":   # every rank of the second process is empty from the start
        rng = np.random.default_rng(1)
        return I.custom_workload("one_process_idle", [rng.integers(8, 300, 50), rng.integers(8, 300, 70), [], []],
                                 seed=3, budget=1024, buffer_size=16)
    if name.startswith("batched"):   # several rounds without leftovers: the batched exchange commits them at once
        rng = np.random.default_rng(len(name))
        n = {"batched_equal": (400, 400, 400, 400), "batched_ragged": (390, 412, 0, 405),
             "batched_nonjoin": (300, 260, 280, 310), "batched_maxfit": (200, 333, 333, 90),
             "batched_idle_process": (0, 0, 290, 300)}[name]
        return I.custom_workload(name, [rng.integers(8, 700, k) for k in n], seed=7, budget=2048, buffer_size=40,
                                 join_mode=0 if name == "batched_nonjoin" else 1, rule=1 if name == "batched_maxfit" else 0)
    return I.protocol_workload(name, 2)


def test_batched_rounds_host_logic():
    """Which rounds the batched exchange may take (dist.batched_rounds): join -- until the longest stream is drained;
    non-join -- until the shortest is; never with a quota, tiny or huge buffers, or a single round."""
    from types import SimpleNamespace as NS
    sys.path.insert(0, ROOT)
    from paper_2606_19989_b200 import dist as D
    n = np.array([100, 250, 0, 31])
    assert D.batched_rounds(n, NS(buffer_size=50, join_mode=1, sample_quota=0)) == 5
    assert D.batched_rounds(n, NS(buffer_size=50, join_mode=0, sample_quota=0)) == 0      # a stream is empty: round 0 is terminal
    assert D.batched_rounds(n + 60, NS(buffer_size=50, join_mode=0, sample_quota=0)) == 2
    assert D.batched_rounds(n + 60, NS(buffer_size=50, join_mode=0, sample_quota=10)) == 0
    assert D.batched_rounds(n, NS(buffer_size=4, join_mode=1, sample_quota=0)) == 0
    assert D.batched_rounds(n, NS(buffer_size=0, join_mode=1, sample_quota=0)) == 0
    assert D.batched_rounds(n, NS(buffer_size=5000, join_mode=1, sample_quota=0)) == 0
    assert D.batched_rounds(n, NS(buffer_size=250, join_mode=1, sample_quota=0)) == 0     # one round: nothing to batch
    assert D.batched_rounds(np.array([10**7]), NS(buffer_size=8, join_mode=1, sample_quota=0)) == 0   # too many rounds


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import odb_inputs as I
    from oracle import odb_oracle
    from paper_2606_19989_b200 import dist as D
    from tests._oracle_engine import OracleEngine
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        coll = D.TorchCollectives()
        for name in CASES:
            wl = _case(name)
            rl = wl.n_ranks // world
            part = I.split_ranks(wl, world)[rank]
            eng = OracleEngine(odb_oracle, part)
            info, round_T = D.run(D.plan_protocol(eng, wl.n_ranks, rank * rl), coll)
            q.put((name, rank, info.n_rounds, info.n_steps, info.stop_reason, info.slots, info.step_samples, round_T))
    finally:
        dist.destroy_process_group()


def _failing_worker(rank, world, port, q, fail_round):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import odb_inputs as I
    from oracle import odb_oracle
    from paper_2606_19989_b200 import dist as D
    from paper_2606_19989_b200 import binding as B
    from tests._oracle_engine import OracleEngine
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        wl = _case("overflow_multiround")
        rl = wl.n_ranks // world
        eng = OracleEngine(odb_oracle, I.split_ranks(wl, world)[rank])
        if rank == 1 and fail_round == "spec":
            def boom(*a):
                raise B.OdbError(B.ODB_ERR_BAD_LENGTH, "OracleEngine.spec_form (injected failure)")
            eng.spec_form = boom
        elif rank == 1:
            eng.fail_at_round = fail_round
        try:
            D.run(D.plan_protocol(eng, wl.n_ranks, rank * rl), D.TorchCollectives())
            q.put((rank, "finished", 0))
        except B.OdbError as e:
            q.put((rank, "raised", int(e.status)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("fail_round", [0, 3, "spec"])
def test_a_failing_process_takes_its_peers_down_instead_of_hanging_them(fail_round):
    """One process's engine fails (a bad length, say) in some round: every process issues that round's collectives
    and then raises, together (the MAX exchange of the error status at the end of every round)."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_failing_worker, args=(r, 2, port, q, fail_round)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict((item[0], item[1:]) for item in (q.get(timeout=120) for _ in range(2)))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert got[0] == ("raised", 2) and got[1] == ("raised", 2)     # ODB_ERR_BAD_LENGTH on both


def test_two_process_gloo_protocol_matches_whole_job_oracle():
    import torch.multiprocessing as mp
    sys.path.insert(0, ROOT)
    from oracle import odb_oracle
    odb_oracle.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = {}
    for _ in range(2 * len(CASES)):
        item = q.get(timeout=240)
        got[(item[0], item[1])] = item[2:]
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for name in CASES:
        wl = _case(name)
        plan, _ = odb_oracle.run_workload(wl, collate=False)
        rl = wl.n_ranks // 2
        for rank in range(2):
            n_rounds, n_steps, stop, slots, step_samples, round_T = got[(name, rank)]
            assert (n_rounds, n_steps, stop) == (plan.n_rounds, plan.n_steps, plan.stop_reason), (name, rank)
            assert round_T == plan.round_T.tolist(), (name, rank)
            assert step_samples == plan.step_samples.tolist(), (name, rank)
            for j in range(rl):
                assert slots[j] == plan.groups_of_rank(rank * rl + j), (name, rank, j)


@pytest.mark.parametrize("n_proc", [2, 4])
def test_lockstep_driver_with_oracle_engines(n_proc):
    """The same protocol generator driven in lock step inside one process (dist.run_lockstep, the driver the
    single-GPU tests use), with oracle-backed engines: 2 and 4 "processes", with and without an arrival
    schedule (status 0 / -1 through the gathered summary, skip rounds)."""
    sys.path.insert(0, ROOT)
    import odb_inputs as I
    from oracle import odb_oracle
    from paper_2606_19989_b200 import dist as D
    from tests._oracle_engine import OracleEngine
    from tests.test_oracle_arrival import _random_schedule
    odb_oracle.build()
    for name in ("unequal", "empty_rank", "overflow_multiround", "overflow_nonjoin_quota", "audit:longtail",
                 "batched_equal", "batched_ragged", "batched_nonjoin", "batched_maxfit", "batched_idle_process"):
        for with_sched in (False, True):
            wl = _case(name) if not name.startswith("audit") else I.protocol_workload(name, 2)
            if wl.n_ranks % n_proc:
                continue
            sched = _random_schedule(np.random.default_rng(5), wl, 8) if with_sched else None
            plan, _ = odb_oracle.run_workload(wl, collate=False, avail_schedule=sched)
            rl = wl.n_ranks // n_proc
            engines = [OracleEngine(odb_oracle, part) for part in I.split_ranks(wl, n_proc)]
            res = D.run_lockstep([D.plan_protocol(e, wl.n_ranks, p * rl,
                                                  None if sched is None else [row[p * rl:(p + 1) * rl] for row in sched])
                                  for p, e in enumerate(engines)])
            if name.startswith("batched") and not with_sched:   # the batched exchange committed rounds (all of them
                committed = len(engines[0].spec_T)              # when the streams are equal)
                assert committed >= 2 and (name != "batched_equal" or committed == plan.n_rounds - 1), (name, committed)
            for p, (info, round_T) in enumerate(res):
                assert (info.n_rounds, info.n_steps, info.stop_reason) == (plan.n_rounds, plan.n_steps, plan.stop_reason), name
                assert round_T == plan.round_T.tolist() and info.step_samples == plan.step_samples.tolist()
                for j in range(rl):
                    assert info.slots[j] == plan.groups_of_rank(p * rl + j), (name, with_sched, p, j)


@pytest.mark.parametrize("bounds", [(0, 1, 4), (0, 1, 2, 4), (0, 3, 4)])
def test_lockstep_unequal_rank_counts(bounds):
    """Processes holding different numbers of ranks (1 + 3, 1 + 1 + 2, 3 + 1 of 4): the shape of the protocol is
    decided from exchanged rank counts, so all issue the same collectives (the lock-step driver raises when they
    diverge) and none takes the batched exchange, whose table layout needs equal counts."""
    sys.path.insert(0, ROOT)
    import odb_inputs as I
    from oracle import odb_oracle
    from paper_2606_19989_b200 import dist as D
    from tests._oracle_engine import OracleEngine
    odb_oracle.build()
    for name in ("batched_equal", "batched_ragged", "batched_nonjoin", "overflow_multiround"):
        wl = _case(name)
        assert wl.n_ranks == 4
        plan, _ = odb_oracle.run_workload(wl, collate=False)
        n_proc = len(bounds) - 1
        engines = [OracleEngine(odb_oracle, part) for part in I.split_ranks(wl, n_proc, bounds=bounds)]
        res = D.run_lockstep([D.plan_protocol(e, wl.n_ranks, bounds[p]) for p, e in enumerate(engines)])
        for p, (info, round_T) in enumerate(res):
            assert not getattr(engines[p], "spec_T", None), (name, bounds)  # the batched exchange was not taken
            assert (info.n_rounds, info.n_steps, info.stop_reason) == (plan.n_rounds, plan.n_steps, plan.stop_reason), name
            assert round_T == plan.round_T.tolist() and info.step_samples == plan.step_samples.tolist()
            for j in range(bounds[p + 1] - bounds[p]):
                assert info.slots[j] == plan.groups_of_rank(bounds[p] + j), (name, bounds, p, j)
