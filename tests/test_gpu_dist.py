"""The multi-process path on ONE GPU: the R ranks of a job are split over 2 or 4
contexts ("processes"), each driven by the very protocol generator a torch.distributed run uses
(paper_2606_19989_b200/dist.py), in lock step -- all contexts are advanced to their next collective,
the collective is done by plain tensor copies / sums, all are resumed, so no kernel ever waits on
another context.  Every process's slots, arenas, step totals and loss weights must equal, bit for
bit, the oracle's result for the WHOLE job restricted to that process's ranks."""
import numpy as np
import pytest

import odb_inputs as I
from tests import _parity as Par

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu tests need a CUDA device (there is no CPU fallback to test)")
    import paper_2606_19989_b200 as P
    P.load()
    return P


@pytest.fixture(scope="module")
def oracle():
    from oracle import odb_oracle
    odb_oracle.build()
    return odb_oracle


def _case(name):
    if name == "tiny":
        return I.make_workload(0)
    if name == "config2_slice":
        return I.make_workload(1, n_ranks=4, n_per_rank=600)
    if name == "config4_slice_nonjoin":
        return I.make_workload(3, n_ranks=4, n_per_rank=700, join_mode=0)
    if name == "overflow_nonjoin_quota":
        wl = I.protocol_workload("overflow_multiround", 3, join_mode=0)
        wl.params["sample_quota"] = int(0.6 * wl.n_samples)
        return wl
    if name.startswith("sampleless_process"):   # one process whose ranks hold no sample at all (soak seed 25)
        rng = np.random.default_rng(25)
        per = [[], rng.integers(1, 1500, 43), rng.integers(1, 1500, 58), rng.integers(1, 100, 20)]
        join = 0 if name.endswith("nonjoin") else 1
        return I.custom_workload(name, per, 25, budget=4096, buffer_size=64, slot_capacity=17, join_mode=join,
                                 sample_quota=0 if join else 42)
    if name == "maxfit_overflow":
        return I.protocol_workload("overflow_multiround", 5, rule=1)
    if name.startswith("batched"):   # several rounds without leftovers: the batched exchange commits them at once
        rng = np.random.default_rng(len(name))
        n = {"batched_equal": (3000, 3000, 3000, 3000), "batched_ragged": (3000, 2817, 0, 3105),
             "batched_nonjoin": (3000, 2600, 2800, 3100), "batched_maxfit": (2000, 3333, 3333, 900),
             "batched_idle_process": (0, 0, 2900, 3000)}[name]
        return I.custom_workload(name, [rng.integers(8, 1500, k) for k in n], seed=7, budget=8192, buffer_size=256,
                                 join_mode=0 if name == "batched_nonjoin" else 1, rule=1 if name == "batched_maxfit" else 0)
    return I.protocol_workload(name, 2)


@pytest.mark.parametrize("n_proc", [2, 4])
@pytest.mark.parametrize("name", ["tiny", "config2_slice", "unequal", "empty_rank", "overflow_multiround",
                                  "overflow_nonjoin_quota", "maxfit_overflow", "config4_slice_nonjoin",
                                  "audit:bimodal", "sampleless_process_join", "sampleless_process_nonjoin",
                                  "batched_equal", "batched_ragged", "batched_nonjoin", "batched_maxfit",
                                  "batched_idle_process"])
def test_lockstep_processes_match_whole_job_oracle(P, oracle, name, n_proc):
    import torch
    from paper_2606_19989_b200 import dist as D
    wl = _case(name)
    if wl.n_ranks % n_proc:
        pytest.skip("ranks do not split evenly")
    plan, ref = oracle.run_workload(wl)
    R, K = wl.n_ranks, plan.n_steps
    rl = R // n_proc
    parts = I.split_ranks(wl, n_proc)
    dws = [Par.DeviceWorkload(w) for w in parts]
    engines = [D.CudaEngine(Par.gpu_params(w), max(w.n_samples, 1), dw.lengths, w.rank_ptr) for w, dw in zip(parts, dws)]
    try:
        res = D.run_lockstep([D.plan_protocol(e, R, p * rl) for p, e in enumerate(engines)])
        outs = []
        for p, (e, w, dw) in enumerate(zip(engines, parts, dws)):
            info, round_T = res[p]
            assert round_T == plan.round_T.tolist()
            assert (info.n_rounds, info.n_steps, info.stop_reason) == (plan.n_rounds, plan.n_steps, plan.stop_reason)
            out = P.OutputBuffers.for_plan(rl, info, dw.device, fill=Par.SENTINEL)
            e.collate(dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out)
            outs.append((info, out))
        D.run_lockstep([D.step_valid_protocol(out.table("step_valid_tokens")) for _, out in outs])
        torch.cuda.synchronize()
        for p, (info, out) in enumerate(outs):
            s0, s1 = p * rl * K, (p + 1) * rl * K
            off0 = int(plan.grp_offset[s0]) if s0 < plan.n_slots else plan.total_elems
            off1 = int(plan.grp_offset[s1]) if s1 < plan.n_slots else plan.total_elems
            q0, q1 = int(plan.grp_sample_ptr[s0]), int(plan.grp_sample_ptr[s1])
            assert int(info.total_elems) == off1 - off0 and int(info.samples_emitted) == q1 - q0
            for name_ in ("grp_count", "grp_width", "grp_round", "grp_real_tokens", "grp_origin"):
                assert np.array_equal(out.table(name_).cpu().numpy(), getattr(plan, name_)[s0:s1]), name_
            assert np.array_equal(out.table("grp_offset").cpu().numpy(), plan.grp_offset[s0:s1] - off0)
            assert np.array_equal(out.table("grp_sample_ptr").cpu().numpy(), plan.grp_sample_ptr[s0:s1 + 1] - q0)
            assert np.array_equal(out.table("grp_sample_ids").cpu().numpy(), plan.grp_sample_ids[q0:q1])
            assert np.array_equal(out.table("grp_valid_tokens").cpu().numpy(), ref["grp_valid_tokens"][s0:s1])
            # global per-step tables: identical on every process
            assert np.array_equal(out.table("step_samples").cpu().numpy(), plan.step_samples)
            assert np.array_equal(out.table("step_valid_tokens").cpu().numpy(), ref["step_valid_tokens"])
            l0, l1 = int(plan.left_ptr[p * rl]), int(plan.left_ptr[(p + 1) * rl])
            assert np.array_equal(out.table("left_ptr").cpu().numpy(), plan.left_ptr[p * rl:(p + 1) * rl + 1] - l0)
            assert np.array_equal(out.table("left_ids").cpu().numpy(), plan.left_ids[l0:l1])
            E = off1 - off0
            for name_ in ("input_ids", "labels", "position_ids", "attention_mask"):
                assert np.array_equal(getattr(out, name_)[:E].cpu().numpy(), ref[name_][off0:off1]), name_
        # loss weights: denominators over all ranks of the job, bit-identical to the single-process oracle
        for mode in (P.ODB_SCALE_SAMPLE, P.ODB_SCALE_TOKEN_APPROX, P.ODB_SCALE_TOKEN_EXACT):
            want = oracle.loss_weights(mode, R, K, plan.grp_count, ref["grp_valid_tokens"], plan.grp_origin)
            bufs = []
            for p, e in enumerate(engines):
                num_local = torch.zeros(max(rl * K, 1), dtype=torch.float64, device="cuda:0")[:rl * K]
                num_world = torch.zeros(max(R * K, 1), dtype=torch.float64, device="cuda:0")[:R * K]
                w = torch.full((max(rl * K, 1),), float("nan"), dtype=torch.float64, device="cuda:0")[:rl * K]
                bufs.append((num_local, num_world, w))
            D.run_lockstep([D.loss_weights_protocol(e, mode, R, p * rl, *bufs[p]) for p, e in enumerate(engines)])
            torch.cuda.synchronize()
            for p in range(n_proc):
                got = bufs[p][2].cpu().numpy().reshape(rl, K)
                assert np.array_equal(got.view(np.uint64), want[p * rl:(p + 1) * rl].view(np.uint64)), (mode, p)
    finally:
        for e in engines:
            e.close()


def test_lockstep_with_arrival_schedule(P, oracle):
    """Status 0 / -1 travel through the gathered summary (S encoded as -1 when finished): two contexts with
    a random arrival schedule equal the whole-job oracle run with the same schedule."""
    import torch
    from paper_2606_19989_b200 import dist as D
    from tests.test_oracle_arrival import _random_schedule
    for seed, join in ((0, 1), (1, 1), (2, 0), (3, 1)):
        wl = I.protocol_workload("unequal" if seed % 2 else "overflow_multiround", seed, join_mode=join)
        rng = np.random.default_rng(50 + seed)
        sched = _random_schedule(rng, wl, 7)
        plan, _ = oracle.run_workload(wl, collate=False, avail_schedule=sched)
        R, K = wl.n_ranks, plan.n_steps
        rl = R // 2
        parts = I.split_ranks(wl, 2)
        dws = [Par.DeviceWorkload(w) for w in parts]
        engines = [D.CudaEngine(Par.gpu_params(w), max(w.n_samples, 1), dw.lengths, w.rank_ptr) for w, dw in zip(parts, dws)]
        try:
            res = D.run_lockstep([D.plan_protocol(e, R, p * rl, [row[p * rl:(p + 1) * rl] for row in sched])
                                  for p, e in enumerate(engines)])
            for p, (e, dw) in enumerate(zip(engines, dws)):
                info, round_T = res[p]
                assert round_T == plan.round_T.tolist()
                assert (info.n_rounds, info.n_steps, info.stop_reason) == (plan.n_rounds, plan.n_steps, plan.stop_reason)
                out = P.OutputBuffers.for_plan(rl, info, dw.device)
                e.collate(dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out)
                torch.cuda.synchronize()
                s0, s1 = p * rl * K, (p + 1) * rl * K
                q0, q1 = int(plan.grp_sample_ptr[s0]), int(plan.grp_sample_ptr[s1])
                assert np.array_equal(out.table("grp_count").cpu().numpy(), plan.grp_count[s0:s1])
                assert np.array_equal(out.table("grp_round").cpu().numpy(), plan.grp_round[s0:s1])
                assert np.array_equal(out.table("grp_sample_ids").cpu().numpy(), plan.grp_sample_ids[q0:q1])
                assert np.array_equal(out.table("step_samples").cpu().numpy(), plan.step_samples)
        finally:
            for e in engines:
                e.close()


def test_batched_exchange_commits_rounds_and_equals_the_round_by_round_protocol(P, oracle):
    """The batched exchange (odb_dist_spec_form / _commit / _status): equal streams -- every data round is committed
    with three collectives; ragged streams -- the tail falls to the per-round protocol; the plan is the oracle's
    either way and equals the protocol with one exchange per round (batched=False)."""
    import torch
    from paper_2606_19989_b200 import dist as D
    for name, all_rounds in (("batched_equal", True), ("batched_ragged", False), ("batched_nonjoin", True)):
        wl = _case(name)
        plan, _ = oracle.run_workload(wl, collate=False)
        R = wl.n_ranks
        parts = I.split_ranks(wl, 2)
        dws = [Par.DeviceWorkload(w) for w in parts]
        for batched in (True, False):
            engines = [D.CudaEngine(Par.gpu_params(w), max(w.n_samples, 1), dw.lengths, w.rank_ptr) for w, dw in zip(parts, dws)]
            try:
                n_coll = [0]

                def counted(gen):
                    reply = None
                    while True:
                        try:
                            req = gen.send(reply)
                        except StopIteration as e:
                            return e.value
                        n_coll[0] += 1
                        reply = yield req

                res = D.run_lockstep([counted(D.plan_protocol(e, R, p * 2, batched=batched)) for p, e in enumerate(engines)])
                for p, e in enumerate(engines):
                    info, round_T = res[p]
                    assert round_T == plan.round_T.tolist(), (name, batched)
                    assert (info.n_rounds, info.n_steps, info.stop_reason) == (plan.n_rounds, plan.n_steps, plan.stop_reason)
                    rec = np.zeros(4, dtype=np.int32)
                    got = P.odb_debug_read(e.ctx.h, 4, rec)
                    if batched:
                        assert got == 16 and rec[0] >= 2
                        assert (rec[0] == plan.n_rounds - 1) == all_rounds, (name, rec)
                    else:
                        assert got < 0
                    out = P.OutputBuffers.for_plan(2, info, dws[p].device)
                    e.collate(dws[p].tokens, dws[p].sample_ptr, dws[p].span_ptr, dws[p].span_lo, dws[p].span_hi, out)
                    torch.cuda.synchronize()
                    K = plan.n_steps
                    s0, s1 = p * 2 * K, (p + 1) * 2 * K
                    assert np.array_equal(out.table("grp_count").cpu().numpy(), plan.grp_count[s0:s1])
                    assert np.array_equal(out.table("grp_width").cpu().numpy(), plan.grp_width[s0:s1])
                    assert np.array_equal(out.table("step_samples").cpu().numpy(), plan.step_samples)
                per_proc = n_coll[0] // 2
                if batched and all_rounds:     # 1 (window) + 4 (batched phase); the terminal check needs no exchange
                    assert per_proc == 5, per_proc
                if not batched:                # 1 + 3 per round, terminal check included
                    assert per_proc == 1 + 3 * plan.n_rounds, per_proc
            finally:
                for e in engines:
                    e.close()


@pytest.mark.parametrize("bounds", [(0, 2, 8), (0, 2, 4, 8), (0, 5, 8), (0, 4, 8)])
def test_lockstep_unequal_rank_counts_take_one_path_everywhere(P, oracle, bounds):
    """8 ranks held by processes with 2 + 6, 2 + 2 + 4, 5 + 3 (and, as the control, 4 + 4) of them, on a job the batched
    exchange would take: whether it is taken is decided from the exchanged rank counts, so every process issues
    the same collectives (run_lockstep raises if they diverge) and the plan is the whole-job oracle's either way."""
    import torch
    from paper_2606_19989_b200 import dist as D
    rng = np.random.default_rng(11)
    wl = I.custom_workload("batched_8", [rng.integers(8, 1500, k) for k in (900, 1000, 950, 0, 1000, 870, 990, 1000)],
                           seed=9, budget=8192, buffer_size=256)
    plan, _ = oracle.run_workload(wl, collate=False)
    R, K = wl.n_ranks, plan.n_steps
    n_proc = len(bounds) - 1
    parts = I.split_ranks(wl, n_proc, bounds=bounds)
    dws = [Par.DeviceWorkload(w) for w in parts]
    engines = [D.CudaEngine(Par.gpu_params(w), max(w.n_samples, 1), dw.lengths, w.rank_ptr) for w, dw in zip(parts, dws)]
    try:
        res = D.run_lockstep([D.plan_protocol(e, R, bounds[p]) for p, e in enumerate(engines)])
        for p, e in enumerate(engines):
            info, round_T = res[p]
            assert round_T == plan.round_T.tolist()
            assert (info.n_rounds, info.n_steps, info.stop_reason) == (plan.n_rounds, plan.n_steps, plan.stop_reason)
            rec = np.zeros(4, dtype=np.int32)
            took_batched = P.odb_debug_read(e.ctx.h, 4, rec) == 16
            assert took_batched == (bounds == (0, 4, 8)), (bounds, p)
            rl = bounds[p + 1] - bounds[p]
            out = P.OutputBuffers.for_plan(rl, info, dws[p].device)
            e.collate(dws[p].tokens, dws[p].sample_ptr, dws[p].span_ptr, dws[p].span_lo, dws[p].span_hi, out)
            torch.cuda.synchronize()
            s0, s1 = bounds[p] * K, bounds[p + 1] * K
            assert np.array_equal(out.table("grp_count").cpu().numpy(), plan.grp_count[s0:s1])
            assert np.array_equal(out.table("grp_width").cpu().numpy(), plan.grp_width[s0:s1])
            assert np.array_equal(out.table("step_samples").cpu().numpy(), plan.step_samples)
    finally:
        for e in engines:
            e.close()


def test_single_process_nccl_world(P, oracle):
    """The torch.distributed driver itself (NCCL, world_size 1 -- the box has one GPU): the protocol
    with real collectives on the library's device buffers equals the oracle."""
    import os
    import torch
    import torch.distributed as dist
    from paper_2606_19989_b200 import dist as D
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29731")
    created = False
    if not dist.is_initialized():
        torch.cuda.set_device(0)
        dist.init_process_group("nccl", rank=0, world_size=1)
        created = True
    try:
        wl = I.protocol_workload("overflow_multiround", 7)
        plan, ref = oracle.run_workload(wl)
        dw = Par.DeviceWorkload(wl)
        e = D.CudaEngine(Par.gpu_params(wl), wl.n_samples, dw.lengths, wl.rank_ptr)
        try:
            coll = D.TorchCollectives()
            info, round_T = D.run(D.plan_protocol(e, wl.n_ranks, 0), coll, device="cuda:0")
            out = P.OutputBuffers.for_plan(wl.n_ranks, info, dw.device, fill=Par.SENTINEL)
            e.collate(dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out)
            D.run(D.step_valid_protocol(out.table("step_valid_tokens")), coll, device="cuda:0")
            torch.cuda.synchronize()
            assert round_T == plan.round_T.tolist()
            Par.compare_plan(plan, info, out)
            Par.compare_full(plan, ref, info, out)
        finally:
            e.close()
    finally:
        if created:
            dist.destroy_process_group()


def test_dist_mode_errors(P):
    wl = I.make_workload(0)
    dw = Par.DeviceWorkload(wl)
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        with pytest.raises(P.OdbError):
            P.odb_commit(ctx.h)                       # not in distributed mode
        with pytest.raises(P.OdbError):
            P.odb_dist_buffers(ctx.h)
        with pytest.raises(P.OdbError):
            P.odb_dist_config(ctx.h, 1, 0, 64)        # world smaller than the local ranks
        P.odb_dist_config(ctx.h, 4, 2, 64)
        empty = P.OutputBuffers(wl.n_ranks, 0, 0, 0, 0, 0, dw.device)
        with pytest.raises(P.OdbError):               # the caller drives the rounds in this mode
            P.odb_run(ctx.h, dw.lengths, wl.rank_ptr, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi,
                      empty.struct)
        with pytest.raises(P.OdbError):               # a 2048-sample budget workload with buffer_size 0: no batched exchange
            P.odb_dist_spec_form(ctx.h, dw.lengths, wl.rank_ptr, 2, 64)
        with pytest.raises(P.OdbError):
            P.odb_dist_spec_status(ctx.h, 4)          # nothing formed
        P.odb_dist_config(ctx.h, 0, 0, 0)             # back to single-process mode
        with pytest.raises(P.OdbError):
            P.odb_dist_spec_form(ctx.h, dw.lengths, wl.rank_ptr, 2, 64)
        Par.run_gpu(wl, dw, staged=False)


def test_lockstep_wide_fuzz(P, oracle):
    """120 random jobs split over 2-4 contexts (ranks with no samples, processes with no samples, quota,
    overflow, arrival schedules): every context equals the whole-job oracle."""
    import torch
    from paper_2606_19989_b200 import dist as D
    for seed in range(120):
        rng = np.random.default_rng(seed)
        n_proc = int(rng.choice([2, 3, 4]))
        rl = int(rng.integers(1, 4))
        R = n_proc * rl
        wl, sched = None, None
        for s2 in range(50):   # a generated job with exactly R ranks
            wl, sched = Par.wide_fuzz_case(1000 * seed + s2, max_ranks=12, max_n=150)
            if wl.n_ranks == R:
                break
        if wl.n_ranks != R:
            continue
        plan, ref = oracle.run_workload(wl, avail_schedule=sched)
        K = plan.n_steps
        parts = I.split_ranks(wl, n_proc)
        dws = [Par.DeviceWorkload(w) for w in parts]
        engines = [D.CudaEngine(Par.gpu_params(w), max(w.n_samples, 1), dw.lengths, w.rank_ptr) for w, dw in zip(parts, dws)]
        try:
            res = D.run_lockstep([D.plan_protocol(e, R, p * rl, None if sched is None else [row[p * rl:(p + 1) * rl] for row in sched])
                                  for p, e in enumerate(engines)])
            for p, (e, dw) in enumerate(zip(engines, dws)):
                info, round_T = res[p]
                assert round_T == plan.round_T.tolist(), seed
                assert (info.n_rounds, info.n_steps, info.stop_reason) == (plan.n_rounds, plan.n_steps, plan.stop_reason), seed
                out = P.OutputBuffers.for_plan(rl, info, dw.device, fill=Par.SENTINEL)
                e.collate(dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out)
                torch.cuda.synchronize()
                s0, s1 = p * rl * K, (p + 1) * rl * K
                off0 = int(plan.grp_offset[s0]) if s0 < plan.n_slots else plan.total_elems
                off1 = int(plan.grp_offset[s1]) if s1 < plan.n_slots else plan.total_elems
                q0, q1 = int(plan.grp_sample_ptr[s0]), int(plan.grp_sample_ptr[s1])
                assert np.array_equal(out.table("grp_count").cpu().numpy(), plan.grp_count[s0:s1]), seed
                assert np.array_equal(out.table("grp_sample_ids").cpu().numpy(), plan.grp_sample_ids[q0:q1]), seed
                assert np.array_equal(out.table("step_samples").cpu().numpy(), plan.step_samples), seed
                E = off1 - off0
                for nm in ("input_ids", "labels"):
                    assert np.array_equal(getattr(out, nm)[:E].cpu().numpy(), ref[nm][off0:off1]), (seed, nm)
        finally:
            for e in engines:
                e.close()
