"""Streaming output: odb_plan (the whole plan, no collation), odb_collate_steps (a step range of
the plan so far as a self-contained plan, double-buffered tables) and the StepStream iterator, against the oracle's
full plan and arenas."""
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


def _range_buffers(P, wl, plan, lo, hi, device):
    """Buffers exactly as large as the range needs (sized by a sizing call in the tests that check it)."""
    R, K = wl.n_ranks, plan.n_steps
    sl = (np.arange(R)[:, None] * K + np.arange(lo, hi)[None, :]).reshape(-1)
    area = plan.grp_count[sl].astype(np.int64) * plan.grp_width[sl].astype(np.int64)
    E = int(((area + 15) // 16 * 16).sum())
    return P.OutputBuffers(R, E, R * (hi - lo), int(plan.grp_count[sl].sum()), hi - lo, 0, device, fill=Par.SENTINEL)


def _workloads():
    multi = I.make_workload(1, n_ranks=3, n_per_rank=3000)
    multi.params["buffer_size"] = 512
    nj = I.protocol_workload("overflow_multiround", 2, join_mode=0)
    nj.params["sample_quota"] = int(0.6 * nj.n_samples)
    return [("tiny", I.make_workload(0)), ("multiround_512", multi), ("unequal", I.protocol_workload("unequal", 1)),
            ("empty_rank", I.protocol_workload("empty_rank", 1)), ("overflow_nonjoin_quota", nj),
            ("whole_stream_cluster", I.make_workload(1, n_ranks=2, n_per_rank=6000))]


@pytest.mark.parametrize("name,wl", _workloads(), ids=[n for n, _ in _workloads()])
def test_odb_plan_then_step_ranges(P, oracle, name, wl):
    """odb_plan gives the oracle's plan; any partition of its steps into ranges, collated range by range, gives the
    oracle's blocks; the full plan is untouched (odb_collate and the loss weights afterwards are the oracle's)."""
    import torch
    plan, ref = oracle.run_workload(wl)
    dw = Par.DeviceWorkload(wl)
    R, K = wl.n_ranks, plan.n_steps
    inputs = (dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi)
    with P.Odb(Par.gpu_params(wl), max(wl.n_samples, 1)) as ctx:
        info = P.odb_plan(ctx.h, dw.lengths, wl.rank_ptr)
        for k in Par.PLAN_SCALARS:
            assert int(getattr(info, k)) == int(getattr(plan, k)), k
        rng = np.random.default_rng(K)
        cuts = sorted(set([0, K] + rng.integers(0, K + 1, 6).tolist() + ([1, K - 1] if K > 1 else [])))
        for lo, hi in list(zip(cuts[:-1], cuts[1:])) + [(0, K), (K, K), (K // 2, K // 2)]:
            empty = P.OutputBuffers(R, 0, 0, 0, 0, 0, dw.device)
            sz = P.odb_collate_steps(ctx.h, lo, hi, *inputs, empty.struct, allow_capacity_error=True)
            out = P.OutputBuffers.for_plan(R, sz, dw.device, fill=Par.SENTINEL)
            got = P.odb_collate_steps(ctx.h, lo, hi, *inputs, out.struct)
            torch.cuda.synchronize()
            Par.compare_step_range(plan, ref, lo, hi, got, out, R)
        full = P.OutputBuffers.for_plan(R, info, dw.device, fill=Par.SENTINEL)
        P.odb_collate(ctx.h, *inputs, full.struct)
        torch.cuda.synchronize()
        Par.compare_plan(plan, info, full)
        Par.compare_full(plan, ref, info, full)
        if R * K:
            w = torch.zeros(R * K, dtype=torch.float64, device=dw.device)
            P.odb_loss_weights(ctx.h, P.ODB_SCALE_TOKEN_EXACT, w)
            want = oracle.loss_weights(P.ODB_SCALE_TOKEN_EXACT, R, K, plan.grp_count, ref["grp_valid_tokens"], plan.grp_origin)
            assert np.array_equal(w.cpu().numpy().reshape(R, K).view(np.uint64), want.view(np.uint64))


@pytest.mark.parametrize("kind", ["overflow_multiround", "unequal", "audit_bimodal"])
def test_round_by_round_streaming(P, oracle, kind):
    """The staged calls with a collate after EVERY round (odb_round_status -> odb_collate_steps over the steps that
    round emitted): each round's batches are available as soon as the round is committed, and they are the oracle's."""
    import torch
    wl = I.protocol_workload(kind, 4) if kind != "audit_bimodal" else I.protocol_workload("audit:bimodal", 4, buffer_size=32)
    plan, ref = oracle.run_workload(wl)
    dw = Par.DeviceWorkload(wl)
    R = wl.n_ranks
    inputs = (dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi)
    with P.Odb(Par.gpu_params(wl), max(wl.n_samples, 1)) as ctx:
        P.odb_reset(ctx.h)
        done, lo, rounds = 0, 0, 0
        while not done:
            P.odb_form_groups(ctx.h, dw.lengths, wl.rank_ptr)
            P.odb_align(ctx.h)
            done, T = P.odb_round_status(ctx.h)
            if T == 0:
                continue
            hi = lo + int((plan.grp_round[: plan.n_steps] == rounds).sum())  # rank 0's slots of this round
            out = _range_buffers(P, wl, plan, lo, hi, dw.device)
            got = P.odb_collate_steps(ctx.h, lo, hi, *inputs, out.struct)
            torch.cuda.synchronize()
            Par.compare_step_range(plan, ref, lo, hi, got, out, R)
            lo, rounds = hi, rounds + 1
        assert lo == plan.n_steps and rounds >= 2
        info = P.odb_plan_query(ctx.h)
        full = P.OutputBuffers.for_plan(R, info, dw.device, fill=Par.SENTINEL)
        P.odb_collate(ctx.h, *inputs, full.struct)
        torch.cuda.synchronize()
        Par.compare_plan(plan, info, full)
        Par.compare_full(plan, ref, info, full)


def test_two_ranges_in_flight_and_step_stream(P, oracle):
    """Two ranges enqueued back to back on two streams into two buffers (the library alternates between two sets
    of range tables), then the StepStream iterator over the whole plan: every batch view is the oracle's block."""
    import torch
    wl = I.make_workload(1, n_ranks=4, n_per_rank=2500)
    wl.params["buffer_size"] = 256
    plan, ref = oracle.run_workload(wl)
    dw = Par.DeviceWorkload(wl)
    R, K = wl.n_ranks, plan.n_steps
    inputs = (dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi)
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        P.odb_plan(ctx.h, dw.lengths, wl.rank_ptr)
        s0, s1 = torch.cuda.Stream(), torch.cuda.Stream()
        m = K // 2
        for _ in range(3):  # the table sets are reused
            o0, o1 = _range_buffers(P, wl, plan, 0, m, dw.device), _range_buffers(P, wl, plan, m, K, dw.device)
            torch.cuda.synchronize()
            i0 = P.odb_collate_steps(ctx.h, 0, m, *inputs, o0.struct, stream=s0.cuda_stream)
            i1 = P.odb_collate_steps(ctx.h, m, K, *inputs, o1.struct, stream=s1.cuda_stream)
            torch.cuda.synchronize()
            Par.compare_step_range(plan, ref, 0, m, i0, o0, R)
            Par.compare_step_range(plan, ref, m, K, i1, o1, R)
        chunk = 7
        stream = P.StepStream(ctx.h, R, K, wl.n_samples, inputs, chunk,
                              max(int(wl.params["budget"]), int(wl.lengths.max())), dw.device)
        seen = 0
        for c in stream:
            assert c.step_lo == seen
            for kk, step in enumerate(c):
                k = c.step_lo + kk
                for r in range(R):
                    s = r * K + k
                    cnt, wid, off = int(plan.grp_count[s]), int(plan.grp_width[s]), int(plan.grp_offset[s])
                    b = step[r]
                    if cnt == 0:
                        assert b is None
                        continue
                    for name in ("input_ids", "labels", "position_ids", "attention_mask"):
                        assert np.array_equal(b[name].cpu().numpy().reshape(-1), ref[name][off:off + cnt * wid]), (name, r, k)
                    assert b["valid_tokens"] == int(ref["grp_valid_tokens"][s])
                    assert b["step_valid_tokens"] == int(ref["step_valid_tokens"][k])
            seen += len(c)
        assert seen == K and len(stream) == (K + chunk - 1) // chunk


def test_step_stream_orders_buffer_reuse_after_async_consumer(P, oracle):
    """A consumer that reads a chunk's views with GPU work it does not wait for (a long delay kernel, then copies, on
    a stream of its own) and asks for the next chunk from that stream: the iterator must hold the overwrite of the
    handed-back buffer until those reads are done.  Every copy, checked at the very end, is the oracle's block."""
    import torch
    wl = I.make_workload(1, n_ranks=4, n_per_rank=2500)
    wl.params["buffer_size"] = 256
    plan, ref = oracle.run_workload(wl)
    dw = Par.DeviceWorkload(wl)
    R, K = wl.n_ranks, plan.n_steps
    inputs = (dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi)
    names = ("input_ids", "labels", "position_ids", "attention_mask")
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        P.odb_plan(ctx.h, dw.lengths, wl.rank_ptr)
        chunk = 5
        stream = P.StepStream(ctx.h, R, K, wl.n_samples, inputs, chunk,
                              max(int(wl.params["budget"]), int(wl.lengths.max())), dw.device)
        assert len(stream) >= 4  # buffers are reused several times
        side = torch.cuda.Stream()
        copies = []
        with torch.cuda.stream(side):  # next() is called with `side` current
            for c in stream:
                torch.cuda._sleep(30_000_000)  # ~15 ms: the next chunk's collation would long be done
                for kk, step in enumerate(c):
                    for r in range(R):
                        b = step[r]
                        if b is not None:
                            copies.append((r, c.step_lo + kk, {n: b[n].clone() for n in names}))
        torch.cuda.synchronize()
    assert len(copies) == int((plan.grp_count > 0).sum())
    for r, k, got in copies:
        s = r * K + k
        cnt, wid, off = int(plan.grp_count[s]), int(plan.grp_width[s]), int(plan.grp_offset[s])
        for n in names:
            assert np.array_equal(got[n].cpu().numpy().reshape(-1), ref[n][off:off + cnt * wid]), (n, r, k)


def _table_allocs(P, ctx):
    v = np.zeros(1, dtype=np.int64)
    assert P.odb_debug_read(ctx.h, 5, v) == 8
    return int(v[0])


def test_step_ranges_allocate_once_and_sizing_calls_keep_the_alternation(P, oracle):
    """After odb_plan the two range-table sets are sized for the whole plan when first used: ranges that grow (longer
    chunks, larger arenas) make no further cudaMalloc (the library's allocation counter stands still), and a sizing
    call before every range does not use up the other set -- two ranges, each sized first, in flight on two streams."""
    import torch
    wl = I.make_workload(1, n_ranks=4, n_per_rank=2500)
    wl.params["buffer_size"] = 256
    plan, ref = oracle.run_workload(wl)
    dw = Par.DeviceWorkload(wl)
    R, K = wl.n_ranks, plan.n_steps
    inputs = (dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi)
    empty = P.OutputBuffers(R, 0, 0, 0, 0, 0, dw.device)
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        P.odb_plan(ctx.h, dw.lengths, wl.rank_ptr)
        s0, s1 = torch.cuda.Stream(), torch.cuda.Stream()
        # first use of each set (small ranges), then growing ranges: no allocation after the first two calls
        cuts = [0, 1, 2, 5, 11, K // 2, K]
        bufs = [_range_buffers(P, wl, plan, lo, hi, dw.device) for lo, hi in zip(cuts[:-1], cuts[1:])]
        torch.cuda.synchronize()
        infos, base = [], None
        for i, (lo, hi) in enumerate(zip(cuts[:-1], cuts[1:])):
            st = (s0, s1)[i & 1]
            infos.append(P.odb_collate_steps(ctx.h, lo, hi, *inputs, bufs[i].struct, stream=st.cuda_stream))
            if i == 1:
                base = _table_allocs(P, ctx)
        assert _table_allocs(P, ctx) == base
        torch.cuda.synchronize()
        for i, (lo, hi) in enumerate(zip(cuts[:-1], cuts[1:])):
            Par.compare_step_range(plan, ref, lo, hi, infos[i], bufs[i], R)
        # sizing call + range, twice, on two streams; the first range is held back so that both are in flight
        m = K // 2
        for _ in range(2):
            outs, got = [], []
            for st, (lo, hi) in ((s0, (0, m)), (s1, (m, K))):
                with torch.cuda.stream(st):
                    torch.cuda._sleep(10_000_000 if st is s0 else 0)
                sz = P.odb_collate_steps(ctx.h, lo, hi, *inputs, empty.struct, stream=st.cuda_stream,
                                         allow_capacity_error=True)
                out = P.OutputBuffers.for_plan(R, sz, dw.device, fill=Par.SENTINEL)
                outs.append(out)
                got.append(P.odb_collate_steps(ctx.h, lo, hi, *inputs, out.struct, stream=st.cuda_stream))
            torch.cuda.synchronize()
            Par.compare_step_range(plan, ref, 0, m, got[0], outs[0], R)
            Par.compare_step_range(plan, ref, m, K, got[1], outs[1], R)
        assert _table_allocs(P, ctx) == base


def test_collate_steps_errors(P):
    import torch
    wl = I.make_workload(0)
    dw = Par.DeviceWorkload(wl)
    inputs = (dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi)
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        empty = P.OutputBuffers(wl.n_ranks, 0, 0, 0, 0, 0, dw.device)
        with pytest.raises(P.OdbError):  # nothing planned yet
            P.odb_collate_steps(ctx.h, 0, 0, *inputs, empty.struct)
        info = P.odb_plan(ctx.h, dw.lengths, wl.rank_ptr)
        for lo, hi in ((-1, 1), (2, 1), (0, info.n_steps + 1)):
            with pytest.raises(P.OdbError):
                P.odb_collate_steps(ctx.h, lo, hi, *inputs, empty.struct)
        small = P.OutputBuffers(wl.n_ranks, 16, wl.n_ranks * info.n_steps, wl.n_samples, info.n_steps, 0, dw.device,
                                fill=Par.SENTINEL)
        got = P.odb_collate_steps(ctx.h, 0, info.n_steps, *inputs, small.struct, allow_capacity_error=True)
        torch.cuda.synchronize()
        assert got.status == P.ODB_ERR_CAPACITY and got.total_elems == info.total_elems
        assert (small.input_ids.cpu().numpy().view(np.uint8) == Par.SENTINEL).all()  # nothing was written
