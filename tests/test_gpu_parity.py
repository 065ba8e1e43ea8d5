"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit, on the same
seeded inputs.  Everything on this path is integer / index work, so the bar is exact equality
(BASELINE.json north_star).  Run on the B200 box: ``pytest -m gpu``."""
import numpy as np
import pytest

import odb_inputs as I
from tests import _parity as Par

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box (there is no CPU fallback)")
    import paper_2606_19989_b200 as P
    P.load()
    return P


def _full_parity(oracle, wl, staged=True):
    plan, ref = oracle.run_workload(wl)
    info, out, round_T = Par.run_gpu(wl, staged=staged)
    Par.compare_plan(plan, info, out, round_T)
    Par.compare_full(plan, ref, info, out)
    return plan, info, out


# ---- input generator: the device token fill equals the host specification ---------------------
def test_synth_tokens_match_host_hash(P):
    import torch
    n = 100_003
    for seed, start in ((0, 0), (4, 2_000_000_000), (7001, 12345)):
        d = torch.empty(n, dtype=torch.int32, device="cuda:0")
        P.odb_synth_tokens(d, start, n, seed, I.VOCAB)
        torch.cuda.synchronize()
        assert np.array_equal(d.cpu().numpy(), I.token_ids(seed, start, n))


# ---- BASELINE.json configs --------------------------------------------------------------------
@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("staged", [True, False])
def test_config1_tiny(P, oracle, rule, staged):
    wl = I.make_workload(0, rule=rule)
    plan, info, out = _full_parity(oracle, wl, staged=staged)
    assert plan.n_rounds == 2 and plan.samples_emitted == 128


@pytest.mark.parametrize("rule", [0, 1])
def test_config2_lowcv_text(P, oracle, rule):
    _full_parity(oracle, I.make_workload(1, rule=rule))


@pytest.mark.parametrize("rule", [0, 1])
def test_config3_multimodal(P, oracle, rule):
    _full_parity(oracle, I.make_workload(2, rule=rule))


def _sampled_parity(oracle, wl, n_sample=48, seed=0):
    """Full-size run in the launch configuration bench.py times (odb_run, one collate launch over the
    whole arena); plan tables compared in full, blocks compared on sampled slots, plus
    any-size properties recomputed on the device."""
    plan, _ = oracle.run_workload(wl, collate=False)
    info, out, _ = Par.run_gpu(wl, staged=False)
    Par.compare_plan(plan, info, out)
    rng = np.random.default_rng(seed)
    n_slots = plan.n_slots
    area = plan.grp_count.astype(np.int64) * plan.grp_width
    pick = set(rng.integers(0, n_slots, n_sample).tolist())
    pick |= {0, n_slots - 1, int(np.argmax(area)), int(np.argmax(plan.grp_width)), int(np.argmax(plan.grp_count))}
    pick |= set(np.flatnonzero(plan.grp_count == 1)[:4].tolist())          # singletons (splits / over-budget)
    # keep the host-side token regeneration bounded
    pick = [s for s in sorted(pick) if area[s] <= 6_000_000][: n_sample + 8]
    Par.compare_sampled_slots(wl, plan, out, pick)
    Par.device_self_consistency(info, out, wl.params["ignore_index"])
    return plan


def _full_size_elementwise(oracle, wl):
    """Full-size run in the launch configuration bench.py times (odb_run, one collate launch over the whole
    arena): plan tables in full, then ALL FOUR ARENAS OVER EVERY SLOT against the oracle, rank by rank."""
    plan, _ = oracle.run_workload(wl, collate=False)
    info, out, _ = Par.run_gpu(wl, staged=False)
    Par.compare_plan(plan, info, out)
    Par.compare_full_by_rank(oracle, wl, plan, out)
    return plan


@pytest.mark.parametrize("rule,join", [(0, 1), (0, 0), (1, 1)])
def test_config4_full_size_every_element(P, oracle, rule, join):
    """BASELINE.json configs[3] (16 x 16384, high-CV long tail) at full size, join and non-join (quota cut):
    every element of input_ids / labels / position_ids / attention_mask of every slot."""
    wl = I.make_workload(3, rule=rule, join_mode=join)
    plan = _full_size_elementwise(oracle, wl)
    if not join:
        assert plan.stop_reason == 2 and plan.samples_left > 0


@pytest.mark.parametrize("cv,budget,rule", [(1.0, 65536, 0), (2.5, 16384, 0), (0.3, 262144, 0), (1.0, 65536, 1)])
def test_config5_full_size_every_element(P, oracle, cv, budget, rule):
    """BASELINE.json configs[4] at full size (32 x 32768 samples, 2.1e9 tokens, 28 GB of outputs; element offsets
    exceed 2^31): the cell bench.py is quoted on (CV 1.0 / L 65536) and the CV 2.5 / L 16384 cell (over-budget
    singletons of up to ~270 K tokens), every element of every slot, rank by rank."""
    plan = _full_size_elementwise(oracle, I.make_workload(4, cv=cv, budget=budget, rule=rule))
    assert plan.total_elems > 2**31


def test_config5_full_size_paper_operating_point(P, oracle):
    """The exact job bench.py times as `paper_operating_point` and `streaming`: BASELINE.json configs[4] (CV 1.0 /
    L 65536) with the paper's 1024-sample grouping buffer -- 33 protocol rounds, 1024 (rank, round) windows
    through the round-parallel planner -- at full size: plan tables in full, every element of every slot."""
    wl = I.make_workload(4, cv=1.0, budget=65536)
    wl.params["buffer_size"] = 1024
    plan = _full_size_elementwise(oracle, wl)
    assert plan.n_rounds == 33 and plan.total_elems > 2**31


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("join", [1, 0])
def test_config4_highcv_longtail(P, oracle, rule, join):
    wl = I.make_workload(3, rule=rule, join_mode=join)
    plan = _sampled_parity(oracle, wl)
    if not join:
        Q = wl.params["sample_quota"]
        assert plan.stop_reason == 2 and Q <= plan.samples_emitted <= Q + int(plan.step_samples.max())


@pytest.mark.parametrize("cv,budget", I.config5_cells())
def test_config5_sweep_cells(P, oracle, cv, budget):
    """All nine (CV, budget) cells of BASELINE.json configs[4] at full size (32 x 32768 samples, ~2.1e9 tokens)."""
    _sampled_parity(oracle, I.make_workload(4, cv=cv, budget=budget), n_sample=24)


@pytest.mark.parametrize("cv,budget", [(1.0, 65536), (2.5, 16384), (0.3, 262144)])
def test_config5_maxfit(P, oracle, cv, budget):
    _sampled_parity(oracle, I.make_workload(4, cv=cv, budget=budget, rule=1), n_sample=16)


# ---- protocol tests (multi-round, overflow, IDLE, empty ranks, quota) --------------------------
@pytest.mark.parametrize("kind", ["audit:" + k for k in I.AUDIT_KINDS] + ["overflow_multiround", "empty_rank", "unequal"])
@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("join", [1, 0])
def test_protocol(P, oracle, kind, rule, join):
    over = dict(rule=rule, join_mode=join)
    wl = I.protocol_workload(kind, 0, **over)
    if not join:
        wl.params["sample_quota"] = int(0.6 * wl.n_samples)
    _full_parity(oracle, wl)


@pytest.mark.parametrize("kind", ["audit:" + k for k in I.AUDIT_KINDS])
def test_protocol_audit_whole_window(P, oracle, kind):
    """The audit distributions with the buffer holding the whole stream (buffer 1000)."""
    _full_parity(oracle, I.protocol_workload(kind, 1, buffer_size=1000))


def test_protocol_fuzz(P, oracle):
    for seed in range(500):
        wl = I.protocol_workload("fuzz", seed)
        try:
            _full_parity(oracle, wl, staged=bool(seed & 1))
        except AssertionError as e:
            raise AssertionError("fuzz seed %d params %r: %s" % (seed, wl.params, e))


def test_many_spans_slow_path(P, oracle):
    """Samples with more than two masked spans take the kernel's CSR span path."""
    rng = np.random.default_rng(5)
    wl = I.protocol_workload("unequal", 3)
    N = wl.n_samples
    lo, hi, ptr = [], [], [0]
    for g in range(N):
        L = int(wl.lengths[g])
        k = int(rng.integers(0, 6))
        cuts = np.sort(rng.choice(np.arange(L + 1), size=min(2 * k, L + 1), replace=False))
        cuts = cuts[: len(cuts) // 2 * 2]
        for a, b in zip(cuts[0::2], cuts[1::2]):
            lo.append(a)
            hi.append(b)
        ptr.append(len(lo))
    wl.span_ptr = np.asarray(ptr, np.int64)
    wl.span_lo = np.asarray(lo, np.int32)
    wl.span_hi = np.asarray(hi, np.int32)
    for shift in (1, 0):
        wl.params["shift_labels"] = shift
        _full_parity(oracle, wl)


# ---- degenerate cases ------------------------------------------------------
def test_degenerate_cases(P, oracle):
    # R = 1: alignment is a no-op
    wl = I.make_workload(0, n_ranks=1)
    _full_parity(oracle, wl)
    # budget below every length: all over-budget singletons
    wl = I.make_workload(0, budget=4)
    plan, _, _ = _full_parity(oracle, wl)
    assert (plan.grp_count[plan.grp_count > 0] == 1).all()
    # huge budget: THRESHOLD gives the longest sample alone + everything else
    wl = I.make_workload(0, budget=1 << 30)
    plan, _, _ = _full_parity(oracle, wl)
    assert plan.n_steps == 2
    # all ranks empty
    wl = I.make_workload(0, n_per_rank=0)
    plan, info, out = _full_parity(oracle, wl)
    assert info.n_steps == 0 and info.total_elems == 0 and info.stop_reason == 0


@pytest.mark.parametrize("rule", [0, 1])
def test_large_window_global_memory_planner(P, oracle, rule):
    """A window of more than ~56 K samples does not fit the shared-memory list-ranking kernel: the
    global-memory version runs (rank 0), next to ranks that split heavily to reach its group count."""
    wl = I.make_workload(0, n_ranks=3, n_per_rank=70_000, budget=1024, rule=rule)
    plan = _sampled_parity(oracle, wl, n_sample=24)
    assert plan.n_steps > 1000 and wl.n_samples == 210_000


@pytest.mark.parametrize("n", [4096, 4097, 9000, 20_000, 32_768, 33_000, 50_000, 65_536])
@pytest.mark.parametrize("rule", [0, 1])
def test_cluster_sort_window_sizes(P, oracle, n, rule):
    """Windows that need a thread-block cluster of 1, 2, 4, 8 and 16 CTAs for the segmented sort (ragged last
    chunks, a rank with a much smaller window beside them), and both list-ranking kernels behind it."""
    rng = np.random.default_rng(n + rule)
    per = [rng.integers(1, 3000, n), rng.integers(1, 3000, max(1, n // 3)), rng.integers(1, 40, n - 5)]
    wl = I.custom_workload("cluster_sort", per, 31, budget=8192, rule=rule)
    plan = _sampled_parity(oracle, wl, n_sample=16)
    assert plan.samples_emitted == wl.n_samples


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("join", [1, 0])
def test_paper_operating_point_buffer_1024(P, oracle, rule, join):
    """The paper's operating point: a 1024-sample grouping buffer per rank, tens of protocol rounds per
    rank stream -- through odb_run, i.e. the persistent round-loop kernel (one launch for every round) --
    on the configs[3] recipe (16 ranks x 16384 samples, high-CV long tail): plan tables in full, every element
    of every slot."""
    wl = I.make_workload(3, rule=rule, join_mode=join)
    wl.params["buffer_size"] = 1024
    plan = _full_size_elementwise(oracle, wl)
    assert plan.n_rounds >= 16


@pytest.mark.parametrize("buffer_size,slot_capacity", [(4096, 0), (1000, 7), (333, 0), (64, 3)])
def test_round_loop_kernel_windows(P, oracle, buffer_size, slot_capacity):
    """Persistent round-loop kernel: full 4096-key windows, ragged windows, overflow + recirculation through
    finite slot capacity, unequal streams (IDLE slots while other ranks continue), both modes with a quota."""
    rng = np.random.default_rng(buffer_size)
    per = [rng.integers(1, 2000, 9000), rng.integers(1, 300, 5000), rng.integers(500, 4000, 2500), np.zeros(0, np.int64)]
    for join in (1, 0):
        wl = I.custom_workload("round_loop", per[: 3 + join], 41, budget=8192, buffer_size=buffer_size,
                               slot_capacity=slot_capacity, join_mode=join)
        if not join:
            wl.params["sample_quota"] = int(0.7 * wl.n_samples)
        plan, _ = oracle.run_workload(wl, collate=False)
        info, out, _ = Par.run_gpu(wl, staged=False)
        Par.compare_plan(plan, info, out)
        Par.compare_full_by_rank(oracle, wl, plan, out)
        # and the staged API (host-driven rounds) gives the same plan
        info2, out2, _ = Par.run_gpu(wl, staged=True)
        Par.compare_plan(plan, info2, out2)


def _stream_lengths(rng, n, hi=3000):
    return rng.integers(1, hi, n)


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("case", ["equal", "ragged_tail", "short_rank", "nonjoin", "nonjoin_quota", "capacity", "tiny_buffer",
                                  "full_chunk"])
def test_round_parallel_planner(P, oracle, case, rule):
    """The round-parallel planner (k_spec_form / k_spec_commit, ODB_OPT_ROUND_PARALLEL): every round that starts
    without leftovers is formed at once, the sequential loop resumes at the first round that overflows.  Equal
    streams (the whole run is round-parallel), ragged tails (the last windows differ: S+min caps T, the tail is
    sequential), a rank that finishes early (IDLE slots beside round-parallel rounds), non-join without a quota
    (the terminal round is the first in which a stream is drained), finite slot capacity (overflow in round 0:
    nothing is committed round-parallel), non-join with a sample quota (the rounds below the quota are round-parallel,
    the round that reaches it and its cut are the loop's), an 8-sample buffer and full 4096-key windows.  Plan tables in full and
    every element of every slot against the oracle; the sequential loop (option off) gives the same."""
    rng = np.random.default_rng(7 + rule)
    kw = dict(budget=8192, rule=rule, join_mode=1)
    if case == "equal":
        per, kw["buffer_size"] = [_stream_lengths(rng, 6000) for _ in range(5)], 500
        expect = ("all", 12)
    elif case == "ragged_tail":
        per, kw["buffer_size"] = [_stream_lengths(rng, n) for n in (5000, 5013, 4990, 5100)], 1000
        expect = ("some", None)  # (4 or 5 rounds: the 13-sample window of the last round caps T below the others' counts)
    elif case == "short_rank":
        per, kw["buffer_size"] = [_stream_lengths(rng, n) for n in (4096, 1024, 4096, 0)], 1024
        expect = ("all", 4)
    elif case == "nonjoin":
        per, kw["buffer_size"], kw["join_mode"] = [_stream_lengths(rng, n) for n in (3000, 2048, 2600)], 256, 0
        expect = ("all", 8)
    elif case == "nonjoin_quota":   # 768 samples per round: the sixth round reaches the quota, the cut is the loop's
        per, kw["buffer_size"], kw["join_mode"] = [_stream_lengths(rng, n) for n in (3000, 2048, 2600)], 256, 0
        kw["sample_quota"] = 4000
        expect = ("quota", 5)
    elif case == "capacity":
        per, kw["buffer_size"], kw["slot_capacity"] = [_stream_lengths(rng, 3000, 200) for _ in range(3)], 512, 3
        expect = ("some", 0)
    elif case == "tiny_buffer":
        per, kw["buffer_size"] = [_stream_lengths(rng, 400, 9000) for _ in range(6)], 8
        expect = ("all", 50)
    else:
        per, kw["buffer_size"] = [_stream_lengths(rng, 3 * 4096) for _ in range(3)], 4096
        expect = ("all", 3)
    wl = I.custom_workload("round_parallel_" + case, per, 77, **kw)
    plan, _ = oracle.run_workload(wl, collate=False)
    rec = []
    info, out, _ = Par.run_gpu(wl, staged=False, spec_rec=rec)
    Par.compare_plan(plan, info, out)
    Par.compare_full_by_rank(oracle, wl, plan, out)
    assert rec[0] is not None, "the round-parallel planner did not run"
    committed, steps, ended = int(rec[0][0]), int(rec[0][1]), int(rec[0][2])
    if expect[0] == "all":
        assert ended == 1 and committed == expect[1] == plan.n_rounds - 1 and steps == plan.n_steps
    elif expect[0] == "quota":
        assert ended == 0 and committed == expect[1] == plan.n_rounds - 1 and plan.stop_reason == 2 and steps < plan.n_steps
    else:
        assert ended == 0 and committed < plan.n_rounds - 1
        assert committed == expect[1] if expect[1] is not None else committed >= 4
    # the sequential loop alone
    rec2 = []
    info2, out2, _ = Par.run_gpu(wl, staged=False, options={P.ODB_OPT_ROUND_PARALLEL: 0}, spec_rec=rec2)
    assert rec2[0] is None
    Par.compare_plan(plan, info2, out2)


def test_round_parallel_planner_fuzz(P, oracle):
    """120 random jobs in the round-parallel planner's regime (grouping buffers of 8 .. 700 samples, up to 12 ranks
    with unequal streams of up to 4000 samples, both rules, join and non-join with and without a quota, finite slot
    capacity in a third of them): the plan tables in full and sampled slots element by element against the oracle.  The planner
    must have run, and the rounds it committed never exceed the plan's."""
    used = 0
    for seed in range(120):
        rng = np.random.default_rng(31_000 + seed)
        R = int(rng.integers(1, 13))
        hi = int(rng.choice([40, 600, 5000]))
        n_max = int(rng.choice([60, 900, 4000]))
        equal = rng.uniform() < 0.4
        n0 = int(rng.integers(n_max // 2, n_max + 1))
        per = [rng.integers(1, hi + 1, n0 if equal else int(rng.integers(0, n_max + 1))) for _ in range(R)]
        B = int(rng.choice([8, 9, 31, 64, 128, 257, 700]))
        wl = I.custom_workload("rp_fuzz", per, seed, budget=int(rng.choice([64, 1024, 8192, 60000])), buffer_size=B,
                               slot_capacity=int(rng.choice([0, 0, 5, 40])), rule=int(rng.integers(0, 2)),
                               join_mode=int(rng.integers(0, 2)), shift_labels=int(rng.integers(0, 2)))
        if not wl.params["join_mode"] and rng.uniform() < 0.5:
            wl.params["sample_quota"] = int(rng.integers(1, max(2, wl.n_samples + 1)))
            wl.params["emitted_so_far"] = int(rng.choice([0, 0, 17]))
        plan, _ = oracle.run_workload(wl, collate=False)
        rec = []
        info, out, _ = Par.run_gpu(wl, staged=False, spec_rec=rec)
        Par.compare_plan(plan, info, out)
        if plan.n_slots:
            pick = sorted(set(rng.integers(0, plan.n_slots, 6).tolist()) | {0, plan.n_slots - 1})
            Par.compare_sampled_slots(wl, plan, out, pick)
        if rec[0] is not None:
            used += 1
            assert 0 <= int(rec[0][0]) <= plan.n_rounds - 1 and int(rec[0][1]) <= plan.n_steps
            if plan.stop_reason != 2:   # (a quota stop is never the planner's: the cut belongs to the loop)
                assert (int(rec[0][2]) == 1) == (int(rec[0][0]) == plan.n_rounds - 1)
            else:
                assert int(rec[0][2]) == 0
    assert used >= 60


def test_run_host_with_small_grouping_buffer(P, oracle):
    """odb_run_host plans on the device too (round-parallel planner + round loop, no per-round host round trip)."""
    wl = I.make_workload(1, n_ranks=4, n_per_rank=2500)
    wl.params["buffer_size"] = 256
    _run_host_case(P, oracle, wl, staging_elems=1 << 16)
    wl = I.custom_workload("run_host_ragged", [np.arange(1, 1500) % 900 + 1, np.arange(1, 900) % 50 + 1], 3, budget=4096,
                           buffer_size=100, join_mode=0)
    _run_host_case(P, oracle, wl)


@pytest.mark.parametrize("staged", [True, False])
def test_collate_bulk_store_variant(P, oracle, staged):
    """ODB_OPT_COLLATE_BULK_STORES: the interior chunks leave through shared memory and bulk asynchronous stores
    instead of 256-bit register stores -- the same bytes (configs[1], configs[2] in both label modes, the
    many-span path, fuzz)."""
    for wl in (I.make_workload(1), I.make_workload(2), I.make_workload(2, rule=1), I.protocol_workload("unequal", 4)):
        for shift in (1, 0):
            wl.params["shift_labels"] = shift
            plan, ref = oracle.run_workload(wl)
            info, out, _ = Par.run_gpu(wl, staged=staged, bulk_stores=True)
            Par.compare_plan(plan, info, out)
            Par.compare_full(plan, ref, info, out)
    for seed in range(60):
        wl, sched = Par.wide_fuzz_case(seed)
        plan, ref = oracle.run_workload(wl)
        info, out, _ = Par.run_gpu(wl, staged=staged, bulk_stores=True)
        Par.compare_plan(plan, info, out)
        Par.compare_full(plan, ref, info, out)


def test_bandwidth_probes_run(P):
    """The mix-ceiling probes of bench.py: every kind runs, and the stores land where they should."""
    import torch
    n = 1 << 22
    src = torch.arange(n, dtype=torch.int32, device="cuda:0")
    o = [torch.full((n,), -1, dtype=torch.int32, device="cuda:0") for _ in range(3)]
    m = torch.full((n,), 7, dtype=torch.uint8, device="cuda:0")
    for kind in range(5):
        for t in o:
            t.fill_(-1)
        ms = P.odb_probe_bandwidth(kind, src, o[0], o[1], o[2], m, n, reps=2)
        torch.cuda.synchronize()
        assert ms > 0
        if kind in (0, 1, 4):
            assert torch.equal(o[0], src)
        if kind in (0, 1):
            assert torch.equal(o[1], src ^ 0x55)


def test_heavy_split_unequal_group_counts(P, oracle):
    """One rank forms thousands of groups, another a handful of big ones: the split closed form turns
    thousands of rows of a few groups into singletons (Alg. 1)."""
    rng = np.random.default_rng(11)
    a = rng.integers(900, 1024, 6000)          # ~1 sample per group at budget 1024
    b = rng.integers(1, 4, 6000)               # hundreds of samples per group
    c = rng.integers(1, 1024, 6000)
    wl = I.custom_workload("heavy_split", [a, b, c], 17, budget=1024, rule=0, join_mode=1)
    plan, info, out = _full_parity(oracle, wl)
    assert plan.n_steps >= 5000


def test_bad_length_is_reported(P):
    import torch
    wl = I.make_workload(0)
    wl.lengths = wl.lengths.copy()
    wl.lengths[17] = 0
    dw_len = torch.from_numpy(wl.lengths).to("cuda:0")
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        with pytest.raises(P.OdbError) as ei:
            ctx.plan(dw_len, wl.rank_ptr)
        assert ei.value.status == P.ODB_ERR_BAD_LENGTH


def test_capacity_and_state_errors(P):
    wl = I.make_workload(0)
    dw = Par.DeviceWorkload(wl)
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        with pytest.raises(P.OdbError) as ei:
            P.odb_align(ctx.h)                      # nothing formed yet
        assert ei.value.status == P.ODB_ERR_STATE
        info = ctx.plan(dw.lengths, wl.rank_ptr)
        small = P.OutputBuffers(wl.n_ranks, info.total_elems - 16, info.n_slots, info.samples_emitted, info.n_steps,
                                info.samples_left, "cuda:0", fill=Par.SENTINEL)
        with pytest.raises(P.OdbError) as ei:
            P.odb_collate(ctx.h, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, small.struct)
        assert ei.value.status == P.ODB_ERR_CAPACITY
        import torch
        torch.cuda.synchronize()
        assert (small.attention_mask.cpu().numpy() == Par.SENTINEL).all()   # nothing written


def test_run_to_run_determinism(P):
    import torch
    wl = I.make_workload(1)
    dw = Par.DeviceWorkload(wl)
    a_info, a, _ = Par.run_gpu(wl, dw, staged=False)
    b_info, b, _ = Par.run_gpu(wl, dw, staged=False)
    for name in ("input_ids", "labels", "position_ids", "attention_mask"):
        assert torch.equal(getattr(a, name), getattr(b, name))
    for name in ("grp_valid_tokens", "step_valid_tokens", "grp_sample_ids"):
        assert torch.equal(a.table(name), b.table(name))


def _run_host_case(P, oracle, wl, ctx=None, staging_elems=None):
    import torch
    plan, ref = oracle.run_workload(wl)
    toks_np = wl.tokens()
    toks = torch.from_numpy(toks_np if len(toks_np) else np.zeros(1, np.int32)).pin_memory()
    pin = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a) if len(a) else np.zeros(1, a.dtype)).to(dt).pin_memory()
    own = ctx is None
    ctx = ctx or P.Odb(Par.gpu_params(wl), max(wl.n_samples, 1))
    if staging_elems:
        P.odb_set_option(ctx.h, P.ODB_OPT_HOST_STAGING_ELEMS, staging_elems)
    try:
        out = P.OutputBuffers(wl.n_ranks, plan.total_elems, plan.n_slots, plan.samples_emitted, plan.n_steps,
                              plan.samples_left, "cpu", fill=Par.SENTINEL)
        info = P.odb_run_host(ctx.h, pin(wl.lengths, torch.int32), wl.rank_ptr, toks, pin(wl.sample_ptr, torch.int64),
                              pin(wl.span_ptr, torch.int64), pin(wl.span_lo, torch.int32), pin(wl.span_hi, torch.int32),
                              out.struct)
    finally:
        if own:
            ctx.close()
    Par.compare_plan(plan, info, out)
    E = plan.total_elems
    # each rank's slice of an arena is one flat memcpy, so gap bytes carry whatever the device
    # staging held; compare blocks only
    inblk = np.zeros(E, dtype=bool)
    for s in range(plan.n_slots):
        o = int(plan.grp_offset[s])
        inblk[o:o + int(plan.grp_count[s]) * int(plan.grp_width[s])] = True
    for name in ("input_ids", "labels", "position_ids", "attention_mask"):
        assert np.array_equal(getattr(out, name)[:E].numpy()[inblk], ref[name][:E][inblk]), name
        tail = getattr(out, name)[E:].numpy().view(np.uint8)
        assert (tail == Par.SENTINEL).all(), name + ": wrote past total_elems"
    assert np.array_equal(out.table("grp_valid_tokens").numpy(), ref["grp_valid_tokens"])
    assert np.array_equal(out.table("step_valid_tokens").numpy(), ref["step_valid_tokens"])


@pytest.mark.parametrize("case", ["config2", "tiny", "tiny_maxfit", "unequal", "empty_rank", "overflow_nonjoin",
                                  "config4_slice_nonjoin"])
def test_run_host_end_to_end(P, oracle, case):
    """odb_run_host: HOST buffers in, HOST buffers out (the e2e leg bench.py times).  Tokens go up
    and results come back rank by rank, one collate launch per rank: rank boundaries fall inside
    collate tiles and chunks, some ranks own no slot elements at all."""
    if case == "config2":
        wl = I.make_workload(1)
    elif case == "tiny":
        wl = I.make_workload(0)
    elif case == "tiny_maxfit":
        wl = I.make_workload(0, rule=1)
    elif case == "overflow_nonjoin":
        wl = I.protocol_workload("overflow_multiround", 1, join_mode=0)
        wl.params["sample_quota"] = int(0.6 * wl.n_samples)
    elif case == "config4_slice_nonjoin":
        wl = I.make_workload(3, n_ranks=5, n_per_rank=700, join_mode=0)
    else:
        wl = I.protocol_workload(case, 2)
    _run_host_case(P, oracle, wl)


@pytest.mark.parametrize("staging", [4096, 8192, 40_000, 1 << 20])
def test_run_host_streams_through_fixed_size_staging(P, oracle, staging):
    """The arenas are far larger than the device staging of odb_run_host (three pieces of `staging` elements; the
    tokens go through a ring of three rank-sized buffers): 8 ranks -> the token ring wraps, hundreds of pieces."""
    _run_host_case(P, oracle, I.make_workload(1), staging_elems=staging)
    wl = I.protocol_workload("overflow_multiround", 5, join_mode=0)
    wl.params["sample_quota"] = int(0.7 * wl.n_samples)
    _run_host_case(P, oracle, wl, staging_elems=staging)
    _run_host_case(P, oracle, I.protocol_workload("empty_rank", 2), staging_elems=staging)


def test_run_host_device_arenas(P, oracle):
    """ODB_OPT_HOST_DEVICE_ARENAS: host inputs, the four arenas stay on the device (collated in place, rank by rank, as
    the tokens land), the tables come back to the host -- every element against the oracle, gaps untouched."""
    import torch
    for wl in (I.make_workload(1, n_ranks=5, n_per_rank=900), I.protocol_workload("empty_rank", 3),
               I.protocol_workload("overflow_multiround", 2)):
        plan, ref = oracle.run_workload(wl)
        toks_np = wl.tokens()
        toks = torch.from_numpy(toks_np if len(toks_np) else np.zeros(1, np.int32)).pin_memory()
        pin = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a) if len(a) else np.zeros(1, a.dtype)).to(dt).pin_memory()
        host = P.OutputBuffers(wl.n_ranks, 0, plan.n_slots, plan.samples_emitted, plan.n_steps, plan.samples_left, "cpu")
        dev = P.OutputBuffers(wl.n_ranks, plan.total_elems, 0, 0, 0, 0, "cuda:0", fill=Par.SENTINEL, tables=False)
        st = host.struct
        st.d_input_ids, st.d_labels = dev.struct.d_input_ids, dev.struct.d_labels
        st.d_position_ids, st.d_attention_mask = dev.struct.d_position_ids, dev.struct.d_attention_mask
        st.arena_capacity = plan.total_elems
        with P.Odb(Par.gpu_params(wl), max(wl.n_samples, 1)) as ctx:
            P.odb_set_option(ctx.h, P.ODB_OPT_HOST_DEVICE_ARENAS, 1)
            info = P.odb_run_host(ctx.h, pin(wl.lengths, torch.int32), wl.rank_ptr, toks, pin(wl.sample_ptr, torch.int64),
                                  pin(wl.span_ptr, torch.int64), pin(wl.span_lo, torch.int32), pin(wl.span_hi, torch.int32), st)
        Par.compare_plan(plan, info, host)
        host.input_ids, host.labels, host.position_ids, host.attention_mask = (dev.input_ids, dev.labels, dev.position_ids,
                                                                               dev.attention_mask)
        Par.compare_full(plan, ref, info, host)


def test_context_reused_across_different_jobs(P, oracle):
    """One context, several jobs back to back on one stream: different rank boundaries (the library uploads them only
    when they changed), the same boundaries again, an arrival schedule in between (the device's arrival counts must
    follow), a job with a bad length (the status record is cleared by the previous plan's slot scan, not by a
    clearing pass: the error must neither stick nor get lost), odb_run and the staged calls mixed."""
    import torch
    rng = np.random.default_rng(5)
    mk = lambda ns, seed, **kw: I.custom_workload("reuse", [rng.integers(1, 900, n) for n in ns], seed, budget=4096, **kw)
    jobs = [mk((300, 200, 100), 1), mk((100, 300, 200), 2), mk((50, 0, 550), 4), mk((300, 200, 100), 5)]
    prm = Par.gpu_params(jobs[0])
    with P.Odb(prm, 600) as ctx:
        def run(wl, staged, sched=None):
            assert wl.params["budget"] == 4096
            dw = Par.DeviceWorkload(wl)
            plan, ref = oracle.run_workload(wl, avail_schedule=sched)
            if staged:
                info = ctx.plan(dw.lengths, wl.rank_ptr, avail_schedule=sched)
                out = P.OutputBuffers.for_plan(wl.n_ranks, info, dw.device, fill=Par.SENTINEL)
                P.odb_collate(ctx.h, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out.struct)
            else:
                out = P.OutputBuffers(wl.n_ranks, plan.total_elems, plan.n_slots, plan.samples_emitted, plan.n_steps,
                                      plan.samples_left, dw.device, fill=Par.SENTINEL)
                info = P.odb_run(ctx.h, dw.lengths, wl.rank_ptr, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo,
                                 dw.span_hi, out.struct)
            torch.cuda.synchronize()
            Par.compare_plan(plan, info, out)
            Par.compare_full(plan, ref, info, out)

        whole = jobs
        for wl in whole + whole[::-1]:                      # same parameters as the context: boundaries change and return
            run(wl, staged=False)
            run(wl, staged=True)
        from tests.test_oracle_arrival import _random_schedule
        sched = _random_schedule(np.random.default_rng(9), whole[0], 5)
        run(whole[0], staged=True, sched=sched)            # arrival counts on the device ...
        run(whole[0], staged=False)                        # ... and "everything has arrived" again
        bad = Par.DeviceWorkload(whole[1])
        bad.lengths[7] = 0
        torch.cuda.synchronize()
        empty = P.OutputBuffers(whole[1].n_ranks, 0, 0, 0, 0, 0, bad.device)
        for _ in range(2):                                  # reported every time, not only once
            with pytest.raises(P.OdbError) as ei:
                P.odb_run(ctx.h, bad.lengths, whole[1].rank_ptr, bad.tokens, bad.sample_ptr, bad.span_ptr, bad.span_lo,
                          bad.span_hi, empty.struct)
            assert ei.value.status == P.ODB_ERR_BAD_LENGTH
        run(whole[1], staged=False)                         # and it does not stick
        run(whole[2], staged=True)


def test_run_host_reuses_context(P, oracle):
    """Two odb_run_host calls on one context (staging buffers, events and counters are reused)."""
    wl = I.make_workload(1, n_ranks=3, n_per_rank=300)
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        _run_host_case(P, oracle, wl, ctx)
        _run_host_case(P, oracle, wl, ctx)


# ---- loss-scaling weights --------------------------------------------------
@pytest.mark.parametrize("case", ["tiny", "config2", "unequal", "empty_rank", "overflow_multiround",
                                  "config4_slice_nonjoin", "heavy_split"])
def test_loss_weights_bit_exact(P, oracle, case):
    """odb_loss_weights vs the oracle, all three modes (Eq. 2; App. B).
    Tolerance: ZERO ulps in fp64 -- both sides perform the same sequence of single correctly rounded
    IEEE operations (int -> double conversions are exact below 2^53, one division for tbar, one
    product, a left-to-right sum over ranks, one division; no FMA contraction on either side)."""
    import torch
    if case == "tiny":
        wl = I.make_workload(0)
    elif case == "config2":
        wl = I.make_workload(1)
    elif case == "config4_slice_nonjoin":
        wl = I.make_workload(3, n_ranks=5, n_per_rank=700, join_mode=0)
    elif case == "heavy_split":
        rng = np.random.default_rng(11)
        wl = I.custom_workload("heavy_split", [rng.integers(8, 64, size=40), rng.integers(900, 1000, size=300),
                                               rng.integers(8, 2000, size=200)], seed=5, budget=4096)
    else:
        wl = I.protocol_workload(case, 6)
    plan, ref = oracle.run_workload(wl)
    dw = Par.DeviceWorkload(wl)
    R, K = wl.n_ranks, plan.n_steps
    with P.Odb(Par.gpu_params(wl), max(wl.n_samples, 1)) as ctx:
        info = ctx.plan(dw.lengths, wl.rank_ptr)
        out = P.OutputBuffers.for_plan(R, info, dw.device)
        w = torch.full((max(R * K, 1),), float("nan"), dtype=torch.float64, device=dw.device)
        with pytest.raises(P.OdbError):  # no collate yet: no valid-token counts
            P.odb_loss_weights(ctx.h, P.ODB_SCALE_TOKEN_EXACT, w)
        P.odb_collate(ctx.h, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out.struct)
        assert np.array_equal(out.table("grp_origin").cpu().numpy(), plan.grp_origin)
        for mode in (P.ODB_SCALE_SAMPLE, P.ODB_SCALE_TOKEN_APPROX, P.ODB_SCALE_TOKEN_EXACT):
            w.fill_(float("nan"))
            P.odb_loss_weights(ctx.h, mode, w)
            torch.cuda.synchronize()
            want = oracle.loss_weights(mode, R, K, plan.grp_count, ref["grp_valid_tokens"], plan.grp_origin)
            got = w[:R * K].cpu().numpy().reshape(R, K)
            assert np.array_equal(got.view(np.uint64), want.view(np.uint64)), (case, mode, np.abs(got - want).max())
        with pytest.raises(P.OdbError):
            P.odb_loss_weights(ctx.h, 7, w)


def test_step_batches_views(P, oracle):
    """StepBatches: zero-copy [count, width] views per step and rank, IDLE slots skipped, against
    the oracle's per-slot collation; the join-mode identity contract seen through the iterator (Thm 1)."""
    import torch
    wl = I.protocol_workload("empty_rank", 3)
    plan, ref = oracle.run_workload(wl)
    dw = Par.DeviceWorkload(wl)
    info, out, _ = Par.run_gpu(wl, dw, staged=False)
    sb = P.StepBatches(out, info, wl.n_ranks)
    assert len(sb) == plan.n_steps
    toks = wl.tokens()
    seen = [[] for _ in range(wl.n_ranks)]
    n_idle = 0
    for k, step in enumerate(sb):
        assert len(step) == wl.n_ranks
        for r, b in enumerate(step):
            s = r * plan.n_steps + k
            if plan.grp_count[s] == 0:
                assert b is None
                n_idle += 1
                continue
            want = plan.collate_slot(s, toks, wl.sample_ptr[:-1], wl.span_ptr, wl.span_lo, wl.span_hi)
            for name in ("input_ids", "attention_mask", "position_ids", "labels"):
                assert b[name].shape == want[name].shape
                assert b[name].data_ptr() == getattr(out, name).data_ptr() + int(plan.grp_offset[s]) * b[name].element_size()
                assert np.array_equal(b[name].cpu().numpy(), want[name]), (name, r, k)
            assert b["valid_tokens"] == want["valid"] and b["step_samples"] == int(plan.step_samples[k])
            seen[r].extend(b["sample_ids"].cpu().tolist())
    assert n_idle > 0
    for r in range(wl.n_ranks):   # every id exactly once per rank (Thm 1)
        n_r = int(wl.rank_ptr[r + 1] - wl.rank_ptr[r])
        assert sorted(seen[r]) == list(range(n_r))
        assert sum(1 for _ in sb.rank_iter(r)) == int((plan.grp_count.reshape(wl.n_ranks, -1)[r] > 0).sum())


# ---- arrival schedules: status 0 "insufficient data", skip rounds (App. C.1) ---------------
def _sched_parity(oracle, wl, sched):
    plan, ref = oracle.run_workload(wl, avail_schedule=sched)
    info, out, round_T = Par.run_gpu(wl, staged=True, avail_schedule=sched)
    Par.compare_plan(plan, info, out, round_T)
    Par.compare_full(plan, ref, info, out)
    return plan


def test_arrival_fixture_e8(P, oracle):
    from tests import _golden as G
    g = G.load("e8_arrival.txt")
    per_rank = [G.ints(x) for x in g["rank_lengths"].split("|")]
    for join, key in ((1, "case1_schedule"), (0, "case1_schedule"), (1, "case3_schedule")):
        wl = I.custom_workload("e8", per_rank, seed=1, budget=int(g["budget"]), join_mode=join)
        plan = _sched_parity(oracle, wl, [G.ints(g[key])])
        if key == "case3_schedule":
            assert plan.n_rounds == 3 and plan.round_T.tolist() == [3]     # one skip round, one emitting, terminal


def test_arrival_random_schedules(P, oracle):
    from tests.test_oracle_arrival import _random_schedule
    for seed in range(60):
        rng = np.random.default_rng(1000 + seed)
        wl = I.protocol_workload("fuzz", seed)
        sched = _random_schedule(rng, wl, int(rng.integers(1, 12)))
        try:
            _sched_parity(oracle, wl, sched)
        except AssertionError as e:
            raise AssertionError("seed %d params %r sched %r: %s" % (seed, wl.params, sched.tolist(), e))
    for kind in ("overflow_multiround", "unequal", "empty_rank"):
        for rule in (0, 1):
            rng = np.random.default_rng(7)
            wl = I.protocol_workload(kind, 3, rule=rule)
            _sched_parity(oracle, wl, _random_schedule(rng, wl, 9))


@pytest.mark.parametrize("latency,rate", [(0, None), (2, None), (3, 50)])
def test_online_run_against_worker_pool_model(P, oracle, latency, rate):
    """plan_online: the protocol rounds against the worker-pool model (outstanding-depth envelope D = max(pf * nw,
    buffer_size); skip rounds while nothing has been delivered, Lemma 2) -- the plan and the arenas are the
    oracle's under the arrival schedule the run saw, and the envelope holds in every round."""
    for kind in ("overflow_multiround", "empty_rank", "unequal"):
        wl = I.protocol_workload(kind, 7)
        n = np.diff(wl.rank_ptr)
        bs = wl.params["buffer_size"] or int(n.max())
        pool = P.WorkerPool.from_loader(n, prefetch_factor=4, num_workers=2, buffer_size=bs, latency=latency, rate=rate)
        dw = Par.DeviceWorkload(wl)
        with P.Odb(Par.gpu_params(wl), max(wl.n_samples, 1)) as ctx:
            assert P.odb_emitted_counts(ctx.h, wl.n_ranks).tolist() == [0] * wl.n_ranks     # a fresh context
            info, log = P.plan_online(ctx, dw.lengths, wl.rank_ptr, pool)
            emitted_end = P.odb_emitted_counts(ctx.h, wl.n_ranks)                            # after termination
            out = P.OutputBuffers.for_plan(wl.n_ranks, info, dw.device, fill=Par.SENTINEL)
            P.odb_collate(ctx.h, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out.struct)
        sched = np.array([e["arrived"] for e in log])
        plan, ref = oracle.run_workload(wl, avail_schedule=sched)
        Par.compare_plan(plan, info, out, [e["T"] for e in log if e["T"] > 0])
        Par.compare_full(plan, ref, info, out)
        assert emitted_end.tolist() == (n - np.diff(plan.left_ptr)).tolist()   # E_r: every view emitted or left over
        assert (np.diff(np.array([e["emitted"] for e in log]), axis=0) >= 0).all()
        assert all((e["outstanding"] <= pool.depth).all() for e in log)
        if latency:
            assert log[0]["T"] == 0 and not (log[0]["arrived"] > 0).any()      # a skip round: nothing delivered yet


def test_set_available_state_errors(P):
    wl = I.make_workload(0)
    dw = Par.DeviceWorkload(wl)
    with P.Odb(Par.gpu_params(wl), wl.n_samples) as ctx:
        P.odb_set_available(ctx.h, [3, 5])
        P.odb_form_groups(ctx.h, dw.lengths, wl.rank_ptr)
        with pytest.raises(P.OdbError):       # inside a round
            P.odb_set_available(ctx.h, [10, 10])


# ---- maximum sizes ------------------------------------------------------------------------------
def _big_slot_parity(oracle, wl, slots):
    """Plan tables in full, the listed (large) slots element by element, any-size properties on the device."""
    plan, _ = oracle.run_workload(wl, collate=False)
    info, out, _ = Par.run_gpu(wl, staged=False)
    Par.compare_plan(plan, info, out)
    Par.compare_sampled_slots(wl, plan, out, slots(plan))
    Par.device_self_consistency(info, out, wl.params["ignore_index"])
    return plan


def test_max_sizes_two_million_sample_windows(P, oracle):
    """Two ranks, one window of 2 M samples each (sort: 9 merge passes; list ranking in global memory;
    ~870 K steps, 1.7 M slots: the slot scan runs over hundreds of tiles), a few hundred splits."""
    rng = np.random.default_rng(21)
    wl = I.custom_workload("big_windows", [rng.integers(1, 41, 2_000_000), rng.integers(1, 41, 2_000_000)], 3,
                           budget=64)
    plan = _sampled_parity(oracle, wl, n_sample=32)
    assert plan.n_steps > 500_000


def test_max_sizes_many_ranks(P, oracle):
    """4096 ranks x 0..96 samples, 26 rounds: the cross-rank reduction and the rank-major tables at a large R."""
    rng = np.random.default_rng(22)
    per = [rng.integers(8, 600, int(rng.integers(0, 97))) for _ in range(4096)]
    wl = I.custom_workload("many_ranks", per, 4, budget=2048, buffer_size=32)
    plan = _sampled_parity(oracle, wl, n_sample=32)
    assert plan.n_rounds > 2


def test_max_sizes_huge_budget(P, oracle):
    """Budget 2^31 - 1: one group of 599,999 rows x 64 columns (3.8e7 elements; the longest sample is a
    singleton, App. D step 1)."""
    rng = np.random.default_rng(23)
    wl = I.custom_workload("huge_budget", [rng.integers(1, 65, 600_000), rng.integers(1, 65, 1000)], 5,
                           budget=2**31 - 1)
    plan = _big_slot_parity(oracle, wl, lambda p: range(p.n_slots))
    assert plan.n_steps == 2 and int(plan.grp_count.max()) == 599_999


def test_max_sizes_huge_singleton(P, oracle):
    """An over-budget singleton of 1.2e8 tokens (U10) under budget 1000: a one-row block 1.2e8 wide."""
    wl = I.custom_workload("huge_singleton", [np.array([120_000_000, 7, 300, 300]), np.array([5, 6, 7, 8])], 6,
                           budget=1000)
    plan = _big_slot_parity(oracle, wl, lambda p: range(p.n_slots))
    assert int(plan.grp_width.max()) == 120_000_000


def test_quota_fixture_e9(P, oracle):
    """The hand-worked quota cases of tests/golden/e9_quota.txt through the CUDA path."""
    from tests import _golden as G
    g = G.load("e9_quota.txt")
    per_rank = [G.ints(x) for x in g["rank_lengths"].split("|")]
    for q, carried in ((5, 0), (4, 0), (8, 0), (5, 3), (100, 0)):
        wl = I.custom_workload("e9", per_rank, seed=2, budget=int(g["budget"]), join_mode=0, sample_quota=q,
                               emitted_so_far=carried)
        plan, info, out = _full_parity(oracle, wl)
        if (q, carried) == (5, 0):
            assert plan.samples_emitted == int(g["samples_emitted"]) and plan.stop_reason == int(g["stop"])


def test_wide_fuzz(P, oracle):
    """300 random jobs (up to 8 ranks x 300 samples, all flags, half of them with an arrival schedule):
    plan tables and arenas bit for bit.  (A scratch soak of the same generators ran 86,000 single-context,
    20,000 lock-step multi-context and 4,000 odb_run_host cases at the end of round 1.)"""
    for seed in range(300):
        wl, sched = Par.wide_fuzz_case(seed)
        try:
            plan, ref = oracle.run_workload(wl, avail_schedule=sched)
            info, out, round_T = Par.run_gpu(wl, staged=True, avail_schedule=sched)
            Par.compare_plan(plan, info, out, round_T)
            Par.compare_full(plan, ref, info, out)
        except AssertionError as e:
            raise AssertionError("wide fuzz seed %d params %r: %s" % (seed, wl.params, e))


@pytest.mark.parametrize("tail", [1, 2, 3])
def test_token_buffer_of_exactly_n_tokens(P, oracle, tail):
    """include/odb.h, conventions: d_tokens needs exactly n_tokens words.  A job whose token count is ``tail`` modulo 4,
    its tokens a 16-byte aligned view in the middle of a larger allocation whose every other word is poison: the
    16-byte unit that holds the last token is read whole, but nothing of the words behind it (or in front of the
    buffer) reaches an output -- plan and arenas are the oracle's, byte for byte."""
    import torch
    for seed in range(64):
        wl = I.protocol_workload("unequal", seed)
        if wl.n_tokens % 4 == tail:
            break
    else:
        pytest.fail("no workload with n_tokens %% 4 == %d" % tail)
    n_tok = wl.n_tokens
    dw = Par.DeviceWorkload(wl)
    poison = torch.full((n_tok + 64,), 0x5A5A5A5A, dtype=torch.int32, device=dw.device)
    view = poison[32:32 + n_tok]
    assert view.data_ptr() % 16 == 0 and view.numel() == n_tok
    view.copy_(dw.tokens[:n_tok])
    dw.tokens = view
    plan, ref = oracle.run_workload(wl)
    for staged in (False, True):
        info, out, _ = Par.run_gpu(wl, dw, staged=staged)
        Par.compare_plan(plan, info, out)
        Par.compare_full(plan, ref, info, out)
    assert (poison[:32] == 0x5A5A5A5A).all() and (poison[32 + n_tok:] == 0x5A5A5A5A).all()  # inputs are read-only
