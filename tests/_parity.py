"""Shared machinery of the GPU parity tests: run one workload through the CUDA path (C ABI via the
binding) and through the CPU oracle, and compare bit for bit."""
from __future__ import annotations

import numpy as np

import odb_inputs as I

SENTINEL = 0x5A
PLAN_SCALARS = ("n_rounds", "n_steps", "stop_reason", "n_slots", "total_elems", "samples_emitted", "samples_left",
                "real_tokens", "padded_elems")
SLOT_TABLES = ("grp_count", "grp_width", "grp_round", "grp_offset", "grp_real_tokens", "grp_origin", "grp_sample_ptr")


class DeviceWorkload:
    """A Workload's arrays resident on the GPU (tokens filled on the device by odb_synth_tokens)."""

    def __init__(self, wl, device="cuda:0", tokens_from_host=None):
        import torch
        import paper_2606_19989_b200 as P
        self.wl = wl
        self.device = device
        t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dt).to(device)
        self.lengths = t(wl.lengths, torch.int32)
        self.sample_ptr = t(wl.sample_ptr, torch.int64)
        self.span_ptr = t(wl.span_ptr, torch.int64)
        self.span_lo = t(wl.span_lo, torch.int32) if len(wl.span_lo) else torch.zeros(1, dtype=torch.int32, device=device)
        self.span_hi = t(wl.span_hi, torch.int32) if len(wl.span_hi) else torch.zeros(1, dtype=torch.int32, device=device)
        n_tok = wl.n_tokens
        self.tokens = torch.empty(n_tok + 16, dtype=torch.int32, device=device)
        if tokens_from_host is not None:
            self.tokens[:n_tok].copy_(torch.from_numpy(tokens_from_host))
        else:
            P.odb_synth_tokens(self.tokens, wl.token_start, n_tok, wl.token_seed, I.VOCAB)
        torch.cuda.synchronize()


def gpu_params(wl):
    import paper_2606_19989_b200 as P
    p = wl.params
    return P.make_params(wl.n_ranks, p["budget"], rule=p["rule"], join_mode=p["join_mode"],
                         sample_quota=p["sample_quota"], emitted_so_far=p["emitted_so_far"],
                         buffer_size=p["buffer_size"], slot_capacity=p["slot_capacity"], pad_id=p["pad_id"],
                         ignore_index=p["ignore_index"], shift_labels=p["shift_labels"])


def run_gpu(wl, dw=None, *, staged=True, fill=SENTINEL, avail_schedule=None, bulk_stores=False, options=None,
            spec_rec=None):
    """Returns (info, OutputBuffers, round_T).  staged=True uses form_groups/align/round_status/
    plan_query/collate; staged=False uses odb_run (two calls: the first sizes the outputs).
    options: {ODB_OPT_*: value}; spec_rec: a list that receives the round-parallel planner's record of the last
    odb_run ([rounds committed, steps, ended the protocol, 0]) or None when that run did not use it."""
    import torch
    import paper_2606_19989_b200 as P
    dw = dw or DeviceWorkload(wl)
    with P.Odb(gpu_params(wl), max(wl.n_samples, 1)) as ctx:
        if bulk_stores:
            P.odb_set_option(ctx.h, P.ODB_OPT_COLLATE_BULK_STORES, 1)
        for opt, val in (options or {}).items():
            P.odb_set_option(ctx.h, opt, val)
        if staged:
            info = ctx.plan(dw.lengths, wl.rank_ptr, avail_schedule=avail_schedule)
            round_T = list(ctx.round_T)
            out = P.OutputBuffers.for_plan(wl.n_ranks, info, dw.device, fill=fill)
            P.odb_collate(ctx.h, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out.struct)
        else:
            empty = P.OutputBuffers(wl.n_ranks, 0, 0, 0, 0, 0, dw.device)
            info = P.odb_run(ctx.h, dw.lengths, wl.rank_ptr, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo,
                             dw.span_hi, empty.struct, allow_capacity_error=True)
            out = P.OutputBuffers.for_plan(wl.n_ranks, info, dw.device, fill=fill)
            info = P.odb_run(ctx.h, dw.lengths, wl.rank_ptr, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo,
                             dw.span_hi, out.struct)
            round_T = None
            if spec_rec is not None:
                rec = np.zeros(4, dtype=np.int32)
                spec_rec.append(rec if P.odb_debug_read(ctx.h, 4, rec) == 16 else None)
        torch.cuda.synchronize()
    return info, out, round_T


def compare_plan(plan, info, out, round_T=None):
    """Plan scalars, per-slot tables, CSR of ids, step samples, leftovers: all bit-exact."""
    for k in PLAN_SCALARS:
        assert int(getattr(info, k)) == int(getattr(plan, k)), (k, int(getattr(info, k)), int(getattr(plan, k)))
    if round_T is not None:
        assert list(round_T) == plan.round_T.tolist()
    for name in SLOT_TABLES + ("grp_sample_ids", "step_samples", "left_ptr", "left_ids"):
        g = out.table(name).cpu().numpy()
        o = getattr(plan, name)
        assert g.shape == o.shape, (name, g.shape, o.shape)
        if not np.array_equal(g, o):
            bad = np.flatnonzero(g != o)
            raise AssertionError("%s differs at %d entries, first %d: gpu %r oracle %r" % (name, len(bad), bad[0],
                                                                                        g[bad[0]], o[bad[0]]))


def compare_full(plan, oracle_out, info, out):
    """Arenas byte for byte (gaps must still hold the sentinel), valid-token tables."""
    E = plan.total_elems
    for name in ("input_ids", "labels", "position_ids", "attention_mask"):
        g = getattr(out, name)[:E].cpu().numpy()
        o = oracle_out[name][:E]
        if not np.array_equal(g, o):
            bad = np.flatnonzero(g != o)
            s = int(np.searchsorted(plan.grp_offset, bad[0], side="right") - 1)
            raise AssertionError("%s differs at %d elements; first at %d (slot %d, offset %d, count %d, width %d): "
                                 "gpu %r oracle %r" % (name, len(bad), bad[0], s, plan.grp_offset[s],
                                                       plan.grp_count[s], plan.grp_width[s], g[bad[0]], o[bad[0]]))
        # tail guard: the 16 spare elements past total_elems were never written
        tail = getattr(out, name)[E:].cpu().numpy().view(np.uint8)
        assert (tail == SENTINEL).all(), name + ": wrote past total_elems"
    assert np.array_equal(out.table("grp_valid_tokens").cpu().numpy(), oracle_out["grp_valid_tokens"])
    assert np.array_equal(out.table("step_valid_tokens").cpu().numpy(), oracle_out["step_valid_tokens"])


def compare_sampled_slots(wl, plan, out, slots, global_ids=False):
    """Collate the listed slots one by one with the oracle (tokens regenerated from the hash for just
    their samples) and compare with the GPU arenas; also the slot's valid-token count."""
    p = wl.params
    gv = out.table("grp_valid_tokens").cpu().numpy()
    for s in slots:
        s = int(s)
        r = s // plan.n_steps
        c, w, off = int(plan.grp_count[s]), int(plan.grp_width[s]), int(plan.grp_offset[s])
        ids = plan.grp_sample_ids[plan.grp_sample_ptr[s]:plan.grp_sample_ptr[s + 1]].astype(np.int64)
        if not global_ids:      # (an offline plan's slots hold global sample ids already)
            ids = ids + wl.rank_ptr[r]
        toks, toff = I.tokens_for_samples(wl, ids)
        tok_start = np.zeros(max(wl.n_samples, 1), dtype=np.int64)
        tok_start[ids] = toff
        ref = plan.collate_slot(s, toks if len(toks) else np.zeros(1, np.int32), tok_start, wl.span_ptr, wl.span_lo,
                                wl.span_hi, pad_id=p["pad_id"], ignore_index=p["ignore_index"],
                                shift_labels=p["shift_labels"])
        n = c * w
        for name in ("input_ids", "labels", "position_ids", "attention_mask"):
            g = getattr(out, name)[off:off + n].cpu().numpy().reshape(c, w)
            assert np.array_equal(g, ref[name]), (name, "slot", s, "count", c, "width", w)
        assert int(gv[s]) == ref["valid"], ("grp_valid_tokens", s)
        # the alignment gap after the block is untouched
        gap_hi = int(plan.grp_offset[s + 1]) if s + 1 < plan.n_slots else plan.total_elems
        if gap_hi > off + n:
            gap = out.attention_mask[off + n:gap_hi].cpu().numpy()
            assert (gap == SENTINEL).all(), ("gap written", s)


def compare_full_by_rank(oracle, wl, plan, out, n_threads=None):
    """Every element of the four arenas, every slot, against the oracle -- rank by rank, so that neither side
    holds the whole output on the host (SURVEY.md section 7 "Host memory for parity"; about 0.9 GB per rank on
    configs[4]).  Per rank: its tokens are regenerated from the hash on the host, the oracle collates its slots
    into sentinel-filled buffers (oracle_collate_range), and the device slice [grp_offset[r K], grp_offset[(r+1) K])
    must equal them byte for byte -- blocks AND alignment gaps (which must still hold the sentinel)."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    p = wl.params
    K, R = plan.n_steps, wl.n_ranks
    gv_dev = out.table("grp_valid_tokens").cpu().numpy()
    if n_threads is None:
        try:
            n_threads = len(os.sched_getaffinity(0))
        except AttributeError:
            n_threads = os.cpu_count() or 1
        n_threads = max(1, min(n_threads, 6, R))

    def one_rank(r):
        g0, g1 = int(wl.rank_ptr[r]), int(wl.rank_ptr[r + 1])
        t0, t1 = int(wl.sample_ptr[g0]), int(wl.sample_ptr[g1])
        toks = I.token_ids(wl.token_seed, wl.token_start + t0, t1 - t0)
        tok_start = np.zeros(max(wl.n_samples, 1), dtype=np.int64)
        tok_start[g0:g1] = wl.sample_ptr[g0:g1] - t0
        ref = oracle.collate_rank(plan, r, toks if len(toks) else np.zeros(1, np.int32), tok_start, wl.span_ptr,
                                  wl.span_lo, wl.span_hi, pad_id=p["pad_id"], ignore_index=p["ignore_index"],
                                  shift_labels=p["shift_labels"], sentinel=SENTINEL)
        e0, e1 = ref["elem_lo"], ref["elem_hi"]
        for name in ("input_ids", "labels", "position_ids", "attention_mask"):
            g = getattr(out, name)[e0:e1].cpu().numpy()
            o = ref[name]
            if not np.array_equal(g, o):
                bad = np.flatnonzero(g != o)
                a = e0 + int(bad[0])
                s = int(np.searchsorted(plan.grp_offset, a, side="right") - 1)
                raise AssertionError("rank %d: %s differs at %d elements; first at arena element %d (slot %d, offset %d, "
                                     "count %d, width %d): gpu %r oracle %r" % (
                                         r, name, len(bad), a, s, plan.grp_offset[s], plan.grp_count[s],
                                         plan.grp_width[s], g[bad[0]], o[bad[0]]))
        assert np.array_equal(gv_dev[r * K:(r + 1) * K], ref["grp_valid_tokens"]), ("grp_valid_tokens", r)
        return e1 - e0

    with ThreadPoolExecutor(max_workers=n_threads) as ex:
        done = sum(ex.map(one_rank, range(R)))
    assert done == plan.total_elems          # the rank slices tile the arena
    # tail guard: the 16 spare elements past total_elems were never written
    E = plan.total_elems
    for name in ("input_ids", "labels", "position_ids", "attention_mask"):
        tail = getattr(out, name)[E:].cpu().numpy().view(np.uint8)
        assert (tail == SENTINEL).all(), name + ": wrote past total_elems"
    sv = gv_dev.astype(np.int64).reshape(R, K).sum(0) if K else np.zeros(0, np.int64)
    assert np.array_equal(out.table("step_valid_tokens").cpu().numpy(), sv)


def compare_step_range(plan, oracle_out, lo, hi, info, out, n_ranks):
    """A step range collated by odb_collate_steps against the oracle's FULL plan and arenas: slot s' = r * n +
    (k - lo) of the range must hold what slot s = r * n_steps + k of the plan holds -- tables, ids, every element of
    the block -- at the range's own offsets (a layout of this build: the exclusive scan of round_up(count * width,
    16) over s'); gaps and the tail keep the sentinel."""
    n, R, K = hi - lo, n_ranks, plan.n_steps
    assert int(info.n_steps) == n and int(info.n_slots) == R * n
    sl = (np.arange(R)[:, None] * K + np.arange(lo, hi)[None, :]).reshape(-1)  # plan slots in range order
    cnt, wid = plan.grp_count[sl].astype(np.int64), plan.grp_width[sl].astype(np.int64)
    area = cnt * wid
    off = np.concatenate([[0], np.cumsum((area + 15) // 16 * 16)])
    sp = np.concatenate([[0], np.cumsum(cnt)])
    E = int(off[-1])
    assert int(info.total_elems) == E and int(info.samples_emitted) == int(sp[-1])
    assert int(info.padded_elems) == int(area.sum()) and int(info.real_tokens) == int(plan.grp_real_tokens[sl].sum())
    tab = lambda name, m: out.table(name).cpu().numpy()[:m]
    assert np.array_equal(tab("grp_count", R * n), plan.grp_count[sl])
    assert np.array_equal(tab("grp_width", R * n), plan.grp_width[sl])
    assert np.array_equal(tab("grp_round", R * n), plan.grp_round[sl])
    assert np.array_equal(tab("grp_real_tokens", R * n), plan.grp_real_tokens[sl])
    assert np.array_equal(tab("grp_origin", R * n), plan.grp_origin[sl])
    assert np.array_equal(tab("grp_offset", R * n), off[:-1])
    assert np.array_equal(tab("grp_sample_ptr", R * n + 1), sp)
    assert np.array_equal(tab("grp_valid_tokens", R * n), oracle_out["grp_valid_tokens"][sl])
    assert np.array_equal(tab("step_samples", n), plan.step_samples[lo:hi])
    assert np.array_equal(tab("step_valid_tokens", n), oracle_out["step_valid_tokens"][lo:hi])
    ids = tab("grp_sample_ids", int(sp[-1]))
    want_ids = [plan.grp_sample_ids[plan.grp_sample_ptr[s]:plan.grp_sample_ptr[s + 1]] for s in sl]
    assert np.array_equal(ids, np.concatenate(want_ids) if want_ids else np.zeros(0, np.int32))
    for name in ("input_ids", "labels", "position_ids", "attention_mask"):
        g = getattr(out, name).cpu().numpy()
        want = np.frombuffer(bytes([SENTINEL]) * (g.nbytes), dtype=g.dtype).copy()
        ref = oracle_out[name]
        for i, s in enumerate(sl):
            a = int(area[i])
            o0 = int(plan.grp_offset[s])
            want[off[i]:off[i] + a] = ref[o0:o0 + a]
        if not np.array_equal(g, want):
            bad = np.flatnonzero(g != want)
            i = int(np.searchsorted(off, bad[0], side="right") - 1)
            raise AssertionError("steps [%d, %d): %s differs at %d elements; first at %d (range slot %d): gpu %r want %r" % (
                lo, hi, name, len(bad), bad[0], i, g[bad[0]], want[bad[0]]))


def device_self_consistency(info, out, ignore_index=-100):
    """Properties that hold at any size, checked on the device output itself: the valid-token table
    equals a recount of labels != ignore_index per slot; step totals are its column sums; the mask
    count equals real_tokens; gaps still hold the sentinel."""
    import torch
    E = int(info.total_elems)
    n_slots, n_steps = int(info.n_slots), int(info.n_steps)
    if n_slots == 0:
        return
    off = out.table("grp_offset")
    cnt = out.table("grp_count").to(torch.int64)
    wid = out.table("grp_width").to(torch.int64)
    area = cnt * wid
    lab = out.labels[:E]
    msk = out.attention_mask[:E]
    # element -> slot via the offsets; in-block flag
    # (chunked to bound memory)
    valid = torch.zeros(n_slots, dtype=torch.int64, device=lab.device)
    real = torch.zeros(n_slots, dtype=torch.int64, device=lab.device)
    gaps_ok = True
    CH = 1 << 26
    for a0 in range(0, E, CH):
        a1 = min(E, a0 + CH)
        idx = torch.arange(a0, a1, device=lab.device, dtype=torch.int64)
        sl = torch.searchsorted(off, idx, right=True) - 1
        inblk = (idx - off[sl]) < area[sl]
        v = (lab[a0:a1] != ignore_index) & inblk
        valid.index_add_(0, sl, v.to(torch.int64))
        real.index_add_(0, sl, ((msk[a0:a1] == 1) & inblk).to(torch.int64))
        gaps_ok = gaps_ok and bool((msk[a0:a1][~inblk] == SENTINEL).all())
    assert gaps_ok, "an alignment gap was written"
    assert torch.equal(valid, out.table("grp_valid_tokens").to(torch.int64))
    assert torch.equal(real, out.table("grp_real_tokens").to(torch.int64))
    assert int(real.sum()) == int(info.real_tokens)
    sv = out.table("grp_valid_tokens").to(torch.int64).view(-1, n_steps).sum(0)
    assert torch.equal(sv, out.table("step_valid_tokens"))


def wide_fuzz_case(seed, max_ranks=8, max_n=300):
    """A random job wider than ``protocol_workload("fuzz")``: up to 8 ranks x 300 samples, lengths up to
    3000, budgets 16 .. 100000, every flag; returns (workload, arrival schedule or None)."""
    from tests.test_oracle_arrival import _random_schedule
    rng = np.random.default_rng(900_000 + seed)
    R = int(rng.integers(1, max_ranks + 1))
    per = [rng.integers(1, int(rng.choice([8, 100, 3000])) + 1, int(rng.integers(0, max_n + 1))) for _ in range(R)]
    wl = I.custom_workload("wide_fuzz", per, seed, budget=int(rng.choice([16, 300, 4096, 100000])),
                           buffer_size=int(rng.choice([0, 1, 7, 64, 300])), slot_capacity=int(rng.choice([0, 1, 3, 17])),
                           rule=int(rng.integers(0, 2)), join_mode=int(rng.integers(0, 2)),
                           shift_labels=int(rng.integers(0, 2)))
    if not wl.params["join_mode"] and rng.uniform() < 0.6:
        wl.params["sample_quota"] = int(rng.integers(1, max(2, wl.n_samples + 1)))
    sched = _random_schedule(rng, wl, int(rng.integers(1, 10))) if seed % 2 == 0 else None
    return wl, sched
