"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage (PAPER.md line, written P:<line>) or the DESIGN.md reading it pins.
None of these re-types the oracle's loops: they use paper-printed values, hand-worked fixtures
(tests/golden/), closed forms, declarative verifiers (a property that the rule's output must have
and that determines it), library routines (numpy.lexsort, torch pad_sequence) and the theorems'
invariants.
"""
import itertools

import numpy as np
import pytest

import odb_inputs as I
from tests import _golden as G


# ---------------------------------------------------------------------------------------
# Eq. 1 and rule THRESHOLD
# ---------------------------------------------------------------------------------------
def test_appD_printed_values(oracle):
    """App. D: groups, padded widths, padded-token costs and B(l) values as printed."""
    g = G.load("appD_threshold.txt")
    L, lens = int(g["budget"]), G.ints(g["lengths"])
    got = oracle.group_window(oracle.RULE_THRESHOLD, L, lens)
    assert got == G.groups(g["groups"])
    assert [max(lens[i] for i in grp) for grp in got] == G.ints(g["padded_to"])
    assert [len(grp) * max(lens[i] for i in grp) for grp in got] == G.ints(g["padded_tokens"])
    for l, b in zip(G.ints(g["target_size_of"]), G.ints(g["target_size"])):
        assert oracle.target_group_size(L, l) == b
    # the same through the whole pipeline (R = 1): widths and areas of the emitted slots
    plan = oracle.OraclePlan(np.array(lens, np.int32), np.array([0, 4], np.int64), budget=L)
    assert plan.groups_of_rank(0) == G.groups(g["groups"])
    assert plan.grp_width.tolist() == G.ints(g["padded_to"])
    assert (plan.grp_width.astype(np.int64) * plan.grp_count).tolist() == G.ints(g["padded_tokens"])
    assert plan.padded_elems == sum(G.ints(g["padded_tokens"]))


def test_eq1_floor_and_clamp(oracle):
    """Eq. 1 P:34 with the floor and the clamp to 1 for l > L_max (U10, U11)."""
    assert oracle.target_group_size(1000, 1) == 1000
    assert oracle.target_group_size(1000, 333) == 3
    assert oracle.target_group_size(1000, 334) == 2
    assert oracle.target_group_size(1000, 1000) == 1
    assert oracle.target_group_size(1000, 1001) == 1
    assert oracle.target_group_size(1000, 10 ** 6) == 1
    for L, l in itertools.product([1, 7, 16384, 2 ** 31 - 1], [1, 2, 3, 5, 1024, 2 ** 31 - 1]):
        b = oracle.target_group_size(L, l)
        assert b >= 1 and (b == 1 or (b * l <= L < (b + 1) * l))


@pytest.mark.parametrize("S,l,L", [(10, 300, 1000), (1, 5, 100), (2, 5, 100), (25, 7, 50), (64, 100, 99), (9, 1, 4)])
def test_threshold_equal_lengths_closed_form(oracle, S, l, L):
    """All lengths equal: sizes in formation order are 1, B, B, ..., remainder; G = 1 + ceil((S-1)/B)."""
    B = max(L // l, 1)
    got = oracle.group_window(oracle.RULE_THRESHOLD, L, [l] * S)
    sizes_formation = [len(g) for g in got][::-1]
    want = [1] + [B] * ((S - 1) // B) + ([(S - 1) % B] if (S - 1) % B else [])
    assert sizes_formation == want
    assert len(got) == 1 + -(-(S - 1) // B)
    # ties by id ascending (U1): concatenation is 0..S-1
    assert [i for g in got for i in g] == list(range(S))


def _verify_threshold(lens, L, groups):
    """Declarative check of section 2.2: consecutive runs of the ascending order; the longest
    sample alone (t starts at 1); every other group's size equals B(l) of the shortest sample of the
    group formed before it, or it is the final partial group (U2)."""
    lens = np.asarray(lens)
    order = np.lexsort((np.arange(len(lens)), lens)).tolist()          # library sort pin (U1)
    assert [i for g in groups for i in g] == order
    form = groups[::-1]                                                 # formation order: long -> short
    assert len(form[0]) == 1
    for j in range(1, len(form)):
        t = max(L // int(lens[form[j - 1][0]]), 1)                       # row 0 = shortest = last added
        if j < len(form) - 1:
            assert len(form[j]) == t
        else:
            assert 1 <= len(form[j]) <= t
    for g in groups:                                                    # budget invariant (U10)
        assert len(g) == 1 or len(g) * max(int(lens[i]) for i in g) <= L


def test_threshold_verifier_random(oracle):
    rng = np.random.default_rng(11)
    for _ in range(300):
        S = int(rng.integers(1, 40))
        hi = int(rng.choice([4, 16, 300, 5000]))
        lens = rng.integers(1, hi + 1, S)
        L = int(rng.choice([1, 8, 64, 1000, 4096]))
        _verify_threshold(lens, L, oracle.group_window(oracle.RULE_THRESHOLD, L, lens))


def test_threshold_exhaustive_small_alphabet(oracle):
    for S in range(1, 7):
        for lens in itertools.product([1, 2, 3, 5], repeat=S):
            for L in (1, 4, 6, 11):
                _verify_threshold(lens, L, oracle.group_window(oracle.RULE_THRESHOLD, L, list(lens)))


def test_threshold_degenerate_cases(oracle):
    """L < min len -> all over-budget singletons; L >= S*max len -> exactly two groups (longest alone)."""
    lens = [50, 60, 70, 80]
    assert oracle.group_window(0, 10, lens) == [[0], [1], [2], [3]]
    assert oracle.group_window(0, 10 ** 9, lens) == [[0, 1, 2], [3]]
    assert oracle.group_window(0, 10 ** 9, [5]) == [[0]]


def test_window_with_explicit_ids(oracle):
    """Grouping a sub-window (ids given) sorts by (len, id) of those ids only."""
    lens = np.array([9, 3, 3, 7, 1, 3], np.int32)
    got = oracle.group_window(0, 6, lens, ids=np.array([5, 0, 2, 3], np.int32))
    assert [i for g in got for i in g] == [2, 5, 3, 0]


# ---------------------------------------------------------------------------------------
# rule MAXFIT_ASC
# ---------------------------------------------------------------------------------------
def _verify_maxfit(lens, L, groups):
    """Brute force on the definition: each group is feasible (max*count <= L) or a singleton, and
    NO longer run starting at the same position is feasible (checked for every longer end)."""
    lens = np.asarray(lens)
    order = np.lexsort((np.arange(len(lens)), lens)).tolist()
    assert [i for g in groups for i in g] == order
    pos = 0
    S = len(order)
    for g in groups:
        n = len(g)
        area = n * max(int(lens[i]) for i in g)
        assert n == 1 or area <= L
        for e in range(pos + n + 1, S + 1):
            run = order[pos:e]
            assert len(run) * max(int(lens[i]) for i in run) > L
        pos += n


def test_maxfit_bruteforce(oracle):
    for S in range(1, 7):
        for lens in itertools.product([1, 2, 3, 5], repeat=S):
            for L in (1, 4, 6, 11):
                _verify_maxfit(lens, L, oracle.group_window(oracle.RULE_MAXFIT_ASC, L, list(lens)))
    rng = np.random.default_rng(5)
    for _ in range(300):
        S = int(rng.integers(1, 21))
        lens = rng.integers(1, int(rng.choice([8, 100, 3000])) + 1, S)
        L = int(rng.choice([1, 16, 256, 4096]))
        _verify_maxfit(lens, L, oracle.group_window(oracle.RULE_MAXFIT_ASC, L, lens))


def test_maxfit_equal_lengths_and_rules_differ(oracle):
    assert [len(g) for g in oracle.group_window(1, 1000, [300] * 10)] == [3, 3, 3, 1]
    g = G.load("e5_rules_differ.txt")
    L, lens = int(g["budget"]), G.ints(g["lengths"])
    assert oracle.group_window(0, L, lens) == G.groups(g["groups_threshold"])
    assert oracle.group_window(1, L, lens) == G.groups(g["groups_maxfit"])
    a = G.load("appD_threshold.txt")
    assert oracle.group_window(1, int(a["budget"]), G.ints(a["lengths"])) == G.groups(a["groups"])


# ---------------------------------------------------------------------------------------
# Eq. 3
# ---------------------------------------------------------------------------------------
def test_target_groups_eq3(oracle):
    """Eq. 3: max over active ranks, positive minima, floor at 1, empty minimum = +inf (U9)."""
    assert oracle.target_groups([3, 2], [4, 4], 0) == 3          # E2
    assert oracle.target_groups([3, 2], [4, 4], 2) == 2          # E3 round 1
    assert oracle.target_groups([1, 0], [1, 0], 2) == 1          # E3 round 2: empty rank does not collapse T
    assert oracle.target_groups([0, 0], [0, 0], 0) == 1          # no active rank: floor at 1
    assert oracle.target_groups([5, 9, 7], [100, 100, 6], 0) == 6  # S_min+ binds
    assert oracle.target_groups([5, 9, 0], [100, 100, 0], 0) == 9  # rank with S=0 is not active
    assert oracle.target_groups([5, 9, 7], [100, 100, 100], 1) == 1
    rng = np.random.default_rng(3)
    for _ in range(200):
        R = int(rng.integers(1, 9))
        S = rng.integers(0, 50, R)
        Gc = np.array([int(rng.integers(1, s + 1)) if s else 0 for s in S])
        C = int(rng.integers(0, 6))
        T = oracle.target_groups(Gc, S, C)
        act = Gc > 0
        if act.any():
            assert 1 <= T <= S[act].min()
            assert T <= Gc[act].max()
            if C == 0 and S[act].min() >= Gc[act].max():
                assert T == Gc[act].max()
            if C > 0:
                assert T <= C


# ---------------------------------------------------------------------------------------
# Alg. 1: split and overflow
# ---------------------------------------------------------------------------------------
def _mk_groups(sizes):
    out, k = [], 0
    for s in sizes:
        out.append(list(range(k, k + s)))
        k += s
    return out


def test_split_properties(oracle):
    """Alg. 1 lines 3-6 (U4, U5): T groups, order of samples unchanged, the untouched
    prefix is the candidate list's prefix, everything after the touched group is singletons."""
    rng = np.random.default_rng(7)
    for _ in range(300):
        sizes = rng.integers(1, 6, int(rng.integers(1, 12))).tolist()
        S, Gc = sum(sizes), len(sizes)
        T = int(rng.integers(Gc, S + 1))
        cand = _mk_groups(sizes)
        got, back = oracle.align_list(cand, T)
        assert back == [] and len(got) == T
        assert [i for g in got for i in g] == list(range(S))
        d = T - Gc
        # walking the candidate groups from the last backward, group of size s gives up min(s-1, d)
        want = []
        for g in reversed(cand):
            k = min(len(g) - 1, d)
            d -= k
            want = [g[:len(g) - k]] + [[x] for x in g[len(g) - k:]] + want
        assert got == want


def test_split_hand_cases(oracle):
    assert oracle.align_list([[0, 1, 2], [3]], 3) == ([[0, 1], [2], [3]], [])              # E2 rank b
    assert oracle.align_list([[0, 1, 2], [3]], 4) == ([[0], [1], [2], [3]], [])
    assert oracle.align_list([[0, 1], [2, 3, 4]], 3) == ([[0, 1], [2, 3], [4]], [])        # last group first
    assert oracle.align_list([[0, 1], [2, 3, 4]], 5) == ([[0], [1], [2], [3], [4]], [])
    assert oracle.align_list([[0], [1]], 2) == ([[0], [1]], [])                            # no-op


def test_overflow_properties(oracle):
    """Alg. 1 line 8 (U6): keep the T largest by sample count, ties by list order, emitted in
    that sorted order; the rest returns to the buffer; nothing lost."""
    rng = np.random.default_rng(9)
    for _ in range(300):
        sizes = rng.integers(1, 5, int(rng.integers(2, 12))).tolist()
        Gc = len(sizes)
        T = int(rng.integers(1, Gc))
        cand = _mk_groups(sizes)
        got, back = oracle.align_list(cand, T)
        assert len(got) == T
        for g in got:
            assert g in cand
        kept_idx = [cand.index(g) for g in got]
        assert len(set(kept_idx)) == T
        keys = [(-len(cand[j]), j) for j in kept_idx]
        assert keys == sorted(keys)                                   # emitted order: size desc, index asc
        dropped = [j for j in range(Gc) if j not in kept_idx]
        for j in dropped:
            for kk in kept_idx:
                assert (-len(cand[kk]), kk) < (-len(cand[j]), j)      # every kept group precedes every dropped one
        assert sorted(back + [i for g in got for i in g]) == list(range(sum(sizes)))


def test_overflow_hand_case(oracle):
    got, back = oracle.align_list([[0, 1], [2], [3]], 2)                                   # E3 rank a
    assert got == [[0, 1], [2]] and back == [3]
    got, back = oracle.align_list([[0], [1, 2], [3], [4, 5]], 3)
    assert got == [[1, 2], [4, 5], [0]] and back == [3]


# ---------------------------------------------------------------------------------------
# hand-worked protocol fixtures E2-E4
# ---------------------------------------------------------------------------------------
def _plan_from_fixture(oracle, g, **kw):
    per = [G.ints(x) for x in g["rank_lengths"].split("|")]
    lens = np.array([l for p in per for l in p], np.int32)
    rp = np.concatenate([[0], np.cumsum([len(p) for p in per])]).astype(np.int64)
    return oracle.OraclePlan(lens, rp, budget=int(g["budget"]), slot_capacity=int(g.get("slot_capacity", 0)),
                             join_mode=int(g.get("join_mode", 1)), **kw)


def test_e2_split_fixture(oracle):
    g = G.load("e2_split.txt")
    assert oracle.group_window(0, int(g["budget"]), [300] * 4) == G.groups(g["candidate_b"])
    p = _plan_from_fixture(oracle, g)
    assert p.round_T.tolist() == [int(g["T"])]
    assert p.groups_of_rank(0) == G.groups(g["groups_a"])
    assert p.groups_of_rank(1) == G.groups(g["groups_b"])
    assert p.n_rounds == int(g["n_rounds"]) and p.samples_emitted == int(g["samples_emitted"])


def test_e3_overflow_join_fixture(oracle):
    g = G.load("e3_overflow_join.txt")
    p = _plan_from_fixture(oracle, g)
    assert p.groups_of_rank(0) == G.groups(g["groups_a"])
    assert p.groups_of_rank(1) == G.groups(g["groups_b"])
    assert p.round_T.tolist() == G.ints(g["round_T"])
    assert (p.n_rounds, p.n_steps, p.samples_emitted, p.stop_reason) == tuple(
        int(g[k]) for k in ("n_rounds", "n_steps", "samples_emitted", "stop_reason"))
    assert p.grp_round.reshape(2, -1).tolist() == [[0, 0, 1], [0, 0, 1]]
    assert p.grp_count.reshape(2, -1).tolist() == [[2, 1, 1], [3, 1, 0]]
    assert p.grp_width.reshape(2, -1).tolist() == [[200, 500, 800], [300, 300, 0]]


def test_e4_overflow_nonjoin_fixture(oracle):
    g = G.load("e4_overflow_nonjoin.txt")
    p = _plan_from_fixture(oracle, g)
    assert p.groups_of_rank(0) == G.groups(g["groups_a"])
    assert p.groups_of_rank(1) == G.groups(g["groups_b"])
    assert (p.n_rounds, p.n_steps, p.samples_emitted, p.stop_reason) == tuple(
        int(g[k]) for k in ("n_rounds", "n_steps", "samples_emitted", "stop_reason"))
    assert p.left_ids[p.left_ptr[0]:p.left_ptr[1]].tolist() == G.ints(g["left_a"])
    assert p.left_ids[p.left_ptr[1]:p.left_ptr[2]].tolist() == G.ints(g["left_b"])


# ---------------------------------------------------------------------------------------
# round loop invariants (Lemma 1, Lemma 2, Thm 1, Thm 2, Thm 4)
# ---------------------------------------------------------------------------------------
def _check_invariants(oracle, wl):
    prm = wl.params
    p = oracle.OraclePlan(wl.lengths, wl.rank_ptr, **prm)
    R, L = wl.n_ranks, prm["budget"]
    n_r = np.diff(wl.rank_ptr)
    # same number of slots on every rank (U14) is asserted by the wrapper; layout sizes
    assert p.n_slots == R * p.n_steps and len(p.grp_count) == p.n_slots
    # Lemma 1: emitted (+) un-emitted = sampler views, per rank, nothing twice
    for r in range(R):
        em = np.concatenate([p.slot_ids(r, k) for k in range(p.n_steps)]) if p.n_steps else np.zeros(0, np.int32)
        lf = p.left_ids[p.left_ptr[r]:p.left_ptr[r + 1]]
        assert sorted(np.concatenate([em, lf]).tolist()) == list(range(int(n_r[r])))
        assert (np.diff(lf) > 0).all()
    assert p.samples_emitted + p.samples_left == wl.n_samples
    assert p.samples_emitted == int(p.grp_count.sum()) == int(p.step_samples.sum())
    # budget invariant per slot (U10) and pad-to-max width
    for r in range(R):
        lens_r = wl.lengths[wl.rank_ptr[r]:wl.rank_ptr[r + 1]]
        for k in range(p.n_steps):
            ids = p.slot_ids(r, k)
            s = r * p.n_steps + k
            assert len(ids) == p.grp_count[s]
            if len(ids):
                assert p.grp_width[s] == lens_r[ids].max()
                assert len(ids) == 1 or len(ids) * int(lens_r[ids].max()) <= L
                assert p.grp_real_tokens[s] == lens_r[ids].sum()
                key = list(zip(lens_r[ids].tolist(), ids.tolist()))
                assert key == sorted(key)                              # rows ascending by (len,id) (U3)
            else:
                assert p.grp_width[s] == 0
    # offsets: exclusive scan of round_up(area,16), rank-major
    area = p.grp_count.astype(np.int64) * p.grp_width
    ru = (area + 15) // 16 * 16
    assert (p.grp_offset == np.concatenate([[0], np.cumsum(ru)[:-1]])).all() if p.n_slots else True
    assert p.total_elems == int(ru.sum()) and p.padded_elems == int(area.sum())
    assert p.real_tokens == int(p.grp_real_tokens.sum())
    # Lemma 2: every emitting round emits at least T >= 1 views on every active rank
    n_emit_rounds = len(p.round_T)
    rounds = p.grp_round.reshape(R, -1) if p.n_steps else np.zeros((R, 0), np.int32)
    cnt = p.grp_count.reshape(R, -1) if p.n_steps else np.zeros((R, 0), np.int32)
    for j in range(n_emit_rounds):
        cols = rounds[0] == j
        assert (rounds[:, cols] == j).all()
        if p.stop_reason != oracle.STOP_QUOTA or j < n_emit_rounds - 1:
            assert cols.sum() == p.round_T[j]
        assert cnt[:, cols].sum() >= 1
        for r in range(R):                                             # an active rank has no IDLE slot in the round
            c = cnt[r, cols]
            assert (c > 0).all() or (c == 0).all()
    # Thm 4 with the D-term 0 in this synchronous model, +1 for the terminal check
    assert p.n_rounds <= int(n_r.max(initial=0)) + 1
    if prm["join_mode"]:
        assert p.stop_reason == oracle.STOP_ALL_FINISHED and p.samples_left == 0      # Thm 1
        assert p.n_rounds == n_emit_rounds + 1
    else:
        Q = prm["sample_quota"]
        if p.stop_reason == oracle.STOP_QUOTA:                                         # Thm 2
            tot = prm["emitted_so_far"] + p.samples_emitted
            assert Q <= tot <= Q + int(p.step_samples.max())
            assert tot - int(p.step_samples[-1]) < Q                                   # stopped at the FIRST such step
        else:
            assert p.stop_reason == oracle.STOP_LOGICAL
            # LOGICAL: some rank is finished -- nothing buffered, nothing pending, so it leaves no sample --
            # and no emitted step had reached the quota (else the run would have stopped there, Thm 2)
            assert (np.diff(p.left_ptr) == 0).any()
            assert Q <= 0 or p.n_steps == 0 or prm["emitted_so_far"] + p.samples_emitted < Q
    return p


@pytest.mark.parametrize("kind", ["audit:" + k for k in I.AUDIT_KINDS] + ["overflow_multiround", "empty_rank",
                                                                           "unequal"])
@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("join", [1, 0])
def test_round_loop_invariants_protocol(oracle, kind, rule, join):
    wl = I.protocol_workload(kind, rule=rule, join_mode=join)
    _check_invariants(oracle, wl)


def test_round_loop_invariants_fuzz(oracle):
    for seed in range(400):
        _check_invariants(oracle, I.protocol_workload("fuzz", seed=seed))


def test_quota_closure_audit(oracle):
    """Cor. 1: quota closure on the six audit distributions, non-join, several quotas."""
    for kind in I.AUDIT_KINDS:
        for frac in (0.1, 0.5, 0.95):
            wl = I.protocol_workload("audit:" + kind, join_mode=0)
            wl.params["sample_quota"] = int(frac * wl.n_samples)
            p = _check_invariants(oracle, wl)
            assert p.stop_reason in (oracle.STOP_QUOTA, oracle.STOP_LOGICAL)


def test_empty_rank_liveness(oracle):
    """App. F structure: one rank assigned zero samples; join mode terminates, that rank
    only holds IDLE slots, every other rank emits everything."""
    wl = I.protocol_workload("empty_rank")
    p = _check_invariants(oracle, wl)
    R = wl.n_ranks
    cnt = p.grp_count.reshape(R, -1)
    assert (cnt[R - 1] == 0).all() and p.n_steps > 0
    assert cnt[:R - 1].sum(axis=1).tolist() == np.diff(wl.rank_ptr)[:R - 1].tolist()
    # non-join: a finished rank at round 1 stops the logical iteration before anything is emitted
    p2 = oracle.OraclePlan(wl.lengths, wl.rank_ptr, **dict(wl.params, join_mode=0))
    assert p2.stop_reason == oracle.STOP_LOGICAL and p2.n_steps == 0 and p2.samples_emitted == 0


def test_degenerate_inputs(oracle):
    # all ranks empty
    p = oracle.OraclePlan(np.zeros(0, np.int32), np.zeros(4, np.int64), budget=100)
    assert (p.n_steps, p.n_rounds, p.stop_reason, p.total_elems) == (0, 1, 0, 0)
    # R = 1: alignment is a no-op, T = G
    lens = np.array([5, 9, 2, 7, 7, 1], np.int32)
    p = oracle.OraclePlan(lens, np.array([0, 6], np.int64), budget=14)
    assert p.groups_of_rank(0) == oracle.group_window(0, 14, lens)
    # len < 1 is rejected
    with pytest.raises(ValueError):
        oracle.OraclePlan(np.array([3, 0], np.int32), np.array([0, 2], np.int64), budget=10)
    # under THRESHOLD the longest sample of a window is always a singleton (t starts at 1)
    rng = np.random.default_rng(2)
    for _ in range(50):
        lens = rng.integers(1, 100, int(rng.integers(2, 50)))
        g = oracle.group_window(0, int(rng.integers(1, 500)), lens)
        assert len(g[-1]) == 1


def test_bj_configs_plan_shapes(oracle):
    """Configs 1-3 of BASELINE.json: single emitting round, only split fires, invariants hold."""
    for idx in (0, 1, 2):
        for rule in (0, 1):
            wl = I.make_workload(idx, rule=rule)
            p = oracle.OraclePlan(wl.lengths, wl.rank_ptr, **wl.params)
            assert p.n_rounds == 2 and p.samples_left == 0
            cnt = p.grp_count.reshape(wl.n_ranks, -1)
            assert (cnt > 0).all()
    wl = I.make_workload(0)
    _check_invariants(oracle, wl)


def test_fill_ratio_trend(oracle):
    """Soft check of 'per-group token counts converge to L_max' and of Table 17's trend
    (pad% falls as the buffer grows) on a synthetic CV~1 workload."""
    rng = np.random.default_rng(0)
    sig2 = np.log(2.0)
    lens = np.clip(np.rint(rng.lognormal(np.log(1500) - sig2 / 2, np.sqrt(sig2), 8192)), 1, 8192).astype(np.int32)
    pads = []
    for bf in (10, 100, 1000, 8192):
        p = oracle.OraclePlan(lens, np.array([0, len(lens)], np.int64), budget=8192, buffer_size=bf)
        pads.append(1 - p.real_tokens / p.padded_elems)
    assert pads[0] > pads[1] > pads[2] > pads[3]
    assert pads[3] < 0.02


# ---------------------------------------------------------------------------------------
# collation (C.4): E6 fixture, torch pad_sequence, valid counts
# ---------------------------------------------------------------------------------------
def test_e6_collate_fixture(oracle):
    g = G.load("e6_collate.txt")
    toks = [G.ints(x) for x in g["tokens"].split("|")]
    lens = np.array([len(t) for t in toks], np.int32)
    tokens = np.array([x for t in toks for x in t], np.int32)
    tok_start = np.array([0, len(toks[0])], np.int64)
    spans = G.groups(g["spans"])
    span_ptr = np.array([0, len(spans[0]) // 2, len(spans[0]) // 2 + len(spans[1]) // 2], np.int64)
    flat = [x for s in spans for x in s]
    span_lo, span_hi = np.array(flat[0::2], np.int32), np.array(flat[1::2], np.int32)
    p = oracle.OraclePlan(lens, np.array([0, 2], np.int64), budget=int(g["budget"]), rule=int(g["rule"]))
    assert p.n_steps == 1 and p.grp_count.tolist() == [2] and p.grp_width.tolist() == [3]
    assert p.grp_real_tokens.tolist() == [int(g["real_tokens"])]
    for shift in (1, 0):
        o = p.collate_slot(0, tokens, tok_start, span_ptr, span_lo, span_hi, shift_labels=shift)
        assert o["input_ids"].tolist() == G.groups(g["input_ids"])
        assert o["attention_mask"].tolist() == G.groups(g["attention_mask"])
        assert o["position_ids"].tolist() == G.groups(g["position_ids"])
        assert o["labels"].tolist() == G.groups(g["labels_shift%d" % shift])
        assert o["valid"] == int(g["valid_shift%d" % shift])


@pytest.mark.parametrize("shift", [1, 0])
def test_collate_matches_pad_sequence(oracle, shift):
    """Collation reduces to a library routine: torch pad_sequence for ids / labels, arange < len for
    mask and positions (Tiny config and a multimodal-shaped small case with two spans per sample)."""
    import torch
    from torch.nn.utils.rnn import pad_sequence
    for wl in (I.make_workload(0), I.make_workload(2, n_ranks=2, n_per_rank=48)):
        wl.params["shift_labels"] = shift
        tokens = wl.tokens()
        plan, out = oracle.run_workload(wl, tokens)
        for s in range(plan.n_slots):
            r, k = divmod(s, plan.n_steps)
            ids = plan.slot_ids(r, k)
            seqs, labs = [], []
            for i in ids:
                gidx = int(wl.rank_ptr[r]) + int(i)
                t = torch.from_numpy(tokens[wl.sample_ptr[gidx]:wl.sample_ptr[gidx + 1]].astype(np.int64))
                lab = t.clone()
                for j in range(int(wl.span_ptr[gidx]), int(wl.span_ptr[gidx + 1])):
                    lab[int(wl.span_lo[j]):int(wl.span_hi[j])] = -100
                if shift:
                    lab = torch.cat([lab[1:], torch.tensor([-100])])
                seqs.append(t)
                labs.append(lab)
            want_ids = pad_sequence(seqs, batch_first=True, padding_value=0).numpy()
            want_lab = pad_sequence(labs, batch_first=True, padding_value=-100).numpy()
            lens = torch.tensor([len(x) for x in seqs])
            ar = torch.arange(want_ids.shape[1])[None, :]
            want_mask = (ar < lens[:, None]).numpy()
            want_pos = (ar * (ar < lens[:, None])).numpy()
            c, w = int(plan.grp_count[s]), int(plan.grp_width[s])
            assert want_ids.shape == (c, w)
            o = int(plan.grp_offset[s])
            sl = slice(o, o + c * w)
            assert (out["input_ids"][sl].reshape(c, w) == want_ids).all()
            assert (out["labels"][sl].reshape(c, w) == want_lab).all()
            assert (out["attention_mask"][sl].reshape(c, w) == want_mask).all()
            assert (out["position_ids"][sl].reshape(c, w) == want_pos).all()
            assert out["grp_valid_tokens"][s] == int((want_lab != -100).sum())
            # gap elements after the block keep the sentinel: never written
            nxt = int(plan.grp_offset[s + 1]) if s + 1 < plan.n_slots else plan.total_elems
            assert (out["attention_mask"][o + c * w:nxt] == 0x5A).all()
        sv = out["grp_valid_tokens"].reshape(wl.n_ranks, -1).sum(axis=0)
        assert (out["step_valid_tokens"] == sv).all()


def test_collate_slot_equals_collate_all(oracle):
    wl = I.protocol_workload("overflow_multiround")
    tokens = wl.tokens()
    plan, out = oracle.run_workload(wl, tokens)
    for s in range(0, plan.n_slots, 7):
        o = plan.collate_slot(s, tokens, wl.sample_ptr[:-1], wl.span_ptr, wl.span_lo, wl.span_hi)
        c, w, off = int(plan.grp_count[s]), int(plan.grp_width[s]), int(plan.grp_offset[s])
        assert (out["labels"][off:off + c * w].reshape(c, w) == o["labels"]).all()
        assert out["grp_valid_tokens"][s] == o["valid"]


def test_collate_rank_tiles_collate_all(oracle):
    """collate_rank (the rank-by-rank form the full-size GPU parity tests use, with only the rank's own tokens
    regenerated from the hash) concatenated over the ranks IS collate_all's arenas, gaps included."""
    for wl in (I.protocol_workload("empty_rank", 1), I.protocol_workload("overflow_multiround", 2, join_mode=0),
               I.make_workload(0)):
        plan, out = oracle.run_workload(wl)
        at = 0
        for r in range(wl.n_ranks):
            g0, g1 = int(wl.rank_ptr[r]), int(wl.rank_ptr[r + 1])
            t0, t1 = int(wl.sample_ptr[g0]), int(wl.sample_ptr[g1])
            toks = I.token_ids(wl.token_seed, wl.token_start + t0, t1 - t0)
            tok_start = np.full(max(wl.n_samples, 1), -(1 << 40), dtype=np.int64)   # other ranks: never dereferenced
            tok_start[g0:g1] = wl.sample_ptr[g0:g1] - t0
            ref = oracle.collate_rank(plan, r, toks if len(toks) else np.zeros(1, np.int32), tok_start, wl.span_ptr,
                                      wl.span_lo, wl.span_hi, shift_labels=wl.params["shift_labels"])
            assert ref["elem_lo"] == at
            at = ref["elem_hi"]
            for name in ("input_ids", "labels", "position_ids", "attention_mask"):
                assert np.array_equal(ref[name], out[name][ref["elem_lo"]:ref["elem_hi"]]), (wl.name, r, name)
            K = plan.n_steps
            assert np.array_equal(ref["grp_valid_tokens"], out["grp_valid_tokens"][r * K:(r + 1) * K])
        assert at == plan.total_elems


# ---------------------------------------------------------------------------------------
# input generator: counter-based token ids
# ---------------------------------------------------------------------------------------
def test_token_hash_reference_values():
    """SplitMix64 finaliser: mix64(0) = 0 and the first published SplitMix64 outputs for seed 0 are
    mix64(k * golden); token = ((mix >> 32) * VOCAB) >> 32 stays inside the vocabulary."""
    def mix64(z):
        z &= (1 << 64) - 1
        z ^= z >> 30
        z = (z * 0xBF58476D1CE4E5B9) & ((1 << 64) - 1)
        z ^= z >> 27
        z = (z * 0x94D049BB133111EB) & ((1 << 64) - 1)
        z ^= z >> 31
        return z
    # java.util.SplittableRandom / SplitMix64 with seed 0: first output 0xE220A8397B1DCDAF
    assert mix64(0x9E3779B97F4A7C15) == 0xE220A8397B1DCDAF
    for seed, start in ((0, 0), (4, 12345), (7001, 2 ** 33 + 5)):
        got = I.token_ids(seed, start, 64)
        want = [(((mix64(seed * 0x9E3779B97F4A7C15 + start + j) >> 32) * I.VOCAB) >> 32) for j in range(64)]
        assert got.tolist() == want
        assert got.min() >= 0 and got.max() < I.VOCAB


def test_e9_quota_fixture(oracle):
    g = G.load("e9_quota.txt")
    per_rank = [G.ints(x) for x in g["rank_lengths"].split("|")]
    lens = np.array([x for r in per_rank for x in r], np.int32)
    rp = np.array([0, 4, 8], np.int64)
    p = oracle.OraclePlan(lens, rp, budget=int(g["budget"]), join_mode=0, sample_quota=int(g["quota"]))
    assert p.groups_of_rank(0) == G.groups(g["groups_a"]) and p.groups_of_rank(1) == G.groups(g["groups_b"])
    assert p.left_ids[p.left_ptr[0]:p.left_ptr[1]].tolist() == G.ints(g["left_a"])
    assert p.left_ids[p.left_ptr[1]:p.left_ptr[2]].tolist() == G.ints(g["left_b"])
    assert p.samples_emitted == int(g["samples_emitted"]) and p.stop_reason == int(g["stop"])
    assert p.n_rounds == int(g["n_rounds"])
    for q, key in ((4, "quota4_steps"), (8, "quota8_steps")):
        p = oracle.OraclePlan(lens, rp, budget=int(g["budget"]), join_mode=0, sample_quota=q)
        assert p.n_steps == int(g[key]) and p.stop_reason == oracle.STOP_QUOTA
    p = oracle.OraclePlan(lens, rp, budget=int(g["budget"]), join_mode=0, sample_quota=5, emitted_so_far=3)
    assert p.n_steps == int(g["carried3_quota5_steps"])
    # join mode ignores the quota
    p = oracle.OraclePlan(lens, rp, budget=int(g["budget"]), join_mode=1, sample_quota=5)
    assert p.n_steps == 3 and p.stop_reason == oracle.STOP_ALL_FINISHED
