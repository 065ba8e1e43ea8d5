"""Pins of the oracle's OFFLINE planners (GMT / BMT, App. I; HFG, App. J
PAPER.md:631).  Each is pinned to something other than itself: the App. D values under the padded-area rule, a
declarative verifier of the greedy packing (feasible, maximal, consecutive runs of the sorted order), the
wrap-around / striding properties the paper states, reductions of BMT to GMT, and numpy's lexsort for HFG."""
import numpy as np
import pytest

from tests import _golden as G


def _batches_of(plan, W):
    """The global batch list behind a strided plan: batch j sits in slot (j % W, j // W)."""
    return [plan.slot_ids(j % W, j // W).tolist() for j in range(plan.n_steps * W)]


def _verify_greedy(batches, lengths, budget, order):
    """`batches` = the greedy max-fit packing of `order` (ids ascending by (len, tie)): consecutive runs, each
    feasible on padded area (or an over-budget singleton), each maximal (the next sample would not fit)."""
    flat = [i for b in batches for i in b]
    assert flat == list(order)
    for j, b in enumerate(batches):
        mx = max(lengths[i] for i in b)
        assert len(b) == 1 or mx * len(b) <= budget
        if j + 1 < len(batches):
            nxt = batches[j + 1][0]
            assert (len(b) + 1) * max(mx, lengths[nxt]) > budget


def test_gmt_appD_fixture(oracle):
    g = G.load("f4_gmt_appD.txt")
    L = G.ints(g["lengths"])
    W = int(g["world"])
    plan = oracle.OraclePlan.offline(oracle.OraclePlan.PLANNER_GMT, L, W, budget=int(g["budget"]))
    for r in range(W):
        want = [G.ints(x) for x in g["rank%d" % r].split("|")]
        assert plan.groups_of_rank(r) == want
        assert plan.grp_width[r * plan.n_steps:(r + 1) * plan.n_steps].tolist() == G.ints(g["widths_rank%d" % r])
    assert plan.step_samples.tolist() == G.ints(g["step_samples"])
    assert plan.n_rounds == 1 and plan.stop_reason == 0 and plan.samples_left == 0


@pytest.mark.parametrize("W", [1, 2, 3, 8])
def test_gmt_greedy_wraparound_striding(oracle, W):
    rng = np.random.default_rng(W)
    for trial in range(40):
        N = int(rng.integers(1, 60))
        L = rng.integers(1, 400, N)
        budget = int(rng.choice([50, 400, 3000]))
        plan = oracle.OraclePlan.offline(0, L, W, budget=budget)
        order = np.lexsort((np.arange(N), L))                      # ascending (length, id): a library routine
        allb = _batches_of(plan, W)
        # the number of distinct batches: the list is padded by repeating the leading ones
        Gn = next(g for g in range(1, len(allb) + 1) if all(allb[j] == allb[j % g] for j in range(len(allb)))
                  and sum(len(b) for b in allb[:g]) == N)
        _verify_greedy(allb[:Gn], L, budget, order)
        assert len(allb) - Gn <= W - 1                              # "at most W-1 repeated batches per epoch"
        assert len(allb) % W == 0 and plan.n_steps == -(-Gn // W)   # identical step count on every rank
        assert plan.samples_emitted == N + sum(len(b) for b in allb[Gn:])
        assert sorted(i for b in allb[:Gn] for i in b) == list(range(N))   # full-epoch coverage, zero truncation


def test_bmt_properties_and_reduction_to_gmt(oracle):
    rng = np.random.default_rng(5)
    for trial in range(40):
        N = int(rng.integers(1, 80))
        W = int(rng.integers(1, 5))
        L = rng.integers(1, 300, N)
        budget = int(rng.choice([64, 500, 2000]))
        size = int(rng.integers(1, 25))
        perm = rng.permutation(N)
        key = rng.integers(0, 2**31 - 1, N)
        plan = oracle.OraclePlan.offline(1, L, W, budget=budget, perm=perm, shuffle_key=key, size=size)
        allb = _batches_of(plan, W)
        # undo wrap-around: the first Gn batches cover every id exactly once
        Gn = next(g for g in range(1, len(allb) + 1) if sum(len(b) for b in allb[:g]) == N
                  and sorted(i for b in allb[:g] for i in b) == list(range(N)))
        assert len(allb) - Gn <= W - 1 and all(allb[j] == allb[j % Gn] for j in range(len(allb)))
        pos = np.empty(N, np.int64)
        pos[perm] = np.arange(N)                                   # position of a sample in the shuffled order
        bucket_of = lambda i: int(pos[i]) // size
        per_bucket = {}
        for b in allb[:Gn]:
            assert len({bucket_of(i) for i in b}) == 1              # packing never leaves a bucket
            per_bucket.setdefault(bucket_of(b[0]), []).append(b)
        for bk, bs in per_bucket.items():
            ids = perm[bk * size:(bk + 1) * size]
            order = ids[np.lexsort((np.arange(len(ids)), L[ids]))]  # within-bucket (length, shuffled position)
            bs_sorted = sorted(bs, key=lambda b: (L[b[0]], pos[b[0]]))
            _verify_greedy(bs_sorted, L, budget, order)
        # the batch shuffle: keys of the pre-shuffle batch indices are ascending along the final list.  Pre-shuffle
        # index of a batch = rank among batches ordered by (bucket, first row's (length, position)).
        pre = sorted(range(Gn), key=lambda j: (bucket_of(allb[j][0]), L[allb[j][0]], pos[allb[j][0]]))
        pre_index = {j: t for t, j in enumerate(pre)}
        ks = [(int(key[pre_index[j]]), pre_index[j]) for j in range(Gn)]
        assert ks == sorted(ks)
    # one bucket, identity shuffle, ascending keys: BMT is GMT
    L = rng.integers(1, 300, 57)
    a = oracle.OraclePlan.offline(1, L, 3, budget=700, perm=np.arange(57), shuffle_key=np.arange(57), size=57)
    b = oracle.OraclePlan.offline(0, L, 3, budget=700)
    assert a.groups_of_rank(1) == b.groups_of_rank(1) and a.total_elems == b.total_elems


def test_hfg_against_lexsort(oracle):
    rng = np.random.default_rng(9)
    for trial in range(40):
        N = int(rng.integers(1, 90))
        W = int(rng.integers(1, 6))
        bs = int(rng.integers(1, 7))
        mega = int(rng.integers(1, 40))
        L = rng.integers(1, 500, N)
        perm = rng.permutation(N)
        plan = oracle.OraclePlan.offline(2, L, W, perm=perm, size=mega, batch_size=bs)
        # the index list: per megabatch, the reverse of numpy's ascending (length, position) order
        idx = []
        for m0 in range(0, N, mega):
            ids = perm[m0:m0 + mega]
            idx.extend(ids[np.lexsort((np.arange(len(ids)), L[ids]))][::-1].tolist())
        n_per = -(-N // W)
        padded = [idx[i % N] for i in range(n_per * W)]            # padded to a multiple of W with the leading indices
        for r in range(W):
            mine = padded[r::W]                                     # stride-sharded
            want = [mine[i:i + bs] for i in range(0, n_per, bs)]    # fixed batch size, last one ragged
            assert plan.groups_of_rank(r) == want
        assert plan.n_steps == -(-n_per // bs) and plan.samples_emitted == n_per * W
        s = plan.grp_sample_ptr
        for q in range(plan.n_slots):
            ids = plan.grp_sample_ids[s[q]:s[q + 1]]
            assert plan.grp_width[q] == (L[ids].max() if len(ids) else 0)


def test_offline_layout_and_collation(oracle):
    """Offsets / totals of an offline plan follow the same layout rules, and its slots collate like any other
    (global ids: tok_start indexed by global sample id)."""
    import odb_inputs as I
    wl = I.offline_workload(3, 0, n=70)
    for planner, kw in ((0, {}), (1, dict(perm=wl.perm, shuffle_key=wl.shuffle_key, size=16)),
                        (2, dict(perm=wl.perm, size=24, batch_size=5))):
        plan = oracle.OraclePlan.offline(planner, wl.lengths, 3, budget=wl.params["budget"], **kw)
        area = plan.grp_count.astype(np.int64) * plan.grp_width
        off = np.concatenate([[0], np.cumsum((area + 15) // 16 * 16)])
        assert np.array_equal(plan.grp_offset, off[:-1]) and plan.total_elems == off[-1]
        assert plan.padded_elems == area.sum()
        toks = wl.tokens()
        out = plan.collate_all(toks, wl.sample_ptr[:-1], wl.span_ptr, wl.span_lo, wl.span_hi)
        for q in range(0, plan.n_slots, 3):
            o = plan.collate_slot(q, toks, wl.sample_ptr[:-1], wl.span_ptr, wl.span_lo, wl.span_hi)
            c, w, a0 = int(plan.grp_count[q]), int(plan.grp_width[q]), int(plan.grp_offset[q])
            assert np.array_equal(out["input_ids"][a0:a0 + c * w].reshape(c, w), o["input_ids"])
            ids = plan.grp_sample_ids[plan.grp_sample_ptr[q]:plan.grp_sample_ptr[q + 1]]
            for b, g in enumerate(ids):                              # row b IS sample g, right-padded
                n = int(wl.lengths[g])
                assert np.array_equal(o["input_ids"][b, :n], toks[wl.sample_ptr[g]:wl.sample_ptr[g] + n])
                assert (o["attention_mask"][b] == (np.arange(w) < n)).all()
