"""Pins of the oracle's loss-scaling weights (section 2.3 "Loss scaling"
P:60-65, App. B, the three modes P:738) against things other than the oracle itself:
the hand-worked fixture e7 (exact fractions), Eq. 2's identity sum_r w_r Lbar_r = L* evaluated in
exact rational arithmetic on random per-token losses, the paper's statements about when the modes
coincide, and the origin table against a declarative description of split / overflow."""
from fractions import Fraction

import numpy as np
import pytest

import odb_inputs as I
from tests import _golden as G


@pytest.fixture(scope="module")
def oracle():
    from oracle import odb_oracle
    odb_oracle.build()
    return odb_oracle


def _fracs(s):
    return [Fraction(x) for x in s.split()]


def _close(w, fr):
    """fp64 value of a correctly rounded quotient chain vs the exact rational: a few ulps."""
    return abs(Fraction(float(w)) - fr) <= abs(fr) * Fraction(4, 2 ** 52)


def test_e7_fixture(oracle):
    g = G.load("e7_loss_scaling.txt")
    e2 = G.load("e2_split.txt")
    # the origin table of the fixture's plan comes out of the oracle's literal split loop
    per_rank = [G.ints(x) for x in e2["rank_lengths"].split("|")]
    lens = np.array([x for r in per_rank for x in r], np.int32)
    p = oracle.OraclePlan(lens, np.array([0, 4, 8], np.int64), budget=int(e2["budget"]))
    assert p.grp_origin.tolist() == G.ints(g["origin_a"]) + G.ints(g["origin_b"])
    assert p.grp_count.tolist() == G.ints(g["counts_a"]) + G.ints(g["counts_b"])
    count = np.array(G.ints(g["counts_a"]) + G.ints(g["counts_b"]), np.int32)
    valid = np.array(G.ints(g["valid_a"]) + G.ints(g["valid_b"]), np.int32)
    for mode, key in ((oracle.SCALE_TOKEN_EXACT, "exact"), (oracle.SCALE_SAMPLE, "sample"),
                      (oracle.SCALE_TOKEN_APPROX, "approx")):
        w = oracle.loss_weights(mode, 2, 3, count, valid, p.grp_origin)
        for r, name in enumerate("ab"):
            want = _fracs(g["%s_%s" % (key, name)])
            for k in range(3):
                assert _close(w[r, k], want[k]), (key, name, k, w[r, k], want[k])


def test_eq2_identity_exact_rational(oracle):
    """Eq. 2: with w_r = t_r / T_tok, sum_r w_r * mean_r(loss) equals the per-token reference
    loss L* = (1/T_tok) sum of all token losses.  Evaluated with Fractions on random integer losses;
    the oracle's fp64 weights must reproduce L* to rounding, and sample-level weights must NOT when
    tokens per sample differ across ranks."""
    rng = np.random.default_rng(7)
    R, K = 5, 4
    count = rng.integers(1, 6, size=(R, K)).astype(np.int32)
    valid = np.zeros((R, K), np.int32)
    losses = {}
    for r in range(R):
        for k in range(K):
            t = int(rng.integers(1, 40)) * int(count[r, k])
            valid[r, k] = t
            losses[r, k] = [Fraction(int(x), 1000) for x in rng.integers(0, 9000, size=t)]
    origin = np.tile(np.arange(K, dtype=np.int32), R)
    w = oracle.loss_weights(oracle.SCALE_TOKEN_EXACT, R, K, count.ravel(), valid.ravel(), origin)
    ws = oracle.loss_weights(oracle.SCALE_SAMPLE, R, K, count.ravel(), valid.ravel(), origin)
    differs = 0
    for k in range(K):
        T = sum(int(valid[r, k]) for r in range(R))
        L_star = sum(sum(losses[r, k]) for r in range(R)) / T
        means = [sum(losses[r, k]) / int(valid[r, k]) for r in range(R)]
        got = sum(Fraction(float(w[r, k])) * means[r] for r in range(R))
        assert abs(got - L_star) <= abs(L_star) * Fraction(1, 10 ** 14)
        assert abs(sum(Fraction(float(w[r, k])) for r in range(R)) - 1) <= Fraction(1, 10 ** 15)
        got_s = sum(Fraction(float(ws[r, k])) * means[r] for r in range(R))
        differs += abs(got_s - L_star) > abs(L_star) * Fraction(1, 10 ** 6)
    assert differs == K  # sample-level is biased on every step of this input


def test_sample_level_equals_token_level_iff_equal_tokens_per_sample(oracle):
    """P:65 / App. B: sample-level weighting is exact when t_r / n_r is identical across ranks."""
    R, K = 4, 3
    count = np.array([[1, 2, 3], [4, 1, 2], [2, 2, 2], [3, 5, 1]], np.int32)
    per = np.array([17, 29, 5], np.int32)  # tokens per sample, same on every rank within a step
    valid = count * per[None, :]
    origin = np.tile(np.arange(K, dtype=np.int32), R)
    a = oracle.loss_weights(oracle.SCALE_TOKEN_EXACT, R, K, count.ravel(), valid.ravel(), origin)
    b = oracle.loss_weights(oracle.SCALE_SAMPLE, R, K, count.ravel(), valid.ravel(), origin)
    for r in range(R):
        for k in range(K):
            fr = Fraction(int(count[r, k]), int(count[:, k].sum()))
            assert _close(a[r, k], fr) and _close(b[r, k], fr)


def test_approx_equals_exact_when_alignment_is_a_noop(oracle):
    """"Exact mode uses the primary counts when alignment is a no-op": with every slot its own
    candidate group the approximate estimate n_adj * (t_orig / n_orig) is t itself up to one rounding."""
    rng = np.random.default_rng(3)
    R, K = 6, 50
    count = rng.integers(0, 9, size=(R, K)).astype(np.int32)   # zeros = IDLE slots
    valid = (count * rng.integers(0, 300, size=(R, K))).astype(np.int32)
    origin = np.tile(np.arange(K, dtype=np.int32), R)
    a = oracle.loss_weights(oracle.SCALE_TOKEN_EXACT, R, K, count.ravel(), valid.ravel(), origin)
    b = oracle.loss_weights(oracle.SCALE_TOKEN_APPROX, R, K, count.ravel(), valid.ravel(), origin)
    assert np.allclose(a, b, rtol=1e-14, atol=0)
    # IDLE slots and all-zero steps weigh 0; the other steps sum to 1
    assert (a[count == 0] == 0).all()
    s = a.sum(0)
    dead = valid.sum(0) == 0
    assert (s[dead] == 0).all() and np.allclose(s[~dead], 1.0, rtol=1e-14)


def test_approx_conserves_candidate_tokens(oracle):
    """The approximation redistributes a candidate group's tokens over the groups cut from it:
    sum of n_adj * tbar over those groups = t_orig (so a rank's total is unchanged by the estimate)."""
    wl = I.protocol_workload("unequal", 1)
    plan, out = oracle.run_workload(wl)
    R, K = plan.R, plan.n_steps
    cnt, val, org = plan.grp_count.reshape(R, K), out["grp_valid_tokens"].reshape(R, K), plan.grp_origin.reshape(R, K)
    assert (org != np.arange(K)[None, :]).any(), "the input must exercise split"
    for r in range(R):
        for o in np.unique(org[r]):
            sel = org[r] == o
            n_orig, t_orig = int(cnt[r][sel].sum()), int(val[r][sel].sum())
            if n_orig == 0:
                continue
            est = sum(Fraction(int(n)) * Fraction(t_orig, n_orig) for n in cnt[r][sel])
            assert est == t_orig


@pytest.mark.parametrize("kind,over", [("unequal", {}), ("overflow_multiround", {}), ("empty_rank", {}),
                                       ("audit:longtail", {"buffer_size": 128})])
def test_origin_table_declarative(oracle, kind, over):
    """grp_origin against a description that does not replay the split loop: within a round, a rank's
    slots are runs [head, singleton, singleton, ...]; a slot is its own origin unless it is a singleton
    that directly follows (in the sorted order of the window) the slot before it inside ONE candidate
    group.  Checked through what is unique: (i) origin[k] <= k, origin[origin[k]] = origin[k], same
    round; (ii) slots sharing an origin are consecutive, the non-head ones singletons; (iii) the rows
    of such a run, concatenated, are ascending by (len, id) and fit one candidate group of the rule:
    re-grouping the round's window with the oracle's grouping routine yields a group equal to the run."""
    wl = I.protocol_workload(kind, 4, **over)
    plan, _ = oracle.run_workload(wl, collate=False)
    R, K = plan.R, plan.n_steps
    org = plan.grp_origin.reshape(R, K)
    rnd = plan.grp_round.reshape(R, K)
    cnt = plan.grp_count.reshape(R, K)
    seen_split = False
    for r in range(R):
        lens_r = wl.lengths[wl.rank_ptr[r]:wl.rank_ptr[r + 1]]
        for k in range(K):
            o = org[r, k]
            assert o <= k and org[r, o] == o and rnd[r, o] == rnd[r, k]
            if o != k:
                seen_split = True
                assert cnt[r, k] == 1 and (org[r, o:k + 1] == o).all()
        # re-group each round's emitted window: every run must be one candidate group
        for rd in np.unique(rnd[r]):
            ks = np.flatnonzero(rnd[r] == rd)
            ids = [i for k in ks for i in plan.slot_ids(r, k)]
            if not ids:
                continue
            runs = {}
            for k in ks:
                runs.setdefault(org[r, k], []).extend(plan.slot_ids(r, k).tolist())
            multi = [v for o, v in runs.items() if (org[r, ks] == o).sum() > 1]
            if not multi:
                continue
            # candidates of the window the round actually grouped = emitted ids + ids returned by overflow;
            # overflow and split never happen in the same round on one rank, so here the window is `ids`
            cands = oracle.group_window(wl.params["rule"], wl.params["budget"], lens_r, np.array(sorted(ids), np.int32))
            for v in multi:
                assert v in cands, (r, rd, v)
    if kind == "unequal":
        assert seen_split
