"""GPU parity of the offline planners (GMT / BMT, App. I; HFG, App. J)
against the CPU oracle, bit for bit: plan tables (global sample ids per slot, wrap-around repetition, rank
striding) and the collated arenas.  Run on the B200 box: ``pytest -m gpu``."""
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


def _run_gpu_offline(P, wl, planner, W, budget, size=0, batch_size=0, shift=1):
    import torch
    dw = Par.DeviceWorkload(wl)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(dw.device)
    d_perm, d_key = t(wl.perm), t(wl.shuffle_key)
    prm = P.make_params(W, budget, rule=P.ODB_RULE_MAXFIT_ASC, shift_labels=shift)
    with P.Odb(prm, max(wl.n_samples, 1)) as ctx:
        P.odb_offline_plan(ctx.h, planner, dw.lengths, wl.n_samples, d_perm=d_perm, d_shuffle_key=d_key, size=size,
                           batch_size=batch_size)
        info = P.odb_plan_query(ctx.h)
        out = P.OutputBuffers.for_plan(W, info, dw.device, fill=Par.SENTINEL)
        P.odb_collate(ctx.h, dw.tokens, dw.sample_ptr, dw.span_ptr, dw.span_lo, dw.span_hi, out.struct)
        torch.cuda.synchronize()
    return info, out


CASES = [  # n, W, budget, bucket, mega, batch size
    (1, 1, 64, 4, 4, 2), (1, 3, 64, 4, 4, 2), (70, 3, 2048, 16, 24, 5), (1000, 8, 4096, 128, 400, 16),
    (5000, 2, 16384, 1000, 5000, 7), (40_000, 8, 16384, 4096, 12_800, 4), (100_000, 5, 8192, 70_000, 3200, 32),
]


@pytest.mark.parametrize("planner", [0, 1, 2])
@pytest.mark.parametrize("case", CASES)
def test_offline_planner_parity(P, oracle, planner, case):
    n, W, budget, bucket, mega, bs = case
    wl = I.offline_workload(W, n, n=n, mean=200.0, cv=1.2, budget=budget)
    size = bucket if planner == 1 else mega
    plan = oracle.OraclePlan.offline(planner, wl.lengths, W, budget=budget, perm=wl.perm, shuffle_key=wl.shuffle_key,
                                     size=size, batch_size=bs)
    toks = wl.tokens()
    ref = plan.collate_all(toks, wl.sample_ptr[:-1], wl.span_ptr, wl.span_lo, wl.span_hi)
    info, out = _run_gpu_offline(P, wl, planner, W, budget, size=size, batch_size=bs)
    Par.compare_plan(plan, info, out)
    Par.compare_full(plan, ref, info, out)
    assert np.array_equal(out.table("grp_origin").cpu().numpy(), plan.grp_origin)


def test_offline_gmt_large_pool(P, oracle):
    """GMT over one pool of 1.2 M samples (the global sort runs as chunk sorts + merge passes, the list ranking in
    global memory): plan tables in full, sampled slots element by element."""
    wl = I.offline_workload(8, 77, n=1_200_000, mean=96.0, cv=0.7, budget=8192)
    plan = oracle.OraclePlan.offline(0, wl.lengths, 8, budget=8192)
    info, out = _run_gpu_offline(P, wl, 0, 8, 8192)
    Par.compare_plan(plan, info, out)
    rng = np.random.default_rng(0)
    pick = sorted(set(rng.integers(0, plan.n_slots, 24).tolist()) | {0, plan.n_slots - 1})
    Par.compare_sampled_slots(wl, plan, out, pick, global_ids=True)
    Par.device_self_consistency(info, out)


def test_offline_bad_length_and_reuse(P, oracle):
    import torch
    wl = I.offline_workload(2, 3, n=300, budget=2048)
    bad = wl.lengths.copy()
    bad[17] = 0
    with P.Odb(P.make_params(2, 2048, rule=1), 300) as ctx:
        with pytest.raises(P.OdbError) as ei:
            P.odb_offline_plan(ctx.h, 0, torch.from_numpy(bad).to("cuda:0"), 300)
        assert ei.value.status == P.ODB_ERR_BAD_LENGTH
    # an ODB run on a context that planned offline before (and back): the offline state does not leak
    dw = Par.DeviceWorkload(wl)
    with P.Odb(Par.gpu_params(wl), 300) as ctx:
        P.odb_offline_plan(ctx.h, 0, dw.lengths, 300)
        a = P.odb_plan_query(ctx.h)
        info = ctx.plan(dw.lengths, wl.rank_ptr)
        plan, _ = oracle.run_workload(wl, collate=False)
        assert info.n_steps == plan.n_steps and info.total_elems == plan.total_elems and a.n_steps > 0
