"""odb_slot_offsets_static: the entry point for callers that may not allocate device memory.

Some users of libodb do not own the GPU they run on: a data-loading plugin inside a trainer whose framework
has reserved all of HBM for its own allocator, or code in the middle of a training step where cudaMalloc /
cudaFree would stall every stream.  They cannot create an odb_ctx (it allocates), so they get one call that
takes only their own input and output buffers and keeps its working memory (the tile records of the offset
scan) in a fixed array inside the library.  This file checks that call against the regular path
(odb_run -> out.d_grp_offset, info.total_elems): bit for bit, as everywhere else in this suite, since the
result is integer work.  Because every call on a device shares that one array and finds the previous call's
records in it, the check runs several calls back to back, a large table followed by a smaller one and the
large one again.

The file is named test_zz_* so that pytest collects it last: with `-x` a failure here hides no other test.
It needs nothing from the tests before it and passes on its own in a fresh process as well.
"""
import numpy as np
import pytest

import odb_inputs as I
from tests import _parity as Par

GUARD = 8           # spare int64 entries behind the n_slots + 1 the call may write
SENTINEL = -0x5A5A5A5A5A5A5A5B


def _workload(n_ranks, n_per_rank):
    """configs[1]-shaped lengths with a small grouping buffer and budget: many slots, several scan tiles of 1024
    and a ragged last tile."""
    wl = I.make_workload(1, n_ranks=n_ranks, n_per_rank=n_per_rank)
    wl.params["buffer_size"] = 256
    wl.params["budget"] = 2048
    return wl


def test_more_slots_than_the_fixed_scratch_holds_is_refused():
    """The limit is checked before anything touches the GPU, so this runs on a machine without one: one slot more
    than odb_static_max_slots() is ODB_ERR_CAPACITY with a message that names the limit; the pointers (never
    dereferenced) are dummies."""
    import paper_2606_19989_b200 as P
    limit = P.odb_static_max_slots()
    assert limit == 1 << 22
    with pytest.raises(P.OdbError) as ei:
        P.odb_slot_offsets_static(256, 256, limit + 1, 256, stream=0)
    assert ei.value.status == P.ODB_ERR_CAPACITY
    assert str(limit) in str(ei.value)
    with pytest.raises(P.OdbError) as ei:
        P.odb_slot_offsets_static(256, 256, -1, 256, stream=0)
    assert ei.value.status == P.ODB_ERR_INVALID_ARG
    with pytest.raises(P.OdbError) as ei:
        P.odb_slot_offsets_static(256, 256, 4, None, stream=0)
    assert ei.value.status == P.ODB_ERR_INVALID_ARG


@pytest.mark.gpu
def test_static_scratch_offsets_match_the_regular_path_on_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device")
    import paper_2606_19989_b200 as P
    P.load()
    dev = "cuda:0"
    # the regular path (context, library-owned scratch) on two different jobs
    jobs = []
    for n_ranks, n_per_rank in ((8, 4096), (5, 3000)):
        info, out, _ = Par.run_gpu(_workload(n_ranks, n_per_rank), staged=False)
        n = int(info.n_slots)
        assert n > 4 * 1024 and n % 1024 != 0          # several tiles, ragged tail
        want = torch.cat([out.table("grp_offset"), torch.tensor([int(info.total_elems)], dtype=torch.int64, device=dev)])
        jobs.append((out.table("grp_count").clone(), out.table("grp_width").clone(), n, want.clone()))
        del out
    # the entry point without allocation: large, small, large again, then an empty table -- each call finds the
    # tile records of the one before it in the shared array
    empty = (torch.zeros(1, dtype=torch.int32, device=dev), torch.zeros(1, dtype=torch.int32, device=dev), 0,
             torch.zeros(1, dtype=torch.int64, device=dev))
    for count, width, n, want in (jobs[0], jobs[1], jobs[0], empty, jobs[1]):
        got = torch.full((n + 1 + GUARD,), SENTINEL, dtype=torch.int64, device=dev)
        P.odb_slot_offsets_static(count, width, n, got)
        torch.cuda.synchronize()
        assert torch.equal(got[:n + 1], want), "offsets differ from odb_run's at slot %d" % int(
            (got[:n + 1] != want).nonzero()[0])
        assert bool((got[n + 1:] == SENTINEL).all()), "wrote past the n_slots + 1 entries"
        # and, independently of either GPU path, the definition itself
        area = count[:n].cpu().numpy().astype(np.int64) * width[:n].cpu().numpy().astype(np.int64)
        ref = np.concatenate([[0], np.cumsum((area + 15) // 16 * 16)])
        assert np.array_equal(got[:n + 1].cpu().numpy(), ref)
