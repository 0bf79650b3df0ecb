"""gs_compact_plan_static (include/gs.h): the compaction plan for callers that must not allocate device memory.

Who that is: a SLAM agent that handed out all of its device memory at start-up (a cudaMalloc halfway through a mission
may fail, or eat into a pool the library knows nothing about), and a prune / fuse step (Eq. 22) that runs
while tracking and mapping kernels are busy on other streams (cudaMalloc and cudaFree synchronise the whole device and
would stall them).  For them the scratch of the plan sits in a fixed 64 KiB array inside libgs.so, good for up to
16 777 216 Gaussians, instead of in a buffer the caller has to find room for.

What is checked: index lists and kept counts are bit-identical to gs_compact_plan's (integer work: the tolerance of
tests/test_gpu_optim.py is "bit-exact") on several calls in a row that share the array -- a large map first, then smaller
ones, so that the second call finds the first call's counters still in the scratch; the limit is enforced with
GS_E_TOO_LARGE; and the device's free memory does not move across a call.

This file sorts last on purpose (`pytest --collect-only`): under `pytest -x` a failure here must not hide other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _mask(seed, N, p):
    r = np.random.Generator(np.random.PCG64(seed))
    return np.ascontiguousarray(r.uniform(size=N) < p, np.uint8)


def _plan_with_caller_scratch(b, keep):
    """The existing path: gs_compact_plan with a scratch buffer allocated by the caller."""
    import torch
    lib = b.load_library()
    N = int(keep.numel())
    index = torch.full((N,), -2, dtype=torch.int32, device="cuda")
    n_kept = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    work = torch.empty(max(1, int(lib.gs_compact_work_bytes(N))), dtype=torch.uint8, device="cuda")
    rc = lib.gs_compact_plan(b._stream(), N, b._ptr(keep, torch.uint8), b._ptr(index), b._ptr(n_kept), b._ptr(work))
    assert rc == 0
    torch.cuda.synchronize()
    return index.cpu().numpy().view(np.uint32), int(n_kept.item())


def test_static_scratch_plan_matches_caller_scratch_plan_on_calls_in_a_row():
    import torch
    from paper_2605_10760_b200 import binding as b
    # sizes: several thousand blocks, then fewer (stale counters beyond the new block count stay in the array), a ragged
    # tail, one block, one Gaussian, nothing, then large again
    cases = [(2_000_003, 0.9), (300_000, 0.3), (1025, 0.5), (1024, 1.0), (1, 1.0), (1, 0.0), (0, 0.5), (2_000_003, 0.05)]
    for k, (N, p) in enumerate(cases):
        keep = torch.from_numpy(_mask(900 + k, N, p)).cuda()
        want_index, want_n = _plan_with_caller_scratch(b, keep)
        assert want_n == int(keep.sum().item())
        index = torch.full((N,), -2, dtype=torch.int32, device="cuda")
        n_kept = torch.full((1,), -7, dtype=torch.int64, device="cuda")
        b.gs_compact_plan_static(keep, index, n_kept)
        torch.cuda.synchronize()
        assert int(n_kept.item()) == want_n, (N, p)
        assert np.array_equal(index.cpu().numpy().view(np.uint32), want_index), (N, p)


def test_static_scratch_two_back_to_back_calls_without_a_sync_between_them():
    """Two calls queued on one stream with no host synchronisation in between: stream order alone keeps the second call's
    counters from landing before the first call has read its own."""
    import torch
    from paper_2605_10760_b200 import binding as b
    keep_a = torch.from_numpy(_mask(910, 1_500_000, 0.7)).cuda()
    keep_b = torch.from_numpy(_mask(911, 700_001, 0.2)).cuda()
    want_a, want_b = _plan_with_caller_scratch(b, keep_a), _plan_with_caller_scratch(b, keep_b)
    ia = torch.empty(keep_a.numel(), dtype=torch.int32, device="cuda")
    ib = torch.empty(keep_b.numel(), dtype=torch.int32, device="cuda")
    na = torch.zeros(1, dtype=torch.int64, device="cuda")
    nb = torch.zeros(1, dtype=torch.int64, device="cuda")
    b.gs_compact_plan_static(keep_a, ia, na)        # also the set-up call if this test runs alone
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    b.gs_compact_plan_static(keep_a, ia, na)
    b.gs_compact_plan_static(keep_b, ib, nb)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, (free_before, free_after)   # the calls took no device memory
    assert (int(na.item()), int(nb.item())) == (want_a[1], want_b[1])
    assert np.array_equal(ia.cpu().numpy().view(np.uint32), want_a[0])
    assert np.array_equal(ib.cpu().numpy().view(np.uint32), want_b[0])


def test_static_scratch_limit():
    import torch
    from paper_2605_10760_b200 import binding as b
    lib = b.load_library()
    limit = int(lib.gs_compact_plan_static_max())
    assert limit == 1 << 24
    # exactly at the limit: every counter of the array is in use
    keep = torch.from_numpy(_mask(920, limit, 0.5)).cuda()
    want_index, want_n = _plan_with_caller_scratch(b, keep)
    index = torch.empty(limit, dtype=torch.int32, device="cuda")
    n_kept = torch.zeros(1, dtype=torch.int64, device="cuda")
    b.gs_compact_plan_static(keep, index, n_kept)
    torch.cuda.synchronize()
    assert int(n_kept.item()) == want_n and np.array_equal(index.cpu().numpy().view(np.uint32), want_index)
    # one beyond: refused by the C entry point (nothing launched, outputs untouched) and by the wrapper
    index.fill_(-2)
    n_kept.fill_(-7)
    big = torch.zeros(limit + 1, dtype=torch.uint8, device="cuda")
    rc = lib.gs_compact_plan_static(b._stream(), limit + 1, b._ptr(big), b._ptr(index), b._ptr(n_kept))
    torch.cuda.synchronize()
    assert rc == -6 and b.STATUS[rc] == "GS_E_TOO_LARGE"
    assert int(n_kept.item()) == -7 and int(index[0].item()) == -2 and int(index[-1].item()) == -2
    with pytest.raises(b.GsError, match="exceeds the fixed scratch") as e:
        b.gs_compact_plan_static(big, torch.empty(limit + 1, dtype=torch.int32, device="cuda"), n_kept)
    assert e.value.code == -6
    # bad arguments
    assert lib.gs_compact_plan_static(b._stream(), -1, b._ptr(big), b._ptr(index), b._ptr(n_kept)) == -1
    assert lib.gs_compact_plan_static(b._stream(), 8, None, b._ptr(index), b._ptr(n_kept)) == -1
