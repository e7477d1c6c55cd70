"""GPU test of `fstat_select_topk_noalloc` (include/fstat.h), the top-k selection for callers that cannot allocate GPU
memory: a search pipeline whose own arena already owns the whole device (so a cudaMalloc made by the library on its
behalf would fail), or a follow-up stage in a latency-bound loop (cudaMalloc / cudaFree stall every stream of the
device while they run).  The entry point takes no plan and keeps its only scratch, the per-group maxima, in a fixed
1 MiB array inside the library that every call on the device shares.

What is checked: on two calls in a row -- different row counts and row lengths, the second with smaller values, so that
maxima left behind by the first call would mislead the selection if they were ever read -- the outputs are bit-identical
to the plan-based `fstat_select_topk` (the bar this suite uses for index and selection work) and to a plain sort; and a
request beyond the fixed scratch is refused with FSTAT_ESIZE and a message that says what to do.

The file name sorts last on purpose: pytest -x stops at the first failure, so a failure here hides nothing else.  The
test does not depend on what ran before it (it passes alone in a fresh process, where its first call does the one-time
set-up on the device, and after the rest of the suite)."""
import numpy as np
import pytest

from paper_2201_00451_b200 import synth

pytestmark = pytest.mark.gpu


def _sorted_topk(row, k):
    """Descending value, ties by ascending bin (S15), by a plain stable sort."""
    order = np.lexsort((np.arange(row.size), -row.astype(np.float64)))[:k]
    return row[order], order.astype(np.int32)


def _check(binding, torch, plan, rows, k):
    val = torch.full((rows.shape[0], k), float("nan"), dtype=torch.float32, device="cuda")
    idx = torch.full((rows.shape[0], k), -7, dtype=torch.int32, device="cuda")
    binding.select_topk_noalloc(rows, k, (val, idx))
    ref_val, ref_idx = plan.select_topk(rows, k)             # the existing path: scratch from cudaMalloc, owned by the plan
    torch.cuda.synchronize()
    val, idx, host = val.cpu().numpy(), idx.cpu().numpy(), rows.cpu().numpy()
    np.testing.assert_array_equal(idx, ref_idx.cpu().numpy())
    np.testing.assert_array_equal(val, ref_val.cpu().numpy())
    for r in range(host.shape[0]):
        ev, ei = _sorted_topk(host[r], k)
        np.testing.assert_array_equal(idx[r], ei)
        np.testing.assert_array_equal(val[r], ev)


def test_noalloc_topk_matches_plan_path_on_two_calls_in_a_row():
    import torch
    from paper_2201_00451_b200 import binding
    # two plans only to have the existing path to compare with (their n_bins fixes the row length: 14159 and 1008 bins,
    # both with a ragged last group of 512); the rows are 2F rows of the first plan plus noise rows with exact ties
    p1 = synth.small_problem(seed=7, rho=10.0, n_templates=3, n_samples=20000, n_fft=1 << 15, band=0.4321)
    p2 = synth.small_problem(seed=8, rho=None, n_templates=1, n_samples=5000, n_fft=1 << 13, band=0.123)
    with binding.FstatPlan(p1) as plan1, binding.FstatPlan(p2) as plan2:
        assert plan1.n_bins % 512 and plan2.n_bins % 512
        g = torch.Generator(device="cuda").manual_seed(1234)
        twoF = plan1.compute(p1.templates)
        noise = torch.empty((4, plan1.n_bins), dtype=torch.float32, device="cuda").exponential_(0.5, generator=g) * 2 + 40.0
        noise[1, 100] = noise[1, 9000] = noise[1, 3] = 1.0e3                   # a three-way tie for the loudest bin
        rows_a = torch.cat([twoF, noise]).contiguous()                          # 7 rows, values up to 1e3
        rows_b = torch.empty((2, plan2.n_bins), dtype=torch.float32, device="cuda").exponential_(0.5, generator=g)   # 2 rows, values ~ 1
        _check(binding, torch, plan1, rows_a, 8)          # first call (in a fresh process: does the set-up)
        _check(binding, torch, plan2, rows_b, 64)         # second call reuses the array; none of the stale maxima may leak
        _check(binding, torch, plan1, rows_a[:1], 1)      # and back again, one row, k = 1


def test_noalloc_topk_refuses_what_does_not_fit():
    import torch
    from paper_2201_00451_b200 import binding
    n_bins = 1 << 16                                                       # 128 groups per row
    max_rows = binding.NOALLOC_MAX_GROUPS // 128
    rows = torch.zeros((max_rows + 1, n_bins), dtype=torch.float32, device="cuda")
    val = torch.empty((max_rows + 1, 2), dtype=torch.float32, device="cuda")
    idx = torch.empty((max_rows + 1, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(binding.FstatError) as ei:
        binding.select_topk_noalloc(rows, 2, (val, idx))
    assert ei.value.code == binding.FSTAT_ESIZE and "split" in str(ei.value)
    # exactly the maximum is accepted (all-equal rows: the degenerate all-tie path, bins 0 and 1 win)
    binding.select_topk_noalloc(rows[:max_rows], 2, (val[:max_rows], idx[:max_rows]))
    torch.cuda.synchronize()
    assert (idx[:max_rows].cpu().numpy() == np.array([0, 1], dtype=np.int32)).all()
    with pytest.raises(binding.FstatError) as ei:
        binding.select_topk_noalloc(rows[:1], 65, (torch.empty((1, 65), dtype=torch.float32, device="cuda"),
                                                   torch.empty((1, 65), dtype=torch.int32, device="cuda")))
    assert ei.value.code == binding.FSTAT_EINVAL
