"""hepk_fill_histogram_w2_static (include/hepk.h): the weighted fill with its scratch inside the library, for callers
that cannot allocate.  Its output is compared with the existing path's (hepk_fill_histogram_w2 with a caller's workspace)
on calls in a row that share the library's scratch array: a large histogram first, smaller ones after it, so that
anything a call left behind in the array would show.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

from _util import assert_exact, assert_tol, to_np

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hk():
    from paper_1906_06242_b200 import binding
    binding.lib()
    return binding


def _case(seed, n, nbins, weighted=True):
    rng = np.random.default_rng(seed)
    edges = np.linspace(0, 1000, nbins + 1).astype(np.float32)
    x = (rng.exponential(200, n) - 20).astype(np.float32)
    x[:4] = [np.nan, np.inf, -np.inf, 1000.0]
    w = rng.normal(1, 0.1, n).astype(np.float32) if weighted else None
    cu = lambda a: None if a is None else torch.from_numpy(a).cuda()
    return cu(x), cu(w), cu(edges)


def _compare(hk, x, w, edges, rounds=1):
    nb = edges.numel() - 1
    want = hk.fill_histogram_w2(x, w, edges)
    for _ in range(rounds - 1):
        hk.fill_histogram_w2(x, w, edges, *want)
    got = (torch.zeros(nb + 2, dtype=torch.float32, device="cuda"), torch.zeros(nb + 2, dtype=torch.float32, device="cuda"),
           torch.zeros(nb + 2, dtype=torch.int64, device="cuda"))
    for _ in range(rounds):
        hk.fill_histogram_w2_static(x, w, edges, *got)
    torch.cuda.synchronize()
    assert_exact(to_np(got[2]), to_np(want[2]), "counts")
    assert_tol(to_np(got[0]), to_np(want[0]), "sumw")
    assert_tol(to_np(got[1]), to_np(want[1]), "sumw2")
    assert int(got[2].sum()) == rounds * x.numel()


def test_static_scratch_matches_workspace_path_on_calls_in_a_row(hk):
    assert hk.static_hist_scratch_bytes() == 164096
    # 1. the largest histogram the scratch holds (per-CTA float bins; fills the array)
    _compare(hk, *_case(1, 400_003, 4094))
    # 2. right after it, a small one (lane-private bins): what call 1 left in the array must not show
    _compare(hk, *_case(2, 200_001, 100))
    # 3. few entries (fixed-point bins: the weight range goes through the array's header words), accumulated twice
    _compare(hk, *_case(3, 5_000, 100), rounds=2)
    # 4. unweighted, subset of the outputs
    x, w, edges = _case(4, 70_000, 60, weighted=False)
    counts = torch.zeros(62, dtype=torch.int64, device="cuda")
    hk.fill_histogram_w2_static(x, None, edges, None, None, counts)
    assert_exact(to_np(counts), to_np(hk.fill_histogram_w2(x, None, edges, want=("counts",))[2]))


def test_static_scratch_refuses_what_it_cannot_hold(hk):
    x, w, edges = _case(5, 1000, 4095)
    out = torch.zeros(4097, dtype=torch.float32, device="cuda")
    with pytest.raises(Exception, match="4094"):
        hk.fill_histogram_w2_static(x, w, edges, out, None, None)
    assert float(out.abs().sum()) == 0.0
