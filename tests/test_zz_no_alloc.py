"""tddp4_project_static: the Fig. 3 projections through the entry point that allocates nothing --
its histogram scratch is a file-scope device array of the library -- against tddp4_project, the existing path that
cudaMalloc's that scratch per call.  Same kernel, integer counts: the results must be identical, call after call (the
static array keeps the previous call's counts and has to be cleared by each call).  Collected last on purpose."""
import numpy as np
import pytest
import torch

from oracle import projections as OP
from paper_1702_06735_b200 import workloads as W

import samples

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_1702_06735_b200 import binding
    binding.load_library()
    return binding


def ranges():
    return OP.default_ranges(W.M_D0, (W.M_K, W.M_PI, W.M_PI, W.M_PI))


def both_paths(h, p4, n_bins):
    n = p4.shape[1]
    hist_ref, values_ref = h.project(p4, n_bins, ranges(), want_values=True)
    hist = torch.full((5, n_bins), -7, dtype=torch.int64, device="cuda")          # every element has to be written
    values = torch.full((5, n), float("nan"), dtype=torch.float64, device="cuda")
    h.project_static(p4, n_bins, ranges(), hist, values)
    torch.cuda.synchronize()
    assert np.array_equal(hist.cpu().numpy(), hist_ref)                          # integer counts: bit-exact
    assert np.all(hist_ref.sum(axis=1) <= n)
    v, r = values.cpu().numpy(), values_ref.cpu().numpy()
    assert np.max(np.abs(v[:4] - r[:4])) < 1e-11                                  # the tolerances of test_gpu_projections
    assert np.max(np.abs(np.angle(np.exp(1j * (v[4] - r[4]))))) < 1e-10
    return hist_ref


def test_two_calls_in_a_row_match_the_allocating_path(B):
    p4, _, _ = samples.data_sample(("C", 2), 5_003)
    flat, _ = samples.flat_sample(777)
    h = B.Tddp4(samples.model_of(("C", 2)))
    a = torch.from_numpy(np.ascontiguousarray(p4)).cuda()
    b = torch.from_numpy(np.ascontiguousarray(flat)).cuda()
    first = both_paths(h, a, 64)          # fills 5 x 64 counters of the shared array with 5003 events each
    second = both_paths(h, b, 16)         # a smaller sample in fewer bins right after: nothing of the first call may remain
    assert first.sum() == 5 * 5_003 and second.sum() == 5 * 777
    third = both_paths(h, a, 64)          # and the first again, from another handle's point of view unchanged
    assert np.array_equal(third, first)
    h2 = B.Tddp4(samples.model_of(("C", 1)))   # the array belongs to the library, not to a handle
    assert np.array_equal(both_paths(h2, b, 16), second)
    # the oracle's counts, for good measure (exact: none of these events sits on a bin edge at this binning)
    assert np.array_equal(second, OP.histograms(flat, 16, ranges()))


def test_empty_input_and_the_size_limit(B):
    flat, _ = samples.flat_sample(777)
    h = B.Tddp4(samples.model_of(("C", 1)))
    b = torch.from_numpy(np.ascontiguousarray(flat)).cuda()
    hist = torch.full((5, B.PROJECT_STATIC_MAX_BINS), -1, dtype=torch.int64, device="cuda")
    h.project_static(b, B.PROJECT_STATIC_MAX_BINS, ranges(), hist)            # the maximum itself is accepted
    torch.cuda.synchronize()
    ref, _ = h.project(b, B.PROJECT_STATIC_MAX_BINS, ranges())
    assert np.array_equal(hist.cpu().numpy(), ref)
    h.project_static(b[:, :0], 8, ranges(), hist)                               # no events: zeros, not the last call's counts
    torch.cuda.synchronize()
    assert np.all(hist.cpu().numpy().ravel()[:40] == 0)
    too_many = torch.zeros(5, B.PROJECT_STATIC_MAX_BINS + 1, dtype=torch.int64, device="cuda")
    with pytest.raises(B.Tddp4Error, match="TDDP4_PROJECT_STATIC_MAX_BINS"):
        h.project_static(b, B.PROJECT_STATIC_MAX_BINS + 1, ranges(), too_many)
    bad = ranges().copy(); bad[2] = (1.0, 1.0)
    with pytest.raises(B.Tddp4Error):
        h.project_static(b, 16, bad, hist)
