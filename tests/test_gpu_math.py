"""Accuracy of the branch-free fp64 primitives (csrc/jit_shared.cuh) the kernels use instead of IEEE division and square
root in their hot loops, against numpy's correctly rounded results: never more than one ulp off, and -- for the forms
that end in a residual correction (sqrt, division) -- correctly rounded for all but a sliver of the arguments."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def ulps(a, ref):
    return np.abs(a - ref) / np.spacing(np.abs(ref))


@pytest.fixture(scope="module")
def handle():
    import torch
    from paper_1702_06735_b200 import binding, workloads as W
    h = binding.Tddp4(W.config(1).model, "cuda:0")
    yield h, torch
    h.close()


def samples(rng, n):
    """Magnitudes over the whole range the kernels see (1e-12 .. 1e12) plus values next to powers of two."""
    x = np.exp(rng.uniform(np.log(1e-12), np.log(1e12), n))
    edge = 2.0 ** rng.integers(-40, 40, n // 8) * (1.0 + rng.integers(-4, 5, n // 8) * 2.0 ** -52)
    return np.concatenate([x, np.abs(edge)])


def test_branch_free_primitives_against_ieee(handle):
    h, torch = handle
    rng = np.random.default_rng(7)
    x = samples(rng, 1 << 20)
    y = samples(rng, 1 << 20) * rng.choice([-1.0, 1.0], x.size)
    dx, dy = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
    rcp = h.math_probe(0, dx).cpu().numpy()
    sq = h.math_probe(1, dx).cpu().numpy()
    rsq = h.math_probe(2, dx).cpu().numpy()
    dv = h.math_probe(3, dx, dy).cpu().numpy()
    assert ulps(rcp, 1.0 / x).max() <= 1.0
    assert ulps(rsq, 1.0 / np.sqrt(x)).max() <= 2.0           # the reference itself carries two roundings
    assert ulps(sq, np.sqrt(x)).max() <= 1.0
    assert ulps(dv, x / y).max() <= 1.0
    assert np.mean(sq != np.sqrt(x)) < 1e-3                   # residual-corrected forms: correctly rounded almost always
    assert np.mean(dv != x / y) < 1e-3
    neg = h.math_probe(0, torch.from_numpy(-x).cuda()).cpu().numpy()
    assert np.array_equal(neg, -rcp)                          # sign symmetric


def test_sqrt_pos_clamps_non_positive_arguments(handle):
    h, torch = handle
    x = torch.tensor([0.0, -1.0, -1e-300, 1e-320, 4.0], dtype=torch.float64, device="cuda")
    out = h.math_probe(1, x).cpu().numpy()
    assert np.array_equal(out, np.array([0.0, 0.0, 0.0, 0.0, 2.0]))
