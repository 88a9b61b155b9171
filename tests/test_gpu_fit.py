"""The host fit loop on the CUDA handle: pseudo-events generated from the model on the GPU, x and y fitted back
(the paper's benchmark shape: "model fixed, x and y floating")."""
import numpy as np
import pytest

from paper_1702_06735_b200 import fit as F, workloads as W

pytestmark = pytest.mark.gpu


def test_fit_recovers_generated_mixing_parameters():
    from paper_1702_06735_b200 import binding
    cfg = W.config(2)
    mdl = cfg.model
    truth = W.initial_params(mdl)
    truth.x, truth.y = 0.25, 0.15                                # large enough for 100 000 events to pin them down
    flat = W.flat_model()
    hf = binding.Tddp4(flat)
    hf.set_params(W.flat_params(flat))
    p4n, _, _, _ = hf.generate_n(W.BASE_SEED, W.STREAM_NORM, 400_000, 0, 2.0 * hf.weight_bound(), chunk=1 << 22)
    hg = binding.Tddp4(mdl)
    hg.set_params(truth)
    p4, t, _, _ = hg.generate_n(W.BASE_SEED, W.STREAM_DATA, 100_000, 100_000, 1.2, chunk=1 << 22)
    h = binding.Tddp4(mdl)
    h.load_events(0, p4, t)
    h.load_events(1, p4n)
    start = truth.copy(); start.x, start.y = 0.1, 0.05
    res = F.fit(h, start, free_couplings=None, free_xy=True)
    assert res.success and 0 < res.errors["x"] < 0.05 and 0 < res.errors["y"] < 0.05
    # within 5 sigma of the truth (statistical error of the data + of the 400 000-point normalisation sample)
    assert abs(res.par.x - truth.x) < 5 * res.errors["x"] + 0.01 and abs(res.par.y - truth.y) < 5 * res.errors["y"] + 0.01
    h.set_params(truth)
    assert res.nll <= h.nll() + 1e-6
    # couplings floating as well (gauge: c_0 fixed): converges to a lower NLL than the truth point
    res2 = F.fit(h, start, free_couplings="all_but_first", free_xy=True, hesse=False)
    assert res2.nll <= res.nll + 1e-6 and res2.par.c[0] == start.c[0]
