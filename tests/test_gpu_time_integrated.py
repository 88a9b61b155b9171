"""GPU parity of the time-integrated mode (use_resolution = 2) against oracle/time_integrated.py."""
import numpy as np
import pytest

from oracle import time_integrated as TI
from paper_1702_06735_b200 import workloads as W

import samples

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("t_lo,t_hi,x,y", [(0.0, float("inf"), W.X_MIX, W.Y_MIX), (0.2, 3.0, 0.6, -0.25)])
def test_time_integrated_nll_and_gradient(t_lo, t_hi, x, y):
    from paper_1702_06735_b200 import binding
    mdl = W.build_model(range(1, 9), bose=True, t_lo=t_lo, t_hi=t_hi, use_resolution=2)
    par = W.initial_params(mdl)
    par.x, par.y = x, y
    p4, _, _ = samples.data_sample(("C", 3), 1_333)
    p4n, _ = samples.flat_sample(5_001)
    w = np.random.default_rng(8).uniform(0.5, 1.0, 5_001)
    h = binding.Tddp4(mdl)
    h.load_events(0, p4)                                         # no decay times
    h.load_events(1, p4n, None, weight=w)
    for step in range(3):
        ref_nll, ref_N, ref_P = TI.nll(mdl, par, p4, p4n, w)
        h.set_params(par)
        prob = h.empty(p4.shape[1])
        nll = h.nll(prob)
        assert np.max(np.abs(prob.cpu().numpy() / ref_P - 1.0)) < 1e-10
        assert abs(nll - ref_nll) <= 1e-11 * max(abs(ref_nll), 1e-3 * float(np.sum(np.abs(np.log(ref_P)))))
        assert abs(h.nll_parts()["norm"] / ref_N - 1.0) < 1e-12
        ref_g, _ = TI.nll_gradient(mdl, par, p4, p4n, w)
        nll_g, g = h.nll_grad()
        assert abs(nll_g - nll) <= 1e-13 * abs(nll)
        assert np.max(np.abs(g - ref_g)) <= 1e-10 * np.abs(ref_g).max()
        par = par.copy()
        if step == 0:
            par.c[1] *= 0.97; par.width[0] *= 1.02
        else:
            par.x *= 1.1; par.y *= 1.2
