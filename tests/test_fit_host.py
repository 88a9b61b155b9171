"""Host fit loop (paper_1702_06735_b200/fit.py) on CPU: the handle is a stand-in with the two methods the loop uses
(set_params, nll_grad) built on the oracle, so what is under test is the parameter bookkeeping (free-index layout,
scaling, gauge fixing), the minimiser wiring and the error estimate -- not the likelihood."""
import numpy as np

from oracle import gradient as OG
from paper_1702_06735_b200 import fit as F, workloads as W

import samples


class OracleHandle:
    def __init__(self, mdl, p4, t, p4n):
        self.mdl, self.p4, self.t, self.p4n = mdl, p4, t, p4n

    def set_params(self, par):
        self.par = par

    def nll_grad(self):
        g, nll = OG.nll_gradient(self.mdl, self.par, self.p4, self.t, self.p4n)
        return nll, g


def test_free_index_layout():
    assert F.free_indices(3, "all_but_first", True).tolist() == list(range(2, 12)) + [12, 13]
    assert F.free_indices(3, None, True).tolist() == [12, 13]
    assert F.free_indices(2, [0, 5], False).tolist() == [0, 5]


def test_fit_xy_converges_and_reports_errors():
    mdl = samples.model_of(("C", 1))
    truth = W.initial_params(mdl)
    truth.x, truth.y = 0.3, 0.2                                  # large mixing: 600 events constrain it
    p4, t, _ = samples.data_sample(("C", 1), 600)                # generated at the nominal (tiny) x, y: fit just has to converge
    p4n, _ = samples.flat_sample(3000)
    h = OracleHandle(mdl, p4, t, p4n)
    res = F.fit(h, truth, free_couplings=None, free_xy=True)
    assert res.success and res.free.tolist() == [12, 13]
    h.set_params(res.par)
    nll, g = h.nll_grad()
    assert np.max(np.abs(g[res.free])) < 1e-4 * max(1.0, abs(nll)) and nll <= OG.nll_gradient(mdl, truth, p4, t, p4n)[1]
    assert set(res.errors) == {"x", "y"} and all(v > 0 for v in res.errors.values())
    assert np.allclose(res.covariance, res.covariance.T)


def test_fit_couplings_with_gauge_fixed():
    mdl = samples.model_of(("C", 1))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 1), 400)
    p4n, _ = samples.flat_sample(2500)
    h = OracleHandle(mdl, p4, t, p4n)
    start = par.copy(); start.c[1] *= 1.2; start.cbar[2] *= 0.8
    n0 = OG.nll_gradient(mdl, start, p4, t, p4n)[1]
    res = F.fit(h, start, free_couplings="all_but_first", free_xy=False, hesse=False)
    assert res.nll < n0 and res.par.c[0] == start.c[0]           # c_0 is the fixed gauge
    h.set_params(res.par)
    _, g = h.nll_grad()
    assert np.max(np.abs(g[res.free])) < 1e-3
