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


def test_sensitivity_scales_with_the_sample_size():
    """The shape of the paper's Table 1 (sigma(x), sigma(y) at 20 000 / 50 000 / 70 000 events fall
    like 1/sqrt(N)): toy ensembles at x = 0.49 %, y = 0.61 % with the config-2 model standing in for the paper's
    unpublished one.  The Hessian errors times sqrt(N) are constant, and the scatter of the fitted values over the
    ensemble agrees with them (pull RMS ~ 1, pull mean ~ 0)."""
    from paper_1702_06735_b200 import binding
    mdl = W.config(2).model
    par = W.initial_params(mdl)
    flat = W.flat_model()
    rows = F.sensitivity_study(binding, mdl, par, sizes=(20_000, 50_000, 70_000), n_toys=50, n_norm=1_000_000,
                               flat_model=flat, flat_par=W.flat_params(flat))
    assert [r["n_events"] for r in rows] == [20_000, 50_000, 70_000] and all(r["n_toys"] >= 48 for r in rows)
    for key in ("sigma_x_hesse", "sigma_y_hesse"):
        scaled = np.array([r[key] * np.sqrt(r["n_events"]) for r in rows])
        assert np.ptp(scaled) < 0.08 * scaled.mean(), (key, scaled)            # sigma sqrt(N) constant
        assert rows[0][key] > rows[1][key] > rows[2][key]
    for r in rows:
        for v in ("x", "y"):
            # ensemble scatter against the Hessian error: the RMS of 50 toys has a relative error of 10 %; the shared
            # normalisation sample adds a common offset, which the pull mean absorbs
            assert 0.6 < r[f"pull_rms_{v}"] < 1.5, r
            assert abs(r[f"pull_mean_{v}"]) < 1.5, r
