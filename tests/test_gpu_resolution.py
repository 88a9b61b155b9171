"""GPU parity of the decay-time-resolution mode (BASELINE config 5, O-8) through the C-ABI against
oracle/resolution.py: per-event P_i at 1e-10, NLL at 1e-11, along coupling, mixing and mass steps."""
import math

import numpy as np
import pytest

import oracle
from oracle import resolution as OR
from paper_1702_06735_b200 import workloads as W

import samples

pytestmark = pytest.mark.gpu
TOL_P, TOL_NLL = 1e-10, 1e-11


@pytest.fixture(scope="module")
def B():
    from paper_1702_06735_b200 import binding
    binding.load_library()
    return binding


def c5_inputs(n, n_norm, cfg=None):
    cfg = cfg or W.config(5)
    p4, t_true, _ = samples.data_sample(("C", 5), n)
    t, sig = W.smear_times(t_true, cfg)
    p4n, _ = samples.flat_sample(n_norm)
    w = W.efficiency_weights(n_norm, cfg)
    return cfg, p4, t, sig, p4n, w


def check(h, mdl, par, p4, t, sig, p4n, w):
    ref, P_ref, st = OR.nll(mdl, par, p4, t, sig, p4n, w)
    assert st == 0
    h.set_params(par)
    prob = h.empty(p4.shape[1])
    got = h.nll(prob)
    assert samples.rel_err(prob.cpu().numpy(), P_ref) < TOL_P
    scale = max(abs(ref), 1e-3 * float(np.sum(np.abs(np.log(P_ref)))))
    assert abs(got - ref) <= TOL_NLL * scale
    assert h.nll() == got
    return got


@pytest.mark.parametrize("n,n_norm", [(1_031, 5_003), (33, 257)])
def test_config5_model(B, n, n_norm):
    cfg, p4, t, sig, p4n, w = c5_inputs(n, n_norm)
    h = B.Tddp4(cfg.model)
    h.load_events(0, p4, t, sigma_t=sig)
    h.load_events(1, p4n, None, weight=w)
    check(h, cfg.model, W.initial_params(cfg.model), p4, t, sig, p4n, w)


def test_trajectory_with_resolution(B):
    """Coupling step (cached columns + cached time rows), x/y/tau steps (time rows rebuilt), mass step (columns and Gram
    rebuilt): each compared with the oracle, and the cached and rebuilt paths agree bit for bit."""
    cfg, p4, t, sig, p4n, w = c5_inputs(700, 3_000)
    mdl = cfg.model
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t, sigma_t=sig)
    h.load_events(1, p4n, None, weight=w)
    par = W.initial_params(mdl)
    first = check(h, mdl, par, p4, t, sig, p4n, w)
    p2 = par.copy(); p2.c[3] *= 1.02 + 0.01j
    check(h, mdl, p2, p4, t, sig, p4n, w)
    p3 = p2.copy(); p3.x *= 1.3; p3.y *= 0.8
    check(h, mdl, p3, p4, t, sig, p4n, w)
    p4_ = p3.copy(); p4_.tau *= 1.01
    check(h, mdl, p4_, p4, t, sig, p4n, w)
    p5 = p4_.copy(); p5.mass[0] *= 1.001; p5.width[2] *= 0.99
    check(h, mdl, p5, p4, t, sig, p4n, w)
    assert check(h, mdl, par, p4, t, sig, p4n, w) == first       # back to the start: same bits (all caches rebuilt)
    h2 = B.Tddp4(mdl)
    h2.load_events(0, p4, t, sigma_t=sig)
    h2.load_events(1, p4n, None, weight=w)
    h2.set_params(par)
    assert h2.nll() == first


def test_large_mixing_and_edge_times(B):
    """x, y of order one (complex Faddeeva argument far from the imaginary axis), times at the window edges and within a
    fraction of sigma of zero (both branches of the erfc evaluation), infinite upper window edge."""
    cfg = W.config(5)
    for t_hi in (4.0, math.inf):
        mdl = W.build_model(range(1, 9), bose=True, t_lo=0.0, t_hi=t_hi, use_resolution=1)
        p4, _, _ = samples.data_sample(("C", 5), 300)
        p4n, _ = samples.flat_sample(2_000)
        rng = np.random.default_rng(3)
        sig = rng.uniform(0.03, 0.08, 300)
        t = rng.uniform(0.0, 3.9, 300)
        t[:40] = rng.uniform(0.0, 0.02, 40)
        t[40] = 0.0
        t[41] = 4.0 if math.isfinite(t_hi) else 9.0
        h = B.Tddp4(mdl)
        h.load_events(0, p4, t, sigma_t=sig)
        h.load_events(1, p4n)
        for x, y in [(0.0049, 0.0061), (0.8, 0.3), (-2.5, -0.6), (0.0, 0.0)]:
            par = W.initial_params(mdl)
            par.x, par.y = x, y
            check(h, mdl, par, p4, t, sig, p4n, None)


def test_resolution_errors_and_sharded_wrapper(B):
    from paper_1702_06735_b200 import sharded
    cfg, p4, t, sig, p4n, w = c5_inputs(200, 1_000)
    h = B.Tddp4(cfg.model)
    with pytest.raises(B.Tddp4Error) as e:
        h.load_events(0, p4, t)                                  # sigma_t missing
    assert e.value.code == -1
    h.load_events(0, p4, t, sigma_t=sig)
    h.load_events(1, p4n, None, weight=w)
    par = W.initial_params(cfg.model)
    h.set_params(par)
    direct = h.nll()
    sh = sharded.ShardedNLL(h)
    sh.set_params(par)
    assert sh.nll() == direct
    bad = sig.copy(); bad[5] = 0.0                               # sigma = 0: non-finite P_i, reported as such
    h.load_events(0, p4, t, sigma_t=bad)
    assert h.nll(strict=False) == math.inf
