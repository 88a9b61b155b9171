"""GPU parity of tddp4_nll_grad (analytic gradient in one pass) against oracle/gradient.py.
Tolerance: 1e-10 relative to the largest gradient component (each entry is a sum of n terms of either sign)."""
import numpy as np
import pytest

import oracle
from oracle import gradient as OG
from paper_1702_06735_b200 import workloads as W

import samples

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_1702_06735_b200 import binding
    binding.load_library()
    return binding


def check(h, mdl, par, p4, t, p4n, w=None):
    ref, ref_nll = OG.nll_gradient(mdl, par, p4, t, p4n, w)
    h.set_params(par)
    nll, g = h.nll_grad()
    assert abs(nll - ref_nll) <= 1e-11 * abs(ref_nll)
    assert abs(nll - h.nll()) <= 1e-13 * abs(nll)               # same arithmetic per event; grids may differ
    assert np.max(np.abs(g - ref)) <= 1e-10 * np.abs(ref).max()
    return g


@pytest.mark.parametrize("key,n,nn", [(("C", 1), 1_000, 10_000), (("C", 2), 2_049, 9_001), (("C", 3), 4_097, 20_003)])
def test_gradient_configs(B, key, n, nn):
    mdl = samples.model_of(key)
    p4, t, _ = samples.data_sample(key, n)
    p4n, _ = samples.flat_sample(nn)
    w = np.random.default_rng(9).uniform(0.5, 1.0, nn) if key[1] == 3 else None
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t)
    h.load_events(1, p4n, None, weight=w)
    par = W.initial_params(mdl)
    check(h, mdl, par, p4, t, p4n, w)
    p2 = par.copy(); p2.c[0] *= 1.05; p2.mass[0] *= 1.001        # stale columns and Gram matrix are refreshed first
    check(h, mdl, p2, p4, t, p4n, w)
    p3 = p2.copy(); p3.x, p3.y = 0.9, -0.4                       # full-range time functions
    check(h, mdl, p3, p4, t, p4n, w)


def test_gradient_null_directions_and_window(B):
    mdl = W.build_model(range(1, 9), bose=True, t_lo=0.1, t_hi=3.0)
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 3), 1_500)
    t = np.clip(t, 0.1, 3.0)
    p4n, _ = samples.flat_sample(8_000)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t)
    h.load_events(1, p4n)
    g = check(h, mdl, par, p4, t, p4n)
    kc = mdl.n_couplings
    gc = g[:4 * kc].view(complex)
    cc = np.concatenate([par.c, par.cbar])
    size = np.sum(np.abs(cc) * np.abs(gc))
    assert abs(np.sum(cc.real * gc.real + cc.imag * gc.imag)) < 1e-10 * size      # common scale
    assert abs(np.sum(-cc.imag * gc.real + cc.real * gc.imag)) < 1e-10 * size     # common phase


def test_gradient_matches_finite_differences_of_the_gpu_nll(B):
    """The use case: 2 (4 K_c + 2) batched NLL evaluations against one gradient call."""
    mdl = samples.model_of(("C", 3))
    par = W.initial_params(mdl)
    kc = mdl.n_couplings
    p4, t, _ = samples.data_sample(("C", 3), 3_000)
    p4n, _ = samples.flat_sample(10_000)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t); h.load_events(1, p4n)
    h.set_params(par)
    nll, g = h.nll_grad()
    pts, hs = [], []
    for j in range(4 * kc + 2):
        for s in (+1, -1):
            p = par.copy()
            if j < 2 * kc:
                z = p.c[j // 2]; hstep = 1e-6 * abs(z)
                p.c[j // 2] = z + s * hstep * (1 if j % 2 == 0 else 1j)
            elif j < 4 * kc:
                k = (j - 2 * kc) // 2; z = p.cbar[k]; hstep = 1e-6 * abs(z)
                p.cbar[k] = z + s * hstep * (1 if j % 2 == 0 else 1j)
            elif j == 4 * kc:
                hstep = 1e-6; p.x += s * hstep
            else:
                hstep = 1e-6; p.y += s * hstep
            pts.append(p)
        hs.append(hstep)
    vals, _ = h.nll_batch(h.pack_params(pts))
    fd = (vals[0::2] - vals[1::2]) / (2 * np.array(hs))
    assert np.max(np.abs(fd - g)) < 1e-5 * np.abs(g).max()


@pytest.mark.parametrize("x,y,t_hi", [(W.X_MIX, W.Y_MIX, 4.0), (0.7, -0.3, 4.0), (0.05, 0.02, float("inf"))])
def test_gradient_with_resolution(B, x, y, t_hi):
    """Resolution mode (config 5 model): columns, time rows and their x/y derivative rows in one pass."""
    cfg = W.config(5)
    mdl = W.build_model(range(1, 9), bose=True, t_lo=0.0, t_hi=t_hi, use_resolution=1)
    p4, t_true, _ = samples.data_sample(("C", 5), 1_200)
    t, sig = W.smear_times(t_true, cfg)
    t[:30] = np.linspace(0.0, 0.02, 30)                          # both erfc branches
    p4n, _ = samples.flat_sample(6_000)
    w = W.efficiency_weights(6_000, cfg)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t, sigma_t=sig)
    h.load_events(1, p4n, None, weight=w)
    par = W.initial_params(mdl)
    par.x, par.y = x, y
    for step in range(3):
        ref, ref_nll = OG.nll_gradient_resolution(mdl, par, p4, t, sig, p4n, w)
        h.set_params(par)
        nll, g = h.nll_grad()
        assert abs(nll - ref_nll) <= 1e-11 * abs(ref_nll)
        assert abs(nll - h.nll()) <= 1e-13 * abs(nll)
        assert np.max(np.abs(g - ref)) <= 1e-10 * np.abs(ref).max()
        par = par.copy()
        if step == 0:
            par.c[2] *= 1.03; par.mass[1] *= 1.0005               # stale columns + Gram
        else:
            par.x *= 1.2; par.y *= 0.9                           # stale time rows and derivative rows
