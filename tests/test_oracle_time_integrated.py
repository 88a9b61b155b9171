"""Pins of the time-integrated oracle (oracle/time_integrated.py)."""
import numpy as np
from scipy import integrate

import oracle
from oracle import time_integrated as TI
from paper_1702_06735_b200 import workloads as W

import samples


def model(t_lo=0.2, t_hi=3.0):
    return W.build_model([1, 2, 3], t_lo=t_lo, t_hi=t_hi)


def test_probability_is_the_time_integral_of_the_time_dependent_one():
    """P_int(p) = int_window R(p, t) dt / N  with R, N of the time-dependent oracle (same window): quadrature in t."""
    mdl = model()
    par = W.initial_params(mdl)
    par.x, par.y = 0.5, 0.2
    p4, _, _ = samples.data_sample(("C", 1), 6)
    p4n, _ = samples.flat_sample(300)
    _, N, P = TI.nll(mdl, par, p4, p4n)
    norm_td, _ = oracle.norm(mdl, par, p4n)
    assert abs(N / norm_td - 1) < 1e-13                        # the same normalisation integral
    for i in range(6):
        one = np.ascontiguousarray(p4[:, i:i + 1])
        f = lambda t: oracle.rate(mdl, par, one, np.array([t]))[0][0]
        val = integrate.quad(f, mdl.t_lo, mdl.t_hi, epsabs=0, epsrel=1e-12)[0]
        assert abs(val / norm_td / P[i] - 1) < 1e-10


def test_gradient_finite_differences_and_null_directions():
    mdl = model(0.0, np.inf)
    par = W.initial_params(mdl)
    par.x, par.y = 0.4, 0.15
    kc = mdl.n_couplings
    p4, _, _ = samples.data_sample(("C", 1), 150)
    p4n, _ = samples.flat_sample(1200)
    w = np.random.default_rng(2).uniform(0.5, 1, 1200)
    g, nll = TI.nll_gradient(mdl, par, p4, p4n, w)
    assert abs(nll - TI.nll(mdl, par, p4, p4n, w)[0]) < 1e-12 * abs(nll)
    th = np.concatenate([np.asarray(par.c).view(float), np.asarray(par.cbar).view(float), [par.x, par.y]])

    def at(v):
        p = par.copy()
        p.c = v[:2 * kc].view(complex).copy(); p.cbar = v[2 * kc:4 * kc].view(complex).copy()
        p.x, p.y = float(v[4 * kc]), float(v[4 * kc + 1])
        return TI.nll(mdl, p, p4, p4n, w)[0]
    for j in range(len(th)):
        h = 1e-5 * max(abs(th[j]), 1e-2)
        v = [at(th + s * h * np.eye(len(th))[j]) for s in (1, -1, 2, -2)]
        fd = (8 * (v[0] - v[1]) - (v[2] - v[3])) / (12 * h)
        assert abs(g[j] - fd) < 1e-6 * abs(fd) + 1e-12 * abs(nll) / h
    gc = g[:4 * kc].view(complex)
    cc = np.concatenate([par.c, par.cbar])
    size = np.sum(np.abs(cc) * np.abs(gc))
    assert abs(np.sum(cc.real * gc.real + cc.imag * gc.imag)) < 1e-11 * size
    assert abs(np.sum(-cc.imag * gc.real + cc.real * gc.imag)) < 1e-11 * size
