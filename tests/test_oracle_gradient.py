"""Pins of the oracle's analytic NLL gradient (oracle/gradient.py) against things other than itself."""
import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

import oracle
from oracle import gradient as OG
from paper_1702_06735_b200 import workloads as W

import samples

mp.mp.dps = 30


def theta_get(par, kc):
    return np.concatenate([np.asarray(par.c).view(float), np.asarray(par.cbar).view(float), [par.x, par.y]])


def theta_set(par, th, kc):
    p = par.copy()
    p.c = th[:2 * kc].view(complex).copy()
    p.cbar = th[2 * kc:4 * kc].view(complex).copy()
    p.x, p.y = float(th[4 * kc]), float(th[4 * kc + 1])
    return p


@pytest.mark.parametrize("key,n,nn,x,y", [(("C", 1), 200, 1500, W.X_MIX, W.Y_MIX), (("C", 3), 60, 400, 0.7, 0.25)])
def test_gradient_is_the_derivative_of_the_oracle_nll(key, n, nn, x, y):
    mdl = samples.model_of(key)
    par = W.initial_params(mdl)
    par.x, par.y = x, y
    kc = mdl.n_couplings
    p4, t, _ = samples.data_sample(key, n)
    p4n, _ = samples.flat_sample(nn)
    w = np.random.default_rng(3).uniform(0.5, 1.0, nn)
    g, nll = OG.nll_gradient(mdl, par, p4, t, p4n, w)
    ref = oracle.nll(mdl, par, p4, t, p4n, w, want_prob=False)[0]
    assert abs(nll - ref) < 1e-11 * abs(ref)
    th = theta_get(par, kc)
    for j in range(len(th)):
        h = 1e-5 * max(abs(th[j]), 1e-2)
        vals = []
        for s in (+1, -1, +2, -2):
            tj = th.copy(); tj[j] += s * h
            vals.append(oracle.nll(mdl, theta_set(par, tj, kc), p4, t, p4n, w, want_prob=False)[0])
        fd = (8 * (vals[0] - vals[1]) - (vals[2] - vals[3])) / (12 * h)          # 4th-order central difference
        # rounding noise of the difference quotient ~ 1e-13 |NLL| / h; the tight pin is the mpmath test below
        assert abs(g[j] - fd) < 1e-6 * abs(fd) + 1e-12 * abs(ref) / h, (j, g[j], fd)


def test_null_directions():
    """The PDF is normalised: NLL is invariant under a common phase and a common real scale of ALL couplings, so the
    gradient has exactly zero component along both directions."""
    mdl = samples.model_of(("C", 3))
    par = W.initial_params(mdl)
    kc = mdl.n_couplings
    p4, t, _ = samples.data_sample(("C", 3), 300)
    p4n, _ = samples.flat_sample(2000)
    g, _ = OG.nll_gradient(mdl, par, p4, t, p4n)
    gc = g[:4 * kc].view(complex)                 # g_Re + i g_Im per coupling
    cc = np.concatenate([par.c, par.cbar])
    scale_dir = np.sum(cc.real * gc.real + cc.imag * gc.imag)
    phase_dir = np.sum(-cc.imag * gc.real + cc.real * gc.imag)
    size = np.sum(np.abs(cc) * np.abs(gc))
    assert abs(scale_dir) < 1e-11 * size and abs(phase_dir) < 1e-11 * size


def test_time_integral_derivatives_by_quadrature():
    tau, lo, hi = W.TAU_D0, 0.3, 3.5
    G = 1.0 / tau
    for x, y in [(W.X_MIX, W.Y_MIX), (0.9, 0.35)]:
        dTdx, dTdy = OG.time_integral_derivatives(x, y, tau, lo, hi)
        f = [lambda t: np.exp(-G * t) * G * t * np.sinh(y * G * t), lambda t: -np.exp(-G * t) * G * t * np.sin(x * G * t),
             lambda t: np.exp(-G * t) * G * t * np.cosh(y * G * t), lambda t: np.exp(-G * t) * G * t * np.cos(x * G * t)]
        qy0, qx1, qy2, qx3 = [integrate.quad(fi, lo, hi, epsabs=1e-14, epsrel=1e-13)[0] for fi in f]
        assert np.allclose(dTdy, [qy0, 0.0, qy2, 0.0], rtol=1e-10, atol=1e-14)
        assert np.allclose(dTdx, [0.0, qx1, 0.0, qx3], rtol=1e-10, atol=1e-14)
    dTdx, dTdy = OG.time_integral_derivatives(0.3, 0.2, tau, 0.0, np.inf)        # closed forms on [0, inf)
    x, y = 0.3, 0.2
    assert abs(dTdy[0] - tau * 2 * y / (1 - y * y) ** 2) < 1e-14 and abs(dTdy[2] - tau * (1 + y * y) / (1 - y * y) ** 2) < 1e-14
    assert abs(dTdx[1] + tau * 2 * x / (1 + x * x) ** 2) < 1e-14 and abs(dTdx[3] - tau * (1 - x * x) / (1 + x * x) ** 2) < 1e-14


def test_gradient_brute_force_mpmath():
    """5 data events, 40 normalisation events: the NLL as an mpmath function of all 4 K_c + 2 parameters built from the C
    oracle's per-term amplitudes, differentiated numerically at 30 digits."""
    mdl = samples.model_of(("C", 1))
    par = W.initial_params(mdl)
    par.x, par.y = 0.6, 0.2
    kc = mdl.n_couplings
    p4, t, _ = samples.data_sample(("C", 1), 5)
    p4n, _ = samples.flat_sample(40)
    col = OG._columns(mdl, par, p4)
    coln = OG._columns(mdl, par, p4n)
    G = mp.mpf(1) / mp.mpf(par.tau)

    def nll_mp(*th):
        c = [mp.mpc(th[2 * k], th[2 * k + 1]) for k in range(kc)]
        cb = [mp.mpc(th[2 * kc + 2 * k], th[2 * kc + 2 * k + 1]) for k in range(kc)]
        x, y = th[4 * kc], th[4 * kc + 1]

        def bracket(A, Ab, fch, fcs, fsh, fsn):
            aa, bb, cr = abs(A) ** 2, abs(Ab) ** 2, A * mp.conj(Ab)
            return (aa + bb) * fch + (aa - bb) * fcs - 2 * cr.real * fsh - 2 * cr.imag * fsn
        lm, lp, lx = G * (1 - y), G * (1 + y), G * mp.mpc(1, -x)
        T = [(1 / lm + 1 / lp) / 2, (1 / lx).real, (1 / lm - 1 / lp) / 2, (1 / lx).imag]
        N = mp.mpf(0)
        for j in range(coln.shape[1]):
            A = sum(c[k] * mp.mpc(coln[k, j]) for k in range(kc)); Ab = sum(cb[k] * mp.mpc(coln[k, j]) for k in range(kc))
            N += bracket(A, Ab, *T)
        N /= coln.shape[1]
        tot = mp.mpf(0)
        for i in range(col.shape[1]):
            A = sum(c[k] * mp.mpc(col[k, i]) for k in range(kc)); Ab = sum(cb[k] * mp.mpc(col[k, i]) for k in range(kc))
            ti = mp.mpf(float(t[i]))
            Bi = bracket(A, Ab, mp.cosh(y * G * ti), mp.cos(x * G * ti), mp.sinh(y * G * ti), mp.sin(x * G * ti))
            tot -= mp.log(mp.exp(-G * ti) * Bi / N)
        return tot
    th = [mp.mpf(float(v)) for v in theta_get(par, kc)]
    g, nll = OG.nll_gradient(mdl, par, p4, t, p4n)
    assert abs(float(nll_mp(*th)) - nll) < 1e-12 * abs(nll)
    for j in range(len(th)):
        order = tuple(1 if i == j else 0 for i in range(len(th)))
        d = mp.diff(nll_mp, tuple(th), order)
        assert abs(float(d) - g[j]) < 1e-10 * max(abs(float(d)), 1e-3 * np.abs(g).max()), (j, float(d), g[j])


# ---- resolution mode -------------------------------------------------------------------------------------------------------
def test_resolution_lambda_derivatives_mpmath():
    """d h / d lambda and d H / d lambda against 30-digit numerical differentiation of the mpmath definitions."""
    from oracle import resolution as R

    def h_mp(t, lam, s):
        return mp.mpf(1) / 2 * mp.exp(lam * lam * s * s / 2 - lam * t) * mp.erfc((lam * s * s - t) / (mp.sqrt(2) * s))

    def H_mp(t, lam, s):
        return (mp.erf(t / (mp.sqrt(2) * s)) - 2 * h_mp(t, lam, s)) / (2 * lam)
    for lam in (complex(2.4, 0.0), complex(2.45, -0.012), complex(1.9, -2.2)):
        for t, s in ((0.0, 0.05), (0.03, 0.08), (0.7, 0.03), (4.0, 0.06)):
            want = complex(mp.diff(lambda l: h_mp(mp.mpf(t), l, mp.mpf(s)), mp.mpc(lam)))
            got = complex(R.dh_dlam(np.array([t]), lam, np.array([s]))[0])
            assert abs(got - want) <= 1e-12 * max(abs(want), 1e-6), (lam, t, s)
            want = complex(mp.diff(lambda l: H_mp(mp.mpf(t), l, mp.mpf(s)), mp.mpc(lam)))
            got = complex(R.dH_dlam(t, lam, np.array([s]))[0])
            assert abs(got - want) <= 1e-12 * abs(want), (lam, t, s)
        got = complex(R.dH_dlam(np.inf, lam, np.array([0.05]))[0])
        assert abs(got + 1.0 / (2 * lam * lam)) < 1e-15


@pytest.mark.parametrize("x,y", [(W.X_MIX, W.Y_MIX), (0.6, 0.25)])
def test_resolution_gradient_is_the_derivative_of_the_oracle_nll(x, y):
    from oracle import resolution as R
    cfg = W.config(5)
    mdl = cfg.model
    par = W.initial_params(mdl)
    par.x, par.y = x, y
    kc = mdl.n_couplings
    p4, t_true, _ = samples.data_sample(("C", 5), 80)
    t, sig = W.smear_times(t_true, cfg)
    p4n, _ = samples.flat_sample(500)
    w = W.efficiency_weights(500, cfg)
    g, nll = OG.nll_gradient_resolution(mdl, par, p4, t, sig, p4n, w)
    ref = R.nll(mdl, par, p4, t, sig, p4n, w)[0]
    assert abs(nll - ref) < 1e-11 * abs(ref)
    th = theta_get(par, kc)
    for j in list(range(0, 4 * kc, 5)) + [4 * kc, 4 * kc + 1]:
        h = 1e-5 * max(abs(th[j]), 1e-2)
        vals = []
        for s in (+1, -1, +2, -2):
            tj = th.copy(); tj[j] += s * h
            vals.append(R.nll(mdl, theta_set(par, tj, kc), p4, t, sig, p4n, w)[0])
        fd = (8 * (vals[0] - vals[1]) - (vals[2] - vals[3])) / (12 * h)
        assert abs(g[j] - fd) < 1e-6 * abs(fd) + 1e-12 * abs(ref) / h, (j, g[j], fd)
    gc = g[:4 * kc].view(complex)
    cc = np.concatenate([par.c, par.cbar])
    size = np.sum(np.abs(cc) * np.abs(gc))
    assert abs(np.sum(cc.real * gc.real + cc.imag * gc.imag)) < 1e-11 * size      # common scale
    assert abs(np.sum(-cc.imag * gc.real + cc.real * gc.imag)) < 1e-11 * size     # common phase
