"""Pins of the oracle's decay-time-resolution layer (oracle/resolution.py, O-8, BASELINE config 5) against things other
than itself: mpmath quadrature of the defining convolution and of the window integral (real and complex lambda), the
sigma -> 0 and infinite-window limits, the Faddeeva identity through scipy.special.wofz, and the unit integral of the
normalised PDF over the decay-time window."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import special

import oracle
from oracle import resolution as R
from paper_1702_06735_b200 import workloads as W

import samples

mp.mp.dps = 30
TAU, X, Y = W.TAU_D0, W.X_MIX, W.Y_MIX
LAMS = [complex(l) for l in R.lambdas(X, Y, TAU)] + [complex(2.0, -3.0), complex(0.7, 1.9)]


def gauss(z, s):
    return mp.exp(-z * z / (2 * s * s)) / (s * mp.sqrt(2 * mp.pi))


def h_quad(t, lam, s):
    lam = mp.mpc(lam)
    lo = max(0.0, t - 12 * s)
    pts = [lo, t, t + 12 * s] if t > lo else [lo, t + 12 * s]
    return mp.quad(lambda tp: mp.exp(-lam * tp) * gauss(t - tp, s), pts)


@pytest.mark.parametrize("lam", LAMS)
def test_h_is_the_convolution(lam):
    for t, s in [(0.0, 0.05), (0.02, 0.03), (0.4, 0.08), (-0.1, 0.05), (3.9, 0.03), (1.0, 0.5)]:
        want = complex(h_quad(t, lam, s))
        got = complex(R.h(np.array([t]), lam, np.array([s]))[0])
        assert abs(got - want) <= 2e-13 * abs(want), (t, s, lam)


@pytest.mark.parametrize("lam", LAMS)
def test_window_integral_is_the_integral_of_h(lam):
    for a, b, s in [(0.0, 4.0, 0.05), (0.0, 4.0, 0.08), (0.2, 1.1, 0.03), (-0.3, 0.3, 0.1)]:
        want = complex(mp.quad(lambda t: mp.mpc(*_h_mp(t, lam, s)), np.linspace(a, b, 9).tolist()))
        got = complex((R.H(b, lam, np.array([s])) - R.H(a, lam, np.array([s])))[0])
        assert abs(got - want) <= 1e-12 * abs(want), (a, b, s, lam)


def _h_mp(t, lam, s):
    lam = mp.mpc(lam)
    v = mp.mpf(1) / 2 * mp.exp(lam * lam * s * s / 2 - lam * t) * mp.erfc((lam * s * s - t) / (mp.sqrt(2) * s))
    return v.real, v.imag


def test_limits():
    s = np.array([0.05])
    for lam in LAMS:
        # whole real line: int h = int_0^inf e^{-lam t'} dt' = 1/lam
        got = (R.H(math.inf, lam, s) - R.H(-math.inf, lam, s))[0]
        assert abs(got - 1.0 / lam) < 1e-15 * abs(1.0 / lam)
        # [0, inf): (1 + e^{lam^2 s^2/2} erfc(lam s/sqrt2)) / (2 lam)   (SURVEY O-8 special case)
        got = (R.H(math.inf, lam, s) - R.H(0.0, lam, s))[0]
        want = (1.0 + np.exp(lam * lam * s[0] ** 2 / 2) * special.erfc(lam * s[0] / math.sqrt(2))) / (2 * lam)
        assert abs(got - want) < 1e-14 * abs(want)
        # sigma -> 0, t well inside (0, inf): h -> e^{-lam t}
        for t in (0.3, 2.0):
            got = R.h(np.array([t]), lam, np.array([1e-4]))[0]
            assert abs(got - np.exp(-lam * t)) < 1e-7 * abs(np.exp(-lam * t))
    # sigma -> 0 window integral -> (e^{-lam a} - e^{-lam b})/lam, the no-resolution integrals of the C oracle
    T0 = oracle.time_integrals(X, Y, TAU, 0.5, 3.0)
    T = R.time_integrals(np.array([1e-5]), X, Y, TAU, 0.5, 3.0)[:, 0]
    assert np.max(np.abs(T / T0 - 1.0)) < 1e-9


def test_faddeeva_form():
    """h = 1/2 e^{-t^2/(2 sigma^2)} w(i u), u = (lam sigma^2 - t)/(sqrt2 sigma): the same function through wofz."""
    rng = np.random.default_rng(5)
    t = rng.uniform(0.0, 0.4, 200)
    s = rng.uniform(0.03, 0.08, 200)
    for lam in LAMS:
        u = (lam * s * s - t) / (math.sqrt(2) * s)
        want = 0.5 * np.exp(-t * t / (2 * s * s)) * special.wofz(1j * u)
        got = R.h(t, lam, s)
        ok = np.abs(want) > 1e-250
        assert np.max(np.abs(got[ok] / want[ok] - 1.0)) < 1e-12


def test_time_functions_reduce_to_eq1_without_resolution():
    t = np.array([0.3, 1.0, 2.5])
    psi = R.time_functions(t, np.full(3, 1e-5), X, Y, TAU)
    G = 1.0 / TAU
    want = np.exp(-G * t) * np.stack([np.cosh(Y * G * t), np.cos(X * G * t), np.sinh(Y * G * t), np.sin(X * G * t)])
    assert np.max(np.abs(psi - want) / np.abs(want).max(axis=1, keepdims=True)) < 1e-8
    # larger mixing parameters, so that the sinh and sin components are not tiny
    psi = R.time_functions(t, np.full(3, 1e-5), 0.8, 0.3, TAU)
    want = np.exp(-G * t) * np.stack([np.cosh(.3 * G * t), np.cos(.8 * G * t), np.sinh(.3 * G * t), np.sin(.8 * G * t)])
    assert np.max(np.abs(psi - want)) < 1e-8


def test_pdf_integrates_to_the_phase_space_average():
    """For fixed amplitudes (A, Abar) the time integral of R over the window equals T_1(aa+bb) + T_2(aa-bb) - 2 T_3 Re - 2 T_4 Im
    by construction of N; check it by numerical quadrature of R(t) itself (independent of H)."""
    A, Ab = np.array([0.7 - 0.4j]), np.array([-0.2 + 1.1j])
    s, x, y = np.array([0.06]), 0.4, 0.2
    S = np.array([abs(A[0]) ** 2 + abs(Ab[0]) ** 2, abs(A[0]) ** 2 - abs(Ab[0]) ** 2, (A[0] * np.conj(Ab[0])).real,
                  (A[0] * np.conj(Ab[0])).imag])

    def Rt(t):
        return float(R.prob(A, Ab, S, np.array([float(t)]), s, x, y, TAU, 0.0, 4.0)[1][0])
    total = mp.quad(Rt, np.linspace(0.0, 4.0, 17).tolist())
    N = R.prob(A, Ab, S, np.array([1.0]), s, x, y, TAU, 0.0, 4.0)[2][0]
    assert abs(float(total) / N - 1.0) < 1e-10


def test_nll_with_resolution_brute_force():
    """10 events, mpmath at 30 digits from the C oracle's amplitudes and S_m: the assembly of P_i and the sum."""
    mdl = W.config(5).model
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 5), 10)
    p4n, _ = samples.flat_sample(300)
    rng = np.random.default_rng(11)
    sig = rng.uniform(0.03, 0.08, 10)
    w = rng.uniform(0.5, 1.0, 300)
    t = np.minimum(t, 3.9)
    got, P, st = R.nll(mdl, par, p4, t, sig, p4n, w)
    assert st == 0
    A, Ab = oracle.amplitudes(mdl, par, p4)
    _, S = oracle.norm(mdl, par, p4n, w)
    lams = R.lambdas(par.x, par.y, par.tau)
    total = mp.mpf(0)
    for i in range(10):
        hh = [mp.mpc(*_h_mp(t[i], l, sig[i])) for l in lams]
        II = [mp.quad(lambda tt: mp.mpc(*_h_mp(tt, l, sig[i])), [0, 1, 2, 3, 4]) for l in lams]
        psi = [(hh[0] + hh[1]).real / 2, hh[2].real, (hh[0] - hh[1]).real / 2, hh[2].imag]
        T = [(II[0] + II[1]).real / 2, II[2].real, (II[0] - II[1]).real / 2, II[2].imag]
        a, b = mp.mpc(A[i]), mp.mpc(Ab[i])
        aa, bb, cr = abs(a) ** 2, abs(b) ** 2, a * mp.conj(b)
        Ri = (aa + bb) * psi[0] + (aa - bb) * psi[1] - 2 * cr.real * psi[2] - 2 * cr.imag * psi[3]
        Ni = T[0] * S[0] + T[1] * S[1] - 2 * T[2] * S[2] - 2 * T[3] * S[3]
        assert abs(float(Ri / Ni) / P[i] - 1.0) < 1e-12
        total -= mp.log(Ri / Ni)
    assert abs(float(total) - got) < 1e-12 * abs(got)
