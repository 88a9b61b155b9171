"""Pins for steps 4-7 (O-1, O-2, O-8): eq. (1), time integrals, normalisation and NLL of the oracle."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_1702_06735_b200 import workloads as W

X, Y, TAU = W.X_MIX, W.Y_MIX, W.TAU_D0
G = 1.0 / TAU


# ------------------------------------------------------------------------------- eq. (1)
def test_no_mixing_limit_is_twice_direct_rate():
    # x = y = 0: cosh = cos = 1, sinh = sin = 0 -> B = 2 |A_f|^2, independent of Abar_f
    A, Ab = 0.7 - 1.1j, -2.0 + 0.3j
    for t in (0.0, 0.3, 2.0):
        assert oracle.bracket(A, Ab, 0.0, 0.0, G, t) == pytest.approx(2 * abs(A) ** 2, rel=1e-15)


def test_equal_and_opposite_amplitudes():
    A = 0.7 - 1.1j
    for t in (0.1, 0.9, 3.0):
        # cbar = c: 2|A|^2 e^{-y Gamma t};  cbar = -c: 2|A|^2 e^{+y Gamma t}
        assert oracle.bracket(A, A, X, Y, G, t) == pytest.approx(2 * abs(A) ** 2 * math.exp(-Y * G * t), rel=1e-13)
        assert oracle.bracket(A, -A, X, Y, G, t) == pytest.approx(2 * abs(A) ** 2 * math.exp(Y * G * t), rel=1e-13)
        # Abar = 0: |A|^2 (cosh + cos)
        assert oracle.bracket(A, 0j, X, Y, G, t) == pytest.approx(
            abs(A) ** 2 * (math.cosh(Y * G * t) + math.cos(X * G * t)), rel=1e-14)
        # A = 0: |Abar|^2 (cosh - cos)
        assert oracle.bracket(0j, A, 0.3, 0.2, G, t) == pytest.approx(
            abs(A) ** 2 * (math.cosh(0.2 * G * t) - math.cos(0.3 * G * t)), rel=1e-12)


def test_cross_term_signs():
    """Both cross terms enter with a minus sign: check against mpmath with large x, y."""
    A, Ab, x, y, t = 0.7 - 1.1j, -2.0 + 0.3j, 0.8, 0.4, 0.37
    a, b = mp.mpc(A), mp.mpc(Ab)
    u, v = y * G * t, x * G * t
    ref = ((abs(a) ** 2 + abs(b) ** 2) * mp.cosh(u) + (abs(a) ** 2 - abs(b) ** 2) * mp.cos(v)
           - 2 * mp.re(a * mp.conj(b)) * mp.sinh(u) - 2 * mp.im(a * mp.conj(b)) * mp.sin(v))
    assert oracle.bracket(A, Ab, x, y, G, t) == pytest.approx(float(ref), rel=1e-13)


def test_bracket_is_non_negative():
    # (cosh + cos)(cosh - cos) = sinh^2 + sin^2 -> B is a positive-semidefinite form in (A, Abar)
    rng = np.random.default_rng(1)
    for _ in range(2000):
        A, Ab = complex(*rng.standard_normal(2)), complex(*rng.standard_normal(2))
        x, y = rng.uniform(-2, 2), rng.uniform(-0.9, 0.9)
        t = rng.exponential(TAU) * 3
        assert oracle.bracket(A, Ab, x, y, G, t) >= -1e-12 * (abs(A) ** 2 + abs(Ab) ** 2) * math.cosh(y * G * t)


# ------------------------------------------------------------------------------- O-8 time integrals
@pytest.mark.parametrize("x,y", [(X, Y), (0.8, 0.4), (0.0, 0.0), (-0.3, -0.2)])
@pytest.mark.parametrize("window", [(0.0, math.inf), (0.0, 4.0), (0.3, 2.5)])
def test_time_integrals_against_quadrature(x, y, window):
    lo, hi = window
    T = oracle.time_integrals(x, y, TAU, lo, hi)
    fs = [lambda t: math.exp(-G * t) * math.cosh(y * G * t), lambda t: math.exp(-G * t) * math.cos(x * G * t),
          lambda t: math.exp(-G * t) * math.sinh(y * G * t), lambda t: math.exp(-G * t) * math.sin(x * G * t)]
    for m, f in enumerate(fs):
        hi_q = min(hi, 80 * TAU / (1 - abs(y)))           # remainder < e^-80: far below the tolerance
        ref = integrate.quad(f, lo, hi_q, epsabs=1e-14, epsrel=1e-13, limit=200)[0]
        assert T[m] == pytest.approx(ref, rel=1e-10, abs=1e-13)


def test_time_integrals_closed_forms_on_half_line():
    T = oracle.time_integrals(X, Y, TAU)
    ref = [TAU / (1 - Y * Y), TAU / (1 + X * X), TAU * Y / (1 - Y * Y), TAU * X / (1 + X * X)]
    assert np.allclose(T, ref, rtol=1e-14, atol=0)


# ------------------------------------------------------------------------------- normalisation
@pytest.fixture(scope="module")
def sample():
    mdl = W.config(1).model
    par = W.initial_params(mdl)
    p4, t, w, ua = oracle.candidates(mdl, par.tau, 5, 0, 0, 3000)
    return mdl, par, p4, t, w


def test_norm_single_term_closed_form(sample):
    # K = 1, cbar = 0: N = |c|^2 <|a|^2> (T1 + T2)
    mdl0, _, p4, t, w = sample
    mdl = W.build_model([1])
    par = W.initial_params(mdl)
    par.cbar[:] = 0
    _, _, a = oracle.terms(mdl, par, p4)
    T = oracle.time_integrals(par.x, par.y, par.tau)
    ref = abs(par.c[0]) ** 2 * math.fsum(np.abs(a[0]) ** 2) / p4.shape[1] * (T[0] + T[1])
    N, S = oracle.norm(mdl, par, p4)
    assert N == pytest.approx(ref, rel=1e-13)


def test_norm_from_gram_matrix_and_scaling(sample):
    mdl, par, p4, t, w = sample
    N, S = oracle.norm(mdl, par, p4, w)
    _, _, a = oracle.terms(mdl, par, p4)
    # columns per coupling, then G_kl = <w a_k a_l^*>
    cols = np.zeros((mdl.n_couplings, p4.shape[1]), complex)
    for k in range(mdl.n_terms):
        cols[mdl.term_coupling[k]] += a[k]
    Gm = (cols * w) @ cols.conj().T / p4.shape[1]
    c, cb = par.c, par.cbar
    nAA = (c @ Gm @ c.conj()).real
    nBB = (cb @ Gm @ cb.conj()).real
    Xc = c @ Gm @ cb.conj()
    T = oracle.time_integrals(par.x, par.y, par.tau)
    ref = T[0] * (nAA + nBB) + T[1] * (nAA - nBB) - 2 * T[2] * Xc.real - 2 * T[3] * Xc.imag
    assert N == pytest.approx(ref, rel=1e-12)
    assert S[0] == pytest.approx(nAA + nBB, rel=1e-12) and S[3] == pytest.approx(Xc.imag, rel=1e-10)
    # N scales as |s|^2 under (c, cbar) -> s (c, cbar); 1/N_n normalisation, not 1/sum w
    p2 = par.copy(); p2.c = par.c * 3.0; p2.cbar = par.cbar * 3.0
    assert oracle.norm(mdl, p2, p4, w)[0] == pytest.approx(9 * N, rel=1e-13)
    assert oracle.norm(mdl, par, p4, 2 * w)[0] == pytest.approx(2 * N, rel=1e-13)


# ------------------------------------------------------------------------------- NLL invariances
def test_nll_invariances(sample):
    mdl, par, p4, t, w = sample
    data, td = p4[:, :400].copy(), t[:400]
    nrm = p4[:, 400:].copy()
    nll0, N0, P0, st = oracle.nll(mdl, par, data, td, nrm)
    assert st == 0 and np.isfinite(nll0) and (P0 > 0).all()
    # global phase and real scale of (c, cbar) drop out of the normalised PDF
    p2 = par.copy(); ph = np.exp(0.83j); p2.c = par.c * ph; p2.cbar = par.cbar * ph
    assert oracle.nll(mdl, p2, data, td, nrm)[0] == pytest.approx(nll0, rel=1e-13)
    p3 = par.copy(); p3.c = par.c * 2.5; p3.cbar = par.cbar * 2.5
    assert oracle.nll(mdl, p3, data, td, nrm)[0] == pytest.approx(nll0, rel=1e-13)
    # permutation of events
    perm = np.random.default_rng(0).permutation(400)
    assert oracle.nll(mdl, par, data[:, perm].copy(), td[perm], nrm)[0] == pytest.approx(nll0, rel=1e-13)
    # NLL = -sum log P_i with P_i = R_i / N
    R, B = oracle.rate(mdl, par, data, td)
    assert np.allclose(P0, R / N0, rtol=1e-15)
    assert nll0 == pytest.approx(-math.fsum(np.log(R / N0)), rel=1e-14)
    assert np.allclose(R, np.exp(-td / par.tau) * B, rtol=1e-15)


def test_amplitude_is_coupling_weighted_sum_of_terms(sample):
    mdl, par, p4, t, w = sample
    S, F, a = oracle.terms(mdl, par, p4[:, :50].copy())
    A, Ab = oracle.amplitudes(mdl, par, p4[:, :50].copy())
    refA = sum(par.c[mdl.term_coupling[k]] * a[k] for k in range(mdl.n_terms))
    refB = sum(par.cbar[mdl.term_coupling[k]] * a[k] for k in range(mdl.n_terms))
    assert np.allclose(A, refA, rtol=1e-13) and np.allclose(Ab, refB, rtol=1e-13)


def test_pdf_integrates_to_one_by_importance_sampling():
    """int P d(phase space, unit volume) dt = 1: estimate with an independent flat sample and t ~ Exp(tau):
    <w R(p,t) / (Gamma e^{-Gamma t})> / <w> / N -> 1."""
    mdl = W.config(1).model
    par = W.initial_params(mdl)
    n = 400_000
    p4, t, w, _ = oracle.candidates(mdl, par.tau, 99, 0, 0, n)
    pn, _, wn, _ = oracle.candidates(mdl, par.tau, 77, 2, 0, n)
    N, _ = oracle.norm(mdl, par, pn, wn)
    R, B = oracle.rate(mdl, par, p4, t)
    f = w * B * par.tau / N            # R / (Gamma e^{-Gamma t}) = tau B
    est = f.mean()
    err = math.hypot(f.std() / math.sqrt(n), est * 0.01)   # MC error of numerator and of N (~1 %)
    assert abs(est - 1.0) < 5 * err
