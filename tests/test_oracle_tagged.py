"""Pins of oracle/tagged.py (D0bar-tagged rate) against what eq. (1) and the
mathematics fix, none of which restates its formula: the untagged sum, the no-mixing limit, the time integral by
quadrature, and the 30-digit brute force of test_oracle_bruteforce with the roles of the two amplitudes exchanged."""
import numpy as np
from scipy import integrate

import oracle
from oracle import tagged as OT
from paper_1702_06735_b200 import workloads as W

import samples
from test_oracle_bruteforce import brute_nll


def setup(key=("C", 2), n=40, nn=60):
    mdl = samples.model_of(key)
    par = W.initial_params(mdl)
    par.x, par.y = 0.31, 0.17                    # large mixing: every term of eq. (1) matters
    p4, t, _ = samples.data_sample(key, n)
    p4n, _ = samples.flat_sample(nn)
    return mdl, par, p4, t, p4n


def test_tagged_rates_add_up_to_the_untagged_rate():
    mdl, par, p4, t, _ = setup()
    R, _ = oracle.rate(mdl, par, p4, t)
    A, Ab = oracle.amplitudes(mdl, par, p4)
    Rb = OT.rate_dbar(A, Ab, t, par.x, par.y, par.tau)
    G = 1.0 / par.tau
    untagged = 2.0 * np.exp(-G * t) * ((np.abs(A) ** 2 + np.abs(Ab) ** 2) * np.cosh(par.y * G * t)
                                      - 2.0 * (A * np.conj(Ab)).real * np.sinh(par.y * G * t))
    assert np.max(np.abs((R + Rb) / untagged - 1.0)) < 1e-13
    assert np.all(Rb >= 0.0)


def test_no_mixing_limit_is_the_direct_dbar_decay():
    mdl, par, p4, t, _ = setup()
    par.x = par.y = 0.0
    A, Ab = oracle.amplitudes(mdl, par, p4)
    Rb = OT.rate_dbar(A, Ab, t, 0.0, 0.0, par.tau)
    assert np.max(np.abs(Rb / (2.0 * np.exp(-t / par.tau) * np.abs(Ab) ** 2) - 1.0)) < 1e-14


def test_dbar_normalisation_is_the_time_integral_of_the_dbar_rate():
    mdl, par, p4, t, p4n = setup(nn=12)
    A, Ab = oracle.amplitudes(mdl, par, p4n)
    tot = 0.0
    for j in range(p4n.shape[1]):
        f = lambda tt: float(OT.rate_dbar(A[j:j + 1], Ab[j:j + 1], np.array([tt]), par.x, par.y, par.tau)[0])
        tot += integrate.quad(f, 0.0, 90.0 * par.tau, epsabs=0, epsrel=1e-12, limit=400)[0]   # e^{-90 (1 - y)} < 1e-32
    assert abs(OT.norm_dbar(mdl, par, p4n) / (tot / p4n.shape[1]) - 1.0) < 1e-10


def test_tagged_nll_against_the_brute_force_with_exchanged_roles():
    mdl, par, p4, t, p4n = setup(("C", 1), 10, 25)
    par.x, par.y = W.X_MIX * 40, W.Y_MIX * 30
    swapped = par.copy(); swapped.c, swapped.cbar = par.cbar.copy(), par.c.copy()
    ones = np.ones(p4n.shape[1])
    nll_b, _, P_b = brute_nll(mdl, swapped, p4, t, p4n, ones)         # D0bar events = eq. (1) with the couplings exchanged
    nll_d, _, P_d = brute_nll(mdl, par, p4, t, p4n, ones)
    tag = np.array([1, -1] * 5)
    got, P = OT.nll_tagged(mdl, par, p4, t, tag, p4n)
    ref_P = np.where(tag > 0, np.array([float(v) for v in P_d]), np.array([float(v) for v in P_b]))
    assert np.max(np.abs(P / ref_P - 1.0)) < 1e-12
    assert abs(got + float(np.sum(np.log(ref_P)))) < 1e-12 * abs(got)
