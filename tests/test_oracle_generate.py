"""Pins for G4-G6 (O-9): accept-reject generation of the oracle."""
import math

import numpy as np
import pytest

import oracle
from paper_1702_06735_b200 import workloads as W

from helpers import breakup, dot


def test_generate_is_the_accepted_subset_in_candidate_order():
    mdl = W.config(1).model
    par = W.initial_params(mdl)
    n, pilot = 60_000, 5_000
    g = oracle.generate(mdl, par, 42, 0, n, pilot, 1.2, n)
    rho, ua = oracle.candidate_ratio(mdl, par, 42, 0, 0, n)
    env = 1.2 * rho[:pilot].max()
    assert g["envelope"] == env
    mask = ua * env < rho
    idx = np.nonzero(mask)[0]
    assert g["n_accepted"] == len(idx) and np.array_equal(g["index"], idx)
    assert g["n_overflow"] == int((rho > env).sum())
    p4, t, w, _ = oracle.candidates(mdl, par.tau, 42, 0, 0, n)
    assert np.array_equal(g["p4"], p4[:, idx]) and np.array_equal(g["t"], t[idx])
    assert 0.005 < mask.mean() < 0.5


def test_capacity_overflow_is_reported():
    mdl = W.config(1).model
    par = W.initial_params(mdl)
    full = oracle.generate(mdl, par, 42, 0, 20_000, 2_000, 1.2, 20_000)
    cut = oracle.generate(mdl, par, 42, 0, 20_000, 2_000, 1.2, 10)
    assert cut["status"] == 3 and cut["n_accepted"] == full["n_accepted"] > 10
    assert np.array_equal(cut["p4"], full["p4"][:, :10])


def test_flat_sample_is_unweighted_phase_space():
    """Hit-or-miss on w against the rigorous bound: accepted events carry unit weight, so
    plain means over them equal w-weighted means over raw candidates."""
    mdl = W.flat_model()
    par = W.flat_params(mdl)
    wmax = math.prod(breakup(*tr) for tr in W.flat_envelope_inputs(mdl))
    n = 1_500_000
    g = oracle.generate(mdl, par, 42, W.STREAM_NORM, n, 0, 2.0 * wmax, n)
    assert g["n_overflow"] == 0                       # the bound is rigorous
    p4, _, w, _ = oracle.candidates(mdl, par.tau, 42, W.STREAM_NORM, 0, n)
    assert w.max() <= wmax
    eff = g["n_accepted"] / n
    assert eff == pytest.approx(w.mean() / wmax, rel=0.02)

    def s01(p):
        P = p.reshape(4, 4, -1)
        q = P[0] + P[1]
        return dot(q, q)

    f_acc = s01(g["p4"])
    f_all = s01(p4)
    m_acc, e_acc = f_acc.mean(), f_acc.std() / math.sqrt(len(f_acc))
    m_w = (w * f_all).sum() / w.sum()
    assert abs(m_acc - m_w) < 5 * e_acc


def test_accepted_events_follow_the_model_in_decay_time():
    """With Abar = 0 and x = y = 0 the rate factorises: accepted t ~ Exp(tau); with cbar = -c the rate is
    2|A|^2 e^{-Gamma(1-y)t}, so accepted <t> = tau / (1 - y)."""
    mdl = W.config(1).model
    par = W.initial_params(mdl)
    par.cbar = -par.c
    par.y = 0.3
    g = oracle.generate(mdl, par, 7, 0, 400_000, 20_000, 1.5, 400_000)
    t = g["t"]
    exp = par.tau / (1 - par.y)
    assert abs(t.mean() - exp) < 5 * exp / math.sqrt(len(t))
