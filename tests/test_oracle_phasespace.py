"""Pins for G2/G3 (O-9): Raubold-Lynch four-body generation in the oracle."""
import math

import numpy as np
from scipy import integrate

import oracle
from paper_1702_06735_b200 import workloads as W

from helpers import breakup, dot


def _cands(mdl, n, seed=42, stream=0, first=0):
    return oracle.candidates(mdl, W.TAU_D0, seed, stream, first, n)


def test_momentum_conservation_and_mass_shells():
    mdl = W.config(1).model
    p4, t, w, ua = _cands(mdl, 20000)
    P = p4.reshape(4, 4, -1)
    tot = P.sum(0)
    assert np.abs(tot[0] - mdl.m_parent).max() < 1e-12
    assert np.abs(tot[1:]).max() < 1e-12
    for a in range(4):
        m2 = P[a, 0] ** 2 - (P[a, 1:] ** 2).sum(0)
        assert np.abs(m2 - mdl.m_final[a] ** 2).max() < 1e-12
    assert (w >= 0).all() and (t >= 0).all() and ((ua >= 0) & (ua < 1)).all()


def test_invariant_mass_sum_rule():
    mdl = W.config(1).model
    p4, *_ = _cands(mdl, 2000)
    P = p4.reshape(4, 4, -1)
    tot = 0.0
    for i in range(4):
        for j in range(i + 1, 4):
            pij = P[i] + P[j]
            tot = tot + dot(pij, pij)
    assert np.abs(tot - (mdl.m_parent ** 2 + 2 * sum(m * m for m in mdl.m_final))).max() < 1e-12


def test_weight_is_product_of_breakup_momenta_of_the_event():
    mdl = W.config(1).model
    p4, t, w, _ = _cands(mdl, 500)
    P = p4.reshape(4, 4, -1)
    for i in range(0, 500, 7):
        p = P[:, :, i]
        M2 = math.sqrt(dot(p[0] + p[1], p[0] + p[1]))
        M3 = math.sqrt(dot(p[0] + p[1] + p[2], p[0] + p[1] + p[2]))
        ref = (breakup(mdl.m_parent, M3, mdl.m_final[3]) * breakup(M3, M2, mdl.m_final[2])
               * breakup(M2, mdl.m_final[0], mdl.m_final[1]))
        assert abs(w[i] - ref) <= 1e-10 * ref + 1e-15


def test_massless_four_body_volume():
    """<w> * 2^{n-2} pi^{n-1} T^{n-2} / (M (n-2)!) -> (pi/2)^{n-1} M^{2n-4} / ((n-1)! (n-2)!) = pi^3 M^4 / 96
    (BJ:north_star closed form; SURVEY.md 8(c) pins).  4 M samples: MC error ~ 2e-4 relative."""
    mdl = W.Model(m_parent=1.7, m_final=(0.0, 0.0, 0.0, 0.0))
    n = 4_000_000
    _, _, w, _ = _cands(mdl, n)
    M = mdl.m_parent
    T = M
    est = w.mean() * 4 * math.pi ** 3 * T ** 2 / (M * 2)
    err = w.std() / math.sqrt(n) * 4 * math.pi ** 3 * T ** 2 / (M * 2)
    exact = math.pi ** 3 * M ** 4 / 96
    assert abs(est - exact) < 5 * err
    assert err / exact < 5e-4


def test_massive_volume_against_nested_quadrature():
    """<w> T^2 / 2 = int dM2 dM3 p1 p2 p3 over the mass triangle (the Raubold-Lynch measure)."""
    mdl = W.config(1).model
    m = mdl.m_final
    M = mdl.m_parent

    def inner(M3):
        f = lambda M2: breakup(M, M3, m[3]) * breakup(M3, M2, m[2]) * breakup(M2, m[0], m[1])
        return integrate.quad(f, m[0] + m[1], M3 - m[2], epsabs=1e-13, epsrel=1e-11)[0]

    exact = integrate.quad(inner, m[0] + m[1] + m[2], M - m[3], epsabs=1e-13, epsrel=1e-10)[0]
    n = 2_000_000
    _, _, w, _ = _cands(mdl, n)
    T = M - sum(m)
    est = w.mean() * T * T / 2
    err = w.std() / math.sqrt(n) * T * T / 2
    assert abs(est - exact) < 5 * err


def test_flatness_permutation_symmetry_of_the_pions():
    """Lorentz-invariant phase space is symmetric under exchange of the equal-mass pions 1, 2, 3 although
    the generator treats them differently (different decays, different boosts): weighted means of
    s_01, s_02, s_03 must agree, and so must those of s_12, s_13, s_23, and of their squares."""
    mdl = W.config(1).model
    n = 2_000_000
    p4, _, w, _ = _cands(mdl, n)
    P = p4.reshape(4, 4, -1)

    def s(i, j):
        q = P[i] + P[j]
        return dot(q, q)

    for power in (1, 2):
        for group in ([(0, 1), (0, 2), (0, 3)], [(1, 2), (1, 3), (2, 3)]):
            vals, errs = [], []
            for (i, j) in group:
                f = s(i, j) ** power
                mean = (w * f).sum() / w.sum()
                vals.append(mean)
                errs.append((w * (f - mean)).std() / w.mean() / math.sqrt(n))
            for a in range(3):
                for b in range(a + 1, 3):
                    assert abs(vals[a] - vals[b]) < 5 * math.hypot(errs[a], errs[b])


def test_isotropy_of_each_particle():
    mdl = W.config(1).model
    n = 1_000_000
    p4, _, w, _ = _cands(mdl, n)
    P = p4.reshape(4, 4, -1)
    for a in range(4):
        for c in (1, 2, 3):
            f = P[a, c]
            mean = (w * f).sum() / w.sum()
            err = (w * f).std() / w.mean() / math.sqrt(n)
            assert abs(mean) < 5 * err


def test_decay_time_is_exponential():
    mdl = W.config(1).model
    _, t, _, _ = _cands(mdl, 1_000_000)
    tau = W.TAU_D0
    assert abs(t.mean() - tau) < 5 * tau / 1e3
    assert abs((t ** 2).mean() - 2 * tau ** 2) < 5 * math.sqrt(20) * tau ** 2 / 1e3


def test_candidates_are_counter_based():
    mdl = W.config(1).model
    a = _cands(mdl, 100, first=0)
    b = _cands(mdl, 40, first=37)
    for x, y in zip(a, b):
        assert np.array_equal(x[..., 37:77], y)
    c = _cands(mdl, 100, stream=2)
    assert not np.array_equal(a[0], c[0])
