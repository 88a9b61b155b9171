"""Pins of oracle/projections.py (the Fig. 3 observables) against what the definitions and the
mathematics fix; none of them restates the oracle's boost-and-cross-product route."""
import numpy as np
from scipy import stats

from oracle import projections as OP
from paper_1702_06735_b200 import workloads as W

import helpers
import samples


def events(n=4_000):
    p4, _ = samples.flat_sample(n)
    return p4


def transform(p4, L):
    """Apply the 4x4 Lorentz matrix L to every particle of every event."""
    out = np.empty_like(p4)
    for a in range(4):
        out[4 * a:4 * a + 4] = L @ p4[4 * a:4 * a + 4]
    return out


def test_lorentz_invariance():
    p4 = events(500)
    ref = OP.observables(p4)
    rng = np.random.default_rng(5)
    for _ in range(4):
        L = helpers.boost_matrix(rng.uniform(-0.5, 0.5, 3)) @ helpers.rotation(rng)
        got = OP.observables(transform(p4, L))
        assert np.max(np.abs(got[:4] - ref[:4])) < 1e-11
        d = np.angle(np.exp(1j * (got[4] - ref[4])))                 # phi is an angle: compare modulo 2 pi
        assert np.max(np.abs(d)) < 1e-10


def test_helicity_cosine_against_the_invariant_closed_form():
    """cos theta = -(E_a E_S - a.S) / (|a||S|) with energies and momenta in the pair's rest frame written through
    Minkowski products: E_a = a.P / M, E_S = S.P / M (a: first daughter, P: pair, S: the other pair)."""
    p4 = events(300)
    obs = OP.observables(p4)
    for k, (pair, other) in ((2, (OP.PAIR12, OP.PAIR34)), (3, (OP.PAIR34, OP.PAIR12))):
        for i in range(p4.shape[1]):
            ev = helpers.event(p4, i)
            a, P, S = ev[pair[0]], ev[pair[0]] + ev[pair[1]], ev[other[0]] + ev[other[1]]
            M2 = helpers.dot(P, P)
            Ea, Es = helpers.dot(a, P) / np.sqrt(M2), helpers.dot(S, P) / np.sqrt(M2)
            ka, ks = np.sqrt(Ea * Ea - helpers.dot(a, a)), np.sqrt(Es * Es - helpers.dot(S, S))
            assert abs(obs[k, i] + (Ea * Es - helpers.dot(a, S)) / (ka * ks)) < 1e-11


def test_masses_are_the_pair_invariant_masses():
    p4 = events(200)
    obs = OP.observables(p4)
    for i in range(p4.shape[1]):
        ev = helpers.event(p4, i)
        P12, P34 = ev[2] + ev[3], ev[0] + ev[1]
        assert abs(obs[0, i] - np.sqrt(helpers.dot(P12, P12))) < 1e-13
        assert abs(obs[1, i] - np.sqrt(helpers.dot(P34, P34))) < 1e-13


def test_parity_and_exchange_symmetries():
    p4 = events(500)
    ref = OP.observables(p4)
    par = p4.copy()
    for a in range(4):
        par[4 * a + 1:4 * a + 4] *= -1.0                               # p_vec -> -p_vec
    got = OP.observables(par)
    assert np.max(np.abs(got[:4] - ref[:4])) < 1e-13                  # masses and helicity cosines are parity even
    assert np.max(np.abs(np.angle(np.exp(1j * (got[4] + ref[4]))))) < 1e-11   # phi is parity odd
    swp = p4.copy()
    swp[8:12], swp[12:16] = p4[12:16], p4[8:12]                       # exchange the two daughters of the (2,3) pair
    got = OP.observables(swp)
    assert np.max(np.abs(got[2] + ref[2])) < 1e-12 and np.max(np.abs(got[3] - ref[3])) < 1e-12
    assert np.max(np.abs(np.angle(np.exp(1j * (got[4] - ref[4] - np.pi))))) < 1e-10    # n12 flips: phi -> phi + pi


def test_planar_event_has_phi_zero_or_pi():
    m = W.M_PI
    def v(px, py, mass):
        return np.array([np.sqrt(mass * mass + px * px + py * py), px, py, 0.0])
    p0, p1 = v(0.3, 0.2, W.M_K), v(0.1, -0.25, m)
    p2 = v(-0.35, 0.15, m)
    p3 = v(-0.05, -0.10, m)                                            # all in the xy plane; boost-invariant statement
    p4 = np.concatenate([p0, p1, p2, p3])[:, None]
    phi = OP.observables(p4)[4, 0]
    assert min(abs(phi), abs(abs(phi) - np.pi)) < 1e-12


def test_flat_phase_space_gives_flat_angles():
    obs = OP.observables(events(20_000))
    for k, lo, hi in ((2, -1.0, 1.0), (3, -1.0, 1.0), (4, -np.pi, np.pi)):
        assert stats.kstest(obs[k], stats.uniform(lo, hi - lo).cdf).pvalue > 1e-3
    m = (W.M_K, W.M_PI, W.M_PI, W.M_PI)
    r = OP.default_ranges(W.M_D0, m)
    assert np.all(obs[0] >= r[0, 0]) and np.all(obs[0] <= r[0, 1]) and np.all(obs[1] >= r[1, 0]) and np.all(obs[1] <= r[1, 1])
    h = OP.histograms(events(20_000), 25, r)
    assert h.shape == (5, 25) and np.all(h.sum(axis=1) == 20_000)
