"""Pins for step 1 (O-3, O-4): the oracle's index-loop spin factors against independent routes:
Lorentz invariance, closed forms, rest-frame reductions computed with explicit boosts, parity, Bose."""
import math

import numpy as np
import pytest

import oracle
from paper_1702_06735_b200 import workloads as W

from helpers import (L1, boost_matrix, boost_to_rest, breakup, closed_spin_factor, dot, eps4, event, rotation)

PERMS = [(0, 1, 2, 3), (2, 3, 1, 0), (0, 3, 2, 1), (2, 1, 3, 0), (3, 0, 1, 2)]
KINDS = [1, 2, 3, 4, 5, 6]


@pytest.fixture(scope="module")
def events():
    mdl = W.config(1).model
    p4, *_ = oracle.candidates(mdl, W.TAU_D0, 7, 0, 0, 64)
    return [event(p4, i) for i in range(64)]


@pytest.mark.parametrize("sf", KINDS)
def test_closed_forms_match_index_loops(events, sf):
    for p in events[:24]:
        for perm in PERMS:
            a = oracle.spin_factor(sf, perm, p)
            b = closed_spin_factor(sf, perm, p)
            assert a == pytest.approx(b, rel=1e-10, abs=1e-13)


@pytest.mark.parametrize("sf", KINDS)
def test_lorentz_invariance(events, sf):
    rng = np.random.default_rng(3)
    for p in events[:16]:
        ref = oracle.spin_factor(sf, PERMS[0], p)
        for _ in range(3):
            beta = rng.uniform(-0.5, 0.5, 3)
            Lm = boost_matrix(beta) @ rotation(rng)
            assert abs(np.linalg.det(Lm) - 1) < 1e-12          # proper transformation
            q = p @ Lm.T
            assert oracle.spin_factor(sf, PERMS[0], q) == pytest.approx(ref, rel=1e-9, abs=1e-12)


@pytest.mark.parametrize("sf,odd", [(1, False), (2, True), (3, False), (4, False), (5, True), (6, False)])
def test_parity(events, sf, odd):
    flip = np.diag([1.0, -1.0, -1.0, -1.0])
    for p in events[:16]:
        a = oracle.spin_factor(sf, PERMS[0], p)
        b = oracle.spin_factor(sf, PERMS[0], p @ flip)
        assert b == pytest.approx(-a if odd else a, rel=1e-11, abs=1e-14)


@pytest.mark.parametrize("sf", KINDS)
def test_bose_ordering_B_is_ordering_A_on_swapped_pions(events, sf):
    permA = (0, 1, 2, 3)
    permB = (0, 3, 2, 1)
    for p in events[:16]:
        swapped = p[[0, 3, 2, 1]]
        assert oracle.spin_factor(sf, permB, p) == oracle.spin_factor(sf, permA, swapped)


def test_tensor_identities(events):
    """p.L1 = 0; v.v = -4 q*^2; L2 traceless, transverse, L2:L2 = (2/3)(L1.L1)^2 (SURVEY.md 8(c) pins),
    probed through the spin factors themselves: VV-S of a system with itself etc. is not reachable, so the
    identities are checked on helpers.L1 and tied to the oracle through the closed-form test above."""
    for p in events[:8]:
        pV, qV = p[0] + p[1], p[0] - p[1]
        v = L1(pV, qV)
        assert abs(dot(pV, v)) < 1e-13
        qs = breakup(math.sqrt(dot(pV, pV)), W.M_K, W.M_PI)
        assert dot(v, v) == pytest.approx(-4 * qs * qs, rel=1e-12)


def test_rest_frame_reduction_axial(events):
    """S_{AP-S} = -kappa (p_P1 . v) in the rest frame of X (3-vectors), kappa = (m_D^2 + s_X - m_P1^2)/m_D^2."""
    for p in events[:24]:
        for perm in PERMS[:4]:
            r = [p[perm[i]] for i in range(4)]
            pV, qV = r[0] + r[1], r[0] - r[1]
            pX = pV + r[2]
            pD = pX + r[3]
            B = boost_to_rest(pX)
            assert np.abs((B @ pX)[1:]).max() < 1e-12
            v = B @ L1(pV, qV)
            p1 = B @ r[3]
            kappa = (dot(pD, pD) + dot(pX, pX) - dot(r[3], r[3])) / dot(pD, pD)
            ref = -kappa * (p1[1:] @ v[1:])
            assert oracle.spin_factor(4, perm, p) == pytest.approx(ref, rel=1e-10, abs=1e-13)


def test_rest_frame_reduction_tensor(events):
    """S_{TP-D} = -sqrt(s_X) [kappa^2 - 4 p*_D^2/(3 m_D^2)] (p.t)(p.(t x v)) in the rest frame of X."""
    for p in events[:24]:
        for perm in PERMS[:4]:
            r = [p[perm[i]] for i in range(4)]
            pV, qV = r[0] + r[1], r[0] - r[1]
            pX, qX = pV + r[2], pV - r[2]
            pD = pX + r[3]
            B = boost_to_rest(pX)
            v = (B @ L1(pV, qV))[1:]
            t = (B @ L1(pX, qX))[1:]
            p1 = (B @ r[3])[1:]
            mD2, sX = dot(pD, pD), dot(pX, pX)
            kappa = (mD2 + sX - dot(r[3], r[3])) / mD2
            pstar = breakup(math.sqrt(mD2), math.sqrt(sX), math.sqrt(dot(r[3], r[3])))
            ref = -math.sqrt(sX) * (kappa ** 2 - 4 * pstar ** 2 / (3 * mD2)) * (p1 @ t) * (p1 @ np.cross(t, v))
            assert oracle.spin_factor(5, perm, p) == pytest.approx(ref, rel=1e-9, abs=1e-13)


def test_rest_frame_reduction_axial_d_wave(events):
    """S_{AP-D} (axial -> V P in D-wave) in the rest frame of X: the l = 2 tensor of the X decay
    momentum contracted with the bachelor direction and the V polarisation,
    S = -kappa [ (p.t)(t.v) - |t|^2 (p.v) / 3 ], same kappa as the S-wave reduction, all 3-vectors by explicit boosts."""
    for p in events[:24]:
        for perm in PERMS[:4]:
            r = [p[perm[i]] for i in range(4)]
            pV, qV = r[0] + r[1], r[0] - r[1]
            pX, qX = pV + r[2], pV - r[2]
            pD = pX + r[3]
            B = boost_to_rest(pX)
            v = (B @ L1(pV, qV))[1:]
            t = (B @ L1(pX, qX))[1:]
            p1 = (B @ r[3])[1:]
            kappa = (dot(pD, pD) + dot(pX, pX) - dot(r[3], r[3])) / dot(pD, pD)
            ref = -kappa * ((p1 @ t) * (t @ v) - (t @ t) * (p1 @ v) / 3.0)
            assert oracle.spin_factor(6, perm, p) == pytest.approx(ref, rel=1e-9, abs=1e-13)


def test_vv_s_wave_in_rest_frames(events):
    """VV S-wave = v1.v2: each v_i is purely spatial in its own resonance rest frame with |v_i| = 2 q*_i."""
    for p in events[:8]:
        p1, q1 = p[0] + p[1], p[0] - p[1]
        v1 = boost_to_rest(p1) @ L1(p1, q1)
        assert abs(v1[0]) < 1e-12
        assert np.linalg.norm(v1[1:]) == pytest.approx(2 * breakup(math.sqrt(dot(p1, p1)), W.M_K, W.M_PI), rel=1e-12)


def test_parity_odd_times_even_averages_to_zero():
    """<S_even S_odd> = 0 over flat phase space (weights w), within MC error."""
    mdl = W.config(1).model
    n = 200_000
    p4, _, w, _ = oracle.candidates(mdl, W.TAU_D0, 11, 0, 0, n)
    m2 = W.build_model([1, 6])          # VV-S and VV-P on the same systems
    par = W.initial_params(m2)
    S, F, a = oracle.terms(m2, par, p4)
    f = S[0] * S[1]
    mean = (w * f).sum() / w.sum()
    err = (w * f).std() / w.mean() / math.sqrt(n)
    assert abs(mean) < 5 * err
    assert (np.abs(f) > 0).mean() > 0.99          # not trivially zero


def test_eps4_is_determinant():
    rng = np.random.default_rng(0)
    import ctypes as C
    for _ in range(10):
        a, b, c, d = rng.standard_normal((4, 4))
        arr = [x.ctypes.data_as(C.POINTER(C.c_double)) for x in (a, b, c, d)]
        assert oracle.lib().orc_eps4(*arr) == pytest.approx(eps4(a, b, c, d), rel=1e-12, abs=1e-14)
    e = np.eye(4)
    arr = [np.ascontiguousarray(e[i]).ctypes.data_as(C.POINTER(C.c_double)) for i in range(4)]
    assert oracle.lib().orc_eps4(*arr) == 1.0       # eps_{0123} = +1
