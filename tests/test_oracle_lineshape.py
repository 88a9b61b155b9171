"""Pins for steps 2 (O-5, O-6): barrier factors and the relativistic Breit-Wigner of the oracle."""
import math

import numpy as np
import pytest

import oracle
from paper_1702_06735_b200 import workloads as W

from helpers import breakup

MK, MPI = W.M_K, W.M_PI


@pytest.mark.parametrize("name,expect_im", [
    # T_R(m0^2) = i / (m0 Gamma0): closed form; values as printed in SURVEY.md 8(c) O-6
    ("K*(892)0", 23.6088), ("rho(770)0", 8.65988), ("a1(1260)", 1.93573), ("K1(1270)", 8.73515)])
def test_bw_at_pole(name, expect_im):
    m0, g0, L = W.RESONANCES[name]
    ma, mb = (MK, MPI) if name.startswith("K*") else (MPI, MPI) if name.startswith("rho") else (0.775, MPI) \
        if name.startswith("a1") else (0.8955, MPI)
    T = oracle.breit_wigner(m0, g0, L, 1.5, m0 * m0, ma, mb)
    assert abs(T.real) < 1e-9
    assert T.imag == pytest.approx(1.0 / (m0 * g0), rel=1e-13)
    assert T.imag == pytest.approx(expect_im, rel=2e-6)


def _gamma_of_s(m0, g0, L, r, s, ma, mb, ma0=None, mb0=None):
    """Recover Gamma(s) from T: 1/T = m0^2 - s - i m0 Gamma(s)."""
    T = oracle.breit_wigner(m0, g0, L, r, s, ma, mb, ma0, mb0)
    inv = 1.0 / T
    assert inv.real == pytest.approx(m0 * m0 - s, rel=1e-12, abs=1e-13)
    return -inv.imag / m0


@pytest.mark.parametrize("L", [0, 1, 2])
def test_running_width(L):
    m0, g0, r = 0.9, 0.05, 1.5
    assert _gamma_of_s(m0, g0, L, r, m0 * m0, MK, MPI) == pytest.approx(g0, rel=1e-13)
    thr = (MK + MPI) ** 2
    assert _gamma_of_s(m0, g0, L, r, thr * (1 + 1e-12), MK, MPI) < g0 * 1e-4     # closes at threshold
    # independent evaluation of Gamma(s) from its definition (O-6) with math.* and helpers.breakup
    for s in (0.5, 0.7, 0.95, 1.4):
        m = math.sqrt(s)
        q, q0 = breakup(m, MK, MPI), breakup(m0, MK, MPI)
        F = {0: lambda z: 1.0, 1: lambda z: 1 / math.sqrt(1 + z), 2: lambda z: 1 / math.sqrt(9 + 3 * z + z * z)}[L]
        ref = g0 * (q / q0) ** (2 * L + 1) * (m0 / m) * (F((q * r) ** 2) / F((q0 * r) ** 2)) ** 2
        assert _gamma_of_s(m0, g0, L, r, s, MK, MPI) == pytest.approx(ref, rel=1e-12)


def test_bw_modulus_peaks_near_pole():
    m0, g0, L = W.RESONANCES["K*(892)0"]
    s = np.linspace(0.45, 1.6, 4001)
    mod = np.array([abs(oracle.breit_wigner(m0, g0, L, 1.5, v, MK, MPI)) for v in s])
    assert abs(math.sqrt(s[mod.argmax()]) - m0) < 0.01


def test_cascade_pole_uses_daughter_pole_mass():
    # a1 -> rho pi: q from the running rho mass, q0 from the rho's current m0 (O-6)
    m0, g0, L = W.RESONANCES["a1(1260)"]
    mrho = 0.775
    # at s = m0^2 with the running daughter mass equal to its pole mass the width is Gamma0 again
    assert _gamma_of_s(m0, g0, L, 1.5, m0 * m0, mrho, MPI, mrho, MPI) == pytest.approx(g0, rel=1e-13)
    # a lighter running daughter opens phase space: Gamma grows as q/q0 for L = 0
    q, q0 = breakup(m0, 0.6, MPI), breakup(m0, mrho, MPI)
    assert _gamma_of_s(m0, g0, L, 1.5, m0 * m0, 0.6, MPI, mrho, MPI) == pytest.approx(g0 * q / q0, rel=1e-12)
    with pytest.raises(ValueError):
        oracle.breit_wigner(0.9, g0, L, 1.5, 1.0, mrho, MPI, mrho, MPI)       # pole below rho pi threshold


def test_barrier_limits():
    assert oracle.barrier(0, 3.7) == 1.0
    assert oracle.barrier(1, 0.0) == 1.0
    assert oracle.barrier(2, 0.0) == pytest.approx(1 / 3, rel=1e-15)
    z = 1e8
    assert oracle.barrier(1, z) == pytest.approx(z ** -0.5, rel=1e-7)
    assert oracle.barrier(2, z) == pytest.approx(1 / z, rel=1e-7)
    for L in (1, 2):
        v = [oracle.barrier(L, z) for z in (0.0, 0.1, 1.0, 10.0)]
        assert all(a > b for a, b in zip(v, v[1:]))


def test_breakup_momentum():
    assert oracle.breakup(1.0, 0.0, 0.0) == 0.5
    assert oracle.breakup(1.0, 0.6, 0.5) == 0.0                       # below threshold: clamped
    assert oracle.breakup(2.0, 0.3, 0.7) == pytest.approx(
        math.sqrt((4 - 1.0) * (4 - 0.16)) / 4, rel=4e-16)             # sqrt(lambda(M^2,a^2,b^2)) / 2M
    assert oracle.breakup(2.0, 0.3, 0.7) == pytest.approx(oracle.breakup(2.0, 0.7, 0.3), rel=1e-15)


def test_constant_width_breit_wigner():
    """Lineshape kind 1 ("further lineshapes"): T = 1 / (m0^2 - s - i m0 Gamma0).  Pole value
    i / (m0 Gamma0); |T|^2 is a Lorentzian in s with half maximum exactly at s = m0^2 +- m0 Gamma0; the phase goes
    through 90 degrees at the pole and T(s) -> -1/s far above it; it equals the running-width form where Gamma(s) = Gamma0."""
    m0, g0 = 1.403, 0.174
    T0 = oracle.breit_wigner_constant(m0, g0, m0 * m0)
    assert abs(T0.real) < 1e-15 and T0.imag == pytest.approx(1.0 / (m0 * g0), rel=1e-15)
    for sgn in (1.0, -1.0):
        T = oracle.breit_wigner_constant(m0, g0, m0 * m0 + sgn * m0 * g0)
        assert abs(T) ** 2 == pytest.approx(0.5 * abs(T0) ** 2, rel=1e-14)
        assert math.degrees(math.atan2(T.imag, T.real)) == pytest.approx(90.0 + sgn * 45.0, abs=1e-10)   # the phase rises through 90 degrees
    assert oracle.breit_wigner_constant(m0, g0, 1e6) == pytest.approx(-1e-6, rel=1e-5)
    assert oracle.breit_wigner_constant(m0, g0, m0 * m0) == pytest.approx(
        oracle.breit_wigner(m0, g0, 0, 1.5, m0 * m0, 0.8955, MPI), rel=1e-14)


def test_per_resonance_radius_and_lineshape_kind_reach_the_term_amplitude():
    """The radius of a resonance enters its own barrier factor and its running width, nothing else; a constant-width
    entry replaces only that resonance's lineshape.  Checked on whole term amplitudes against products rebuilt here from
    the scalar building blocks (breakup momenta from the event's invariant masses)."""
    import samples
    from helpers import dot, event
    p4, _ = samples.flat_sample(40)
    base = W.build_model([1, 3])                       # K* rho (VV S-wave) and K1(1270) -> K* pi
    par = W.initial_params(base)
    iK, iR, iK1 = (base.res_names.index(n) for n in ("K*(892)0", "rho(770)0", "K1(1270)"))
    S0, F0, a0 = oracle.terms(base, par, p4)
    mod = W.build_model([1, 3])
    mod.res_r[iK] = 3.0                                # K* vertex radius 3 GeV^-1, everything else 1.5
    mod.res_lineshape[iK1] = W.LS_CONSTANT
    S1, F1, a1 = oracle.terms(mod, par, p4)
    assert np.array_equal(S0, S1)                      # spin factors do not know about radii or lineshapes
    for i in range(p4.shape[1]):
        ev = event(p4, i)
        sK = dot(ev[0] + ev[1], ev[0] + ev[1]); sR = dot(ev[2] + ev[3], ev[2] + ev[3])
        sX = dot(ev[0] + ev[1] + ev[2], ev[0] + ev[1] + ev[2])
        qK = breakup(math.sqrt(sK), MK, MPI)
        ratio = oracle.barrier(1, (qK * 3.0) ** 2) / oracle.barrier(1, (qK * 1.5) ** 2)
        for k in (0, 1):                               # both chains contain the K* vertex
            assert F1[k, i] == pytest.approx(F0[k, i] * ratio, rel=1e-13)
        TK3 = oracle.breit_wigner(par.mass[iK], par.width[iK], 1, 3.0, sK, MK, MPI)
        TR = oracle.breit_wigner(par.mass[iR], par.width[iR], 1, 1.5, sR, MPI, MPI)
        assert a1[0, i] == pytest.approx(S1[0, i] * F1[0, i] * TK3 * TR, rel=1e-12)
        TK1c = oracle.breit_wigner_constant(par.mass[iK1], par.width[iK1], sX)
        assert a1[1, i] == pytest.approx(S1[1, i] * F1[1, i] * TK1c * TK3, rel=1e-12)
