"""Flavour-tagged samples ("D0bar-tagged sample (swap A <-> Abar)").  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Eq. (1) is the rate of a meson produced as a D0 into the final state f, with A_f the direct and
Abar_f the via-mixing amplitude (no CP violation, |q/p| = 1, line 28).  For a meson produced as a
D0bar the two amplitudes exchange their roles; written out,

    Rbar(p, t) = e^{-Gamma t} [ (|Abar|^2 + |A|^2) cosh(y Gamma t) + (|Abar|^2 - |A|^2) cos(x Gamma t)
                                - 2 Re(Abar A*) sinh(y Gamma t) - 2 Im(Abar A*) sin(x Gamma t) ],

i.e. the cos and sin terms change sign with respect to eq. (1) and the cosh and sinh terms do not.  Each tag is its own
normalised density: Nbar = T_1 S_1 - T_2 S_2 - 2 T_3 S_3 + 2 T_4 S_4 with the S_m of O-8.  The NLL of a tagged sample is
the sum over both tags.  The CUDA path needs no extra code for this: a D0bar handle is fed (cbar, c) instead of (c, cbar).

Pins (tests/test_oracle_tagged.py): R + Rbar is the untagged rate 2 e^{-Gamma t}[(|A|^2+|Abar|^2) cosh - 2 Re(A Abar*) sinh]
(no x dependence); x = y = 0 gives 2 e^{-Gamma t}|Abar|^2; Rbar integrates to Nbar (quadrature in t); the 10-event
mpmath brute force of test_oracle_bruteforce with the roles exchanged.
"""
from __future__ import annotations

import math

import numpy as np

import oracle


def rate_dbar(A, Abar, t, x, y, tau):
    """Rbar_i for amplitudes A_i, Abar_i (complex arrays) and decay times t_i."""
    G = 1.0 / tau
    aa, bb = np.abs(A) ** 2, np.abs(Abar) ** 2
    cross = Abar * np.conj(A)
    return np.exp(-G * t) * ((bb + aa) * np.cosh(y * G * t) + (bb - aa) * np.cos(x * G * t)
                             - 2.0 * cross.real * np.sinh(y * G * t) - 2.0 * cross.imag * np.sin(x * G * t))


def norm_dbar(mdl, par, p4_norm, w=None):
    """Nbar from the phase-space sums S_1..S_4 of the D0 convention (S_2 and S_4 are odd under A <-> Abar)."""
    _, S = oracle.norm(mdl, par, p4_norm, w)
    T = oracle.time_integrals(par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    return T[0] * S[0] - T[1] * S[1] - 2.0 * T[2] * S[2] + 2.0 * T[3] * S[3]


def nll_tagged(mdl, par, p4, t, tag, p4_norm, w=None):
    """-sum log P over a sample with tag_i = +1 (D0) or -1 (D0bar).  Returns (nll, P[n])."""
    tag = np.asarray(tag)
    R, _ = oracle.rate(mdl, par, p4, t)
    N, _ = oracle.norm(mdl, par, p4_norm, w)
    A, Ab = oracle.amplitudes(mdl, par, p4)
    Rb = rate_dbar(A, Ab, np.asarray(t, float), par.x, par.y, par.tau)
    Nb = norm_dbar(mdl, par, p4_norm, w)
    P = np.where(tag > 0, R / N, Rb / Nb)
    return -math.fsum(np.log(P)), P
