"""Time-integrated variant ("time-integrated variant (drop t)").  TEST INFRASTRUCTURE, NOT THE PRODUCT.

When the decay time is not measured, the density of an event in phase space is eq. (1)
integrated over the decay-time window:  F(p) = T_0 (|A|^2+|Abar|^2) + T_1 (|A|^2-|Abar|^2) - 2 T_2 Re(A Abar*) - 2 T_3 Im(A Abar*)
with T_m the window integrals of e^{-Gamma t}{cosh, cos, sinh, sin} (O-8), normalised by the same form averaged over the
normalisation sample:  P_i = F(p_i) / N,  N = (1/N_n) sum_j w_j F(p_j),  NLL = -sum_i log P_i.
Pins (tests/test_oracle_time_integrated.py): P_i against numerical quadrature in t of the time-dependent oracle
probability, finite differences of the NLL for the gradient, null directions.
"""
from __future__ import annotations

import numpy as np

import oracle
from oracle import gradient as OG


def _forms(mdl, par, p4, coeff):
    col = OG._columns(mdl, par, p4)
    A, Ab = np.asarray(par.c, complex) @ col, np.asarray(par.cbar, complex) @ col
    z = np.stack([A.real, A.imag, Ab.real, Ab.imag])
    return col, z, OG._form(z, coeff[0] + coeff[1], coeff[0] - coeff[1], coeff[2], coeff[3])


def nll(mdl, par, p4, p4_norm, w_norm=None):
    """Returns (nll, N, P[n])."""
    T = oracle.time_integrals(par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    _, _, F = _forms(mdl, par, p4, T)
    _, _, Fn = _forms(mdl, par, p4_norm, T)
    w = np.ones(p4_norm.shape[1]) if w_norm is None else np.asarray(w_norm, float)
    N = np.sum(w * Fn) / p4_norm.shape[1]
    P = F / N
    return float(-np.sum(np.log(P))), float(N), P


def nll_gradient(mdl, par, p4, p4_norm, w_norm=None):
    """(grad[4 K_c + 2], nll) in the layout of oracle.gradient."""
    kc = mdl.n_couplings
    T = oracle.time_integrals(par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    dTdx, dTdy = OG.time_integral_derivatives(par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    w = np.ones(p4_norm.shape[1]) if w_norm is None else np.asarray(w_norm, float)
    n, nn = p4.shape[1], p4_norm.shape[1]
    col, z, F = _forms(mdl, par, p4, T)
    coln, zn, Fn = _forms(mdl, par, p4_norm, T)
    N = np.sum(w * Fn) / nn
    dF = OG._form_grad_z(z, T[0] + T[1], T[0] - T[1], T[2], T[3])
    dN = OG._form_grad_z(zn, T[0] + T[1], T[0] - T[1], T[2], T[3]) * w
    g = np.zeros(4 * kc + 2)
    for k in range(kc):
        for off, (i0, i1) in ((0, (0, 1)), (2 * kc, (2, 3))):
            ar, ai, nr, ni = col[k].real, col[k].imag, coln[k].real, coln[k].imag
            g[off + 2 * k] = -np.sum((dF[i0] * ar + dF[i1] * ai) / F) + n * np.sum(dN[i0] * nr + dN[i1] * ni) / nn / N
            g[off + 2 * k + 1] = -np.sum((-dF[i0] * ai + dF[i1] * ar) / F) + n * np.sum(-dN[i0] * ni + dN[i1] * nr) / nn / N
    for j, dT in enumerate((dTdx, dTdy)):
        Fd = OG._form(z, dT[0] + dT[1], dT[0] - dT[1], dT[2], dT[3])
        Nd = np.sum(w * OG._form(zn, dT[0] + dT[1], dT[0] - dT[1], dT[2], dT[3])) / nn
        g[4 * kc + j] = -np.sum(Fd / F) + n * Nd / N
    return g, float(-np.sum(np.log(F / N)))
