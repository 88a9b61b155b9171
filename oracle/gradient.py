"""Analytic gradient of the NLL with respect to the couplings and the mixing parameters.
TEST INFRASTRUCTURE, NOT THE PRODUCT.

    grad[0 : 2K_c]      d NLL / d(Re c_0, Im c_0, Re c_1, ...)
    grad[2K_c : 4K_c]   d NLL / d(Re cbar_0, Im cbar_0, ...)
    grad[4K_c], [4K_c+1] d NLL / dx, d NLL / dy

The plain definition written out, in real variables (no complex calculus, no Gram matrix, no caches): with
z = (Re A, Im A, Re Abar, Im Abar) the bracket of eq. (1) is the quadratic form

    B = p (z0^2 + z1^2) + q (z2^2 + z3^2) - 2 sh (z0 z2 + z1 z3) - 2 sn (z1 z2 - z0 z3),
    p = cosh(y G t) + cos(x G t),  q = cosh(y G t) - cos(x G t),  sh = sinh(y G t),  sn = sin(x G t),  G = 1/tau,

A and Abar are linear in the couplings (eq. (2)), and NLL = -sum_i log(e^{-G t_i} B_i / N) with
N = (1/N_n) sum_j w_j [same form with (cosh, cos, sinh, sin) replaced by their time integrals T_0..T_3] (O-8), so

    d NLL / d theta = - sum_i (dB_i/d theta) / B_i + n (dN/d theta) / N .

Pins (tests/test_oracle_gradient.py): central differences of oracle.nll, 30-digit mpmath differentiation of a 5-event
brute-force NLL, the two exact null directions (common phase, common real scale of all couplings), quadrature of the
x- and y-derivatives of the time integrals.
"""
from __future__ import annotations

import numpy as np

import oracle


def _columns(mdl, par, p4):
    """a_kappa[K_c][n] = sum of the term amplitudes a_k that share coupling kappa (O-2)."""
    _, _, a = oracle.terms(mdl, par, p4)
    col = np.zeros((mdl.n_couplings, p4.shape[1]), complex)
    for k, kap in enumerate(mdl.term_coupling):
        col[kap] += a[k]
    return col


def time_integral_derivatives(x, y, tau, t_lo, t_hi):
    """d T_m / dx and d T_m / dy, m = cosh, cos, sinh, sin, from I(lam) = (e^{-lam lo} - e^{-lam hi}) / lam:
    dI/dlam = (-lo e^{-lam lo} + hi e^{-lam hi}) / lam - I / lam, with lam-+ = G(1 -+ y), lam_x = G(1 - i x)."""
    G = 1.0 / tau

    def I_dI(lam):
        elo = np.exp(-lam * t_lo)
        ehi = 0.0 if np.isinf(t_hi) else np.exp(-lam * t_hi)
        hi_term = 0.0 if np.isinf(t_hi) else t_hi * ehi
        I = (elo - ehi) / lam
        return I, (-t_lo * elo + hi_term) / lam - I / lam

    _, dIm = I_dI(G * (1.0 - y))
    _, dIp = I_dI(G * (1.0 + y))
    _, dIx = I_dI(G * (1.0 - 1j * x))
    dTdx = np.array([0.0, (-1j * G * dIx).real, 0.0, (-1j * G * dIx).imag])
    dTdy = np.array([0.5 * (-G * dIm + G * dIp), 0.0, 0.5 * (-G * dIm - G * dIp), 0.0]).real
    return dTdx, dTdy


def _form(z, p, q, sh, sn):
    return (p * (z[0] ** 2 + z[1] ** 2) + q * (z[2] ** 2 + z[3] ** 2) - 2.0 * sh * (z[0] * z[2] + z[1] * z[3])
            - 2.0 * sn * (z[1] * z[2] - z[0] * z[3]))


def _form_grad_z(z, p, q, sh, sn):
    """dB/dz (4 components), each an array over events."""
    return np.stack([2.0 * p * z[0] - 2.0 * sh * z[2] + 2.0 * sn * z[3],
                     2.0 * p * z[1] - 2.0 * sh * z[3] - 2.0 * sn * z[2],
                     2.0 * q * z[2] - 2.0 * sh * z[0] - 2.0 * sn * z[1],
                     2.0 * q * z[3] - 2.0 * sh * z[1] + 2.0 * sn * z[0]])


def nll_gradient(mdl, par, p4, t, p4_norm, w_norm=None):
    """Returns (grad[4 K_c + 2], nll).  Window integrals without resolution only (models with use_resolution = 0)."""
    kc = mdl.n_couplings
    c, cb = np.asarray(par.c, complex), np.asarray(par.cbar, complex)
    G = 1.0 / par.tau
    n = p4.shape[1]
    grad = np.zeros(4 * kc + 2)

    # ---- data term: - sum_i (dB_i / d theta) / B_i ---------------------------------------------------------------------
    col = _columns(mdl, par, p4)
    A, Ab = c @ col, cb @ col
    z = np.stack([A.real, A.imag, Ab.real, Ab.imag])
    u, v = par.y * G * t, par.x * G * t
    ch, sh, cs, sn = np.cosh(u), np.sinh(u), np.cos(v), np.sin(v)
    B = _form(z, ch + cs, ch - cs, sh, sn)
    dBdz = _form_grad_z(z, ch + cs, ch - cs, sh, sn)
    for k in range(kc):
        ar, ai = col[k].real, col[k].imag
        grad[2 * k] -= np.sum((dBdz[0] * ar + dBdz[1] * ai) / B)               # dz/dRe c_k = (Re a, Im a, 0, 0)
        grad[2 * k + 1] -= np.sum((-dBdz[0] * ai + dBdz[1] * ar) / B)          # dz/dIm c_k = (-Im a, Re a, 0, 0)
        grad[2 * kc + 2 * k] -= np.sum((dBdz[2] * ar + dBdz[3] * ai) / B)
        grad[2 * kc + 2 * k + 1] -= np.sum((-dBdz[2] * ai + dBdz[3] * ar) / B)
    # d/dx: cos -> -sin, sin -> cos (times G t); d/dy: cosh -> sinh, sinh -> cosh
    grad[4 * kc] -= np.sum(G * t * _form(z, -sn, sn, 0.0, cs) / B)
    grad[4 * kc + 1] -= np.sum(G * t * _form(z, sh, sh, ch, 0.0) / B)

    # ---- normalisation term: n (dN / d theta) / N, N by direct sum over the normalisation sample ------------------------
    coln = _columns(mdl, par, p4_norm)
    w = np.ones(p4_norm.shape[1]) if w_norm is None else np.asarray(w_norm, float)
    An, Abn = c @ coln, cb @ coln
    zn = np.stack([An.real, An.imag, Abn.real, Abn.imag])
    T = oracle.time_integrals(par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    nn = p4_norm.shape[1]
    N = np.sum(w * _form(zn, T[0] + T[1], T[0] - T[1], T[2], T[3])) / nn
    dNdz = _form_grad_z(zn, T[0] + T[1], T[0] - T[1], T[2], T[3]) * w
    dN = np.zeros(4 * kc + 2)
    for k in range(kc):
        ar, ai = coln[k].real, coln[k].imag
        dN[2 * k] = np.sum(dNdz[0] * ar + dNdz[1] * ai) / nn
        dN[2 * k + 1] = np.sum(-dNdz[0] * ai + dNdz[1] * ar) / nn
        dN[2 * kc + 2 * k] = np.sum(dNdz[2] * ar + dNdz[3] * ai) / nn
        dN[2 * kc + 2 * k + 1] = np.sum(-dNdz[2] * ai + dNdz[3] * ar) / nn
    dTdx, dTdy = time_integral_derivatives(par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    dN[4 * kc] = np.sum(w * _form(zn, dTdx[0] + dTdx[1], dTdx[0] - dTdx[1], dTdx[2], dTdx[3])) / nn
    dN[4 * kc + 1] = np.sum(w * _form(zn, dTdy[0] + dTdy[1], dTdy[0] - dTdy[1], dTdy[2], dTdy[3])) / nn
    grad += n * dN / N

    nll = G * np.sum(t) - np.sum(np.log(B)) + n * np.log(N)
    return grad, float(nll)


def nll_gradient_resolution(mdl, par, p4, t, sigma_t, p4_norm, w_norm=None):
    """The same gradient with per-event Gaussian decay-time resolution (O-8, config 5):
    NLL = -sum_i log(R_i / N_i), R_i the quadratic form with the convolved time functions psi_m(t_i, sigma_i),
    N_i = T_0i S_1 + T_1i S_2 - 2 T_2i S_3 - 2 T_3i S_4 with the per-event window integrals T_mi and the phase-space
    averages S_m (direct sums over the normalisation sample).  Returns (grad[4 K_c + 2], nll)."""
    from oracle import resolution as R
    kc = mdl.n_couplings
    c, cb = np.asarray(par.c, complex), np.asarray(par.cbar, complex)
    grad = np.zeros(4 * kc + 2)
    col = _columns(mdl, par, p4)
    A, Ab = c @ col, cb @ col
    z = np.stack([A.real, A.imag, Ab.real, Ab.imag])
    psi = R.time_functions(t, sigma_t, par.x, par.y, par.tau)
    dpsi_dx, dpsi_dy = R.time_function_derivatives(t, sigma_t, par.x, par.y, par.tau)
    T = R.time_integrals(sigma_t, par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    dT_dx, dT_dy = R.time_integral_derivatives(sigma_t, par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)

    def form_m(zz, f):            # quadratic form with (cosh, cos, sinh, sin)-type coefficients f[0..3]
        return _form(zz, f[0] + f[1], f[0] - f[1], f[2], f[3])

    Rv = form_m(z, psi)
    dRdz = _form_grad_z(z, psi[0] + psi[1], psi[0] - psi[1], psi[2], psi[3])
    # phase-space averages and their z-gradients on the normalisation sample, one per time coefficient
    coln = _columns(mdl, par, p4_norm)
    w = np.ones(p4_norm.shape[1]) if w_norm is None else np.asarray(w_norm, float)
    An, Abn = c @ coln, cb @ coln
    zn = np.stack([An.real, An.imag, Abn.real, Abn.imag])
    nn = p4_norm.shape[1]
    unit = np.eye(4)
    S = np.array([np.sum(w * form_m(zn, unit[m])) / nn for m in range(4)])        # coefficient of T_m in N_i
    Nv = T[0] * S[0] + T[1] * S[1] + T[2] * S[2] + T[3] * S[3]
    Wm = np.array([np.sum(T[m] / Nv) for m in range(4)])                          # sum_i T_mi / N_i
    dSdz = [(_form_grad_z(zn, unit[m][0] + unit[m][1], unit[m][0] - unit[m][1], unit[m][2], unit[m][3]) * w) for m in range(4)]
    for k in range(kc):
        ar, ai = col[k].real, col[k].imag
        nr, ni = coln[k].real, coln[k].imag
        for off, (i0, i1) in ((0, (0, 1)), (2 * kc, (2, 3))):
            grad[off + 2 * k] -= np.sum((dRdz[i0] * ar + dRdz[i1] * ai) / Rv)
            grad[off + 2 * k + 1] -= np.sum((-dRdz[i0] * ai + dRdz[i1] * ar) / Rv)
            for m in range(4):
                grad[off + 2 * k] += Wm[m] * np.sum(dSdz[m][i0] * nr + dSdz[m][i1] * ni) / nn
                grad[off + 2 * k + 1] += Wm[m] * np.sum(-dSdz[m][i0] * ni + dSdz[m][i1] * nr) / nn
    for j, (dpsi, dT) in enumerate(((dpsi_dx, dT_dx), (dpsi_dy, dT_dy))):
        dN = dT[0] * S[0] + dT[1] * S[1] + dT[2] * S[2] + dT[3] * S[3]
        grad[4 * kc + j] = -np.sum(form_m(z, dpsi) / Rv) + np.sum(dN / Nv)
    nll = -np.sum(np.log(Rv / Nv))
    return grad, float(nll)
