"""Decay-time resolution layer of the oracle (O-8 of DESIGN.md 3, BASELINE config 5).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

The paper ran without resolution; BASELINE.json configs[4] adds a per-event Gaussian resolution
sigma_t "convolved analytically in the time integrals".  Reading (O-8): the true decay time t' >= 0 is
exponentially distributed inside eq. (1), the observed time is t = t' + sigma z, so every
e^{-lambda t'} in eq. (1) is replaced by its convolution with the Gaussian,

    h(t; lambda, sigma) = int_0^inf e^{-lambda t'} Gauss(t - t'; sigma) dt'
                        = 1/2 exp(lambda^2 sigma^2 / 2 - lambda t) erfc((lambda sigma^2 - t) / (sqrt2 sigma)),

with lambda = Gamma(1 -+ y) for the cosh/sinh terms and lambda = Gamma(1 - i x) for the cos/sin terms, and the
normalisation of event i integrates the same functions over the decay-time window [t_lo, t_hi]:

    H(t) = [erf(t / (sqrt2 sigma)) - 2 h(t)] / (2 lambda),      int_a^b h dt = H(b) - H(a).

Everything here is the plain definition written out with numpy; scipy.special.erfc / erf (complex arguments allowed)
serve as the library primitive.  Amplitudes and the phase-space sums S_1..S_4 come from the C oracle.
Pins: tests/test_oracle_resolution.py (mpmath quadrature of the convolution and of the window integral for real and
complex lambda, sigma -> 0 limit, infinite-window limit 1/lambda, unit integral of the normalised PDF).
"""
from __future__ import annotations

import math

import numpy as np
from scipy import special

SQRT2 = math.sqrt(2.0)


def h(t, lam, sigma):
    """Convolved exponential, definition above.  t, sigma: arrays; lam: real or complex scalar."""
    t = np.asarray(t, dtype=np.float64)
    sigma = np.asarray(sigma, dtype=np.float64)
    u = (lam * sigma * sigma - t) / (SQRT2 * sigma)
    return 0.5 * np.exp(lam * lam * sigma * sigma / 2.0 - lam * t) * special.erfc(u)


def H(t, lam, sigma):
    """Antiderivative of h in t.  t may be +inf (h -> 0, erf -> 1) or -inf."""
    sigma = np.asarray(sigma, dtype=np.float64)
    if np.isscalar(t) and math.isinf(t):
        return np.full(sigma.shape, math.copysign(1.0, t) / (2.0 * lam), dtype=np.result_type(lam, np.float64))
    return (special.erf(np.asarray(t, dtype=np.float64) / (SQRT2 * sigma)) - 2.0 * h(t, lam, sigma)) / (2.0 * lam)


def lambdas(x, y, tau):
    G = 1.0 / tau
    return G * (1.0 - y), G * (1.0 + y), G * (1.0 - 1j * x)


def time_functions(t, sigma, x, y, tau):
    """The four functions that replace e^{-Gamma t}{cosh(y Gamma t), cos(x Gamma t), sinh(y Gamma t), sin(x Gamma t)}."""
    lm, lp, lx = lambdas(x, y, tau)
    hm, hp, hx = h(t, lm, sigma), h(t, lp, sigma), h(t, lx, sigma)
    return np.stack([0.5 * (hm + hp), hx.real, 0.5 * (hm - hp), hx.imag])


def time_integrals(sigma, x, y, tau, t_lo, t_hi):
    """Their integrals over the window, per event: [4][n]."""
    lm, lp, lx = lambdas(x, y, tau)
    Im = H(t_hi, lm, sigma) - H(t_lo, lm, sigma)
    Ip = H(t_hi, lp, sigma) - H(t_lo, lp, sigma)
    Ix = H(t_hi, lx, sigma) - H(t_lo, lx, sigma)
    return np.stack([0.5 * (Im + Ip).real, Ix.real, 0.5 * (Im - Ip).real, Ix.imag])


def prob(A, Abar, S, t, sigma, x, y, tau, t_lo, t_hi):
    """P_i = R_i / N_i with R_i the convolved eq. (1) and N_i = T_1 S_1 + T_2 S_2 - 2 T_3 S_3 - 2 T_4 S_4 (O-8)."""
    aa, bb = np.abs(A) ** 2, np.abs(Abar) ** 2
    cross = A * np.conj(Abar)
    psi = time_functions(t, sigma, x, y, tau)
    R = (aa + bb) * psi[0] + (aa - bb) * psi[1] - 2.0 * cross.real * psi[2] - 2.0 * cross.imag * psi[3]
    T = time_integrals(sigma, x, y, tau, t_lo, t_hi)
    N = T[0] * S[0] + T[1] * S[1] - 2.0 * T[2] * S[2] - 2.0 * T[3] * S[3]
    return R / N, R, N


def nll(mdl, par, p4, t, sigma_t, p4_norm, w_norm=None):
    """NLL = -sum_i log P_i with per-event resolution; returns (nll, P[n], status) like oracle.nll."""
    import oracle
    A, Ab = oracle.amplitudes(mdl, par, p4)
    _, S = oracle.norm(mdl, par, p4_norm, w_norm)
    P, _, _ = prob(A, Ab, S, t, sigma_t, par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    if not np.all(np.isfinite(P)) or np.any(P <= 0.0):
        return math.inf, P, 2
    return -math.fsum(np.log(P)), P, 0


# ---- derivatives with respect to the mixing parameters (for the gradient oracle) ---------------------------------------
def dh_dlam(t, lam, sigma):
    """d h / d lambda, the derivative of the definition: with g0 = exp(-t^2 / (2 sigma^2)),
    d/dlambda [1/2 exp(lambda^2 sigma^2/2 - lambda t) erfc(u)] = (lambda sigma^2 - t) h - sigma g0 / sqrt(2 pi)
    (d erfc(u)/du = -2 e^{-u^2}/sqrt(pi), du/dlambda = sigma/sqrt2, and exp(lambda^2 sigma^2/2 - lambda t) e^{-u^2} = g0)."""
    t = np.asarray(t, dtype=np.float64)
    sigma = np.asarray(sigma, dtype=np.float64)
    g0 = np.exp(-t * t / (2.0 * sigma * sigma))
    return (lam * sigma * sigma - t) * h(t, lam, sigma) - sigma * g0 / math.sqrt(2.0 * math.pi)


def dH_dlam(t, lam, sigma):
    """d H / d lambda of H = [erf(t/(sqrt2 sigma)) - 2 h] / (2 lambda):  -H/lambda - (dh/dlambda)/lambda."""
    sigma = np.asarray(sigma, dtype=np.float64)
    if np.isscalar(t) and math.isinf(t):
        return -H(t, lam, sigma) / lam
    return -H(t, lam, sigma) / lam - dh_dlam(t, lam, sigma) / lam


def time_function_derivatives(t, sigma, x, y, tau):
    """(d psi_m / dx, d psi_m / dy), each [4][n]: d lambda_-+ / dy = -+Gamma, d lambda_x / dx = -i Gamma."""
    G = 1.0 / tau
    lm, lp, lx = lambdas(x, y, tau)
    dm, dp, dx = dh_dlam(t, lm, sigma), dh_dlam(t, lp, sigma), -1j * G * dh_dlam(t, lx, sigma)
    z = np.zeros_like(np.asarray(t, dtype=np.float64))
    return (np.stack([z, dx.real, z, dx.imag]),
            np.stack([0.5 * (-G * dm + G * dp).real, z, 0.5 * (-G * dm - G * dp).real, z]))


def time_integral_derivatives(sigma, x, y, tau, t_lo, t_hi):
    """(d T_m / dx, d T_m / dy) of the per-event window integrals, each [4][n]."""
    G = 1.0 / tau
    lm, lp, lx = lambdas(x, y, tau)
    dm = dH_dlam(t_hi, lm, sigma) - dH_dlam(t_lo, lm, sigma)
    dp = dH_dlam(t_hi, lp, sigma) - dH_dlam(t_lo, lp, sigma)
    dx = -1j * G * (dH_dlam(t_hi, lx, sigma) - dH_dlam(t_lo, lx, sigma))
    z = np.zeros_like(np.asarray(sigma, dtype=np.float64))
    return (np.stack([z, dx.real, z, dx.imag]),
            np.stack([0.5 * (-G * dm + G * dp).real, z, 0.5 * (-G * dm - G * dp).real, z]))
