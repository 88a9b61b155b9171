"""Brute-force pin (BJ:north_star): the whole likelihood on 10 data + 25 normalisation
events recomputed in mpmath at 30 digits by a different route than the oracle: closed-form spin factors
(dot products and a determinant instead of index loops), breakup momenta from the Kallen function of
squared masses instead of the factored form, lineshape written as a complex fraction, closed-form time
integrals on [0, inf).  A dropped term, wrong sign, index or transposed operand in the oracle fails here."""
import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_1702_06735_b200 import workloads as W

mp.mp.dps = 30


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def madd(a, b):
    return [x + y for x, y in zip(a, b)]


def msub(a, b):
    return [x - y for x, y in zip(a, b)]


def mL1(p, q):
    f = mdot(p, q) / mdot(p, p)
    return [qi - pi * f for pi, qi in zip(p, q)]


def meps(a, b, c, d):
    return mp.det(mp.matrix([[a[i], b[i], c[i], d[i]] for i in range(4)]))


def kallen_q(s, sa, sb):
    lam = s * s + sa * sa + sb * sb - 2 * (s * sa + s * sb + sa * sb)
    return mp.sqrt(lam / (4 * s)) if lam > 0 else mp.mpf(0)


def F(L, z):
    return {0: mp.mpf(1), 1: 1 / mp.sqrt(1 + z), 2: 1 / mp.sqrt(9 + 3 * z + z * z)}[L]


def bw(m0, g0, L, r, s, sa, sb, sa0, sb0):
    q, q0 = kallen_q(s, sa, sb), kallen_q(m0 * m0, sa0, sb0)
    gam = g0 * (q / q0) ** (2 * L + 1) * m0 / mp.sqrt(s) * (F(L, (q * r) ** 2) / F(L, (q0 * r) ** 2)) ** 2
    return 1 / mp.mpc(m0 * m0 - s, -m0 * gam)


LD = {0: 0, 1: 0, 2: 1, 3: 2, 4: 1, 5: 2, 6: 1}


def radius(mdl, R):
    r = (getattr(mdl, "res_r", None) or [0.0] * mdl.n_res)[R]
    return mp.mpf(r if r > 0 else mdl.r_res)


def lineshape(mdl, R, m0, g0, s, sa, sb, sa0, sb0):
    """Kind 0: running-width Breit-Wigner with the resonance's own radius; kind 1: constant width."""
    kind = (getattr(mdl, "res_lineshape", None) or [0] * mdl.n_res)[R]
    if kind == 1:
        return 1 / mp.mpc(m0[R] * m0[R] - s, -m0[R] * g0[R])
    return bw(m0[R], g0[R], mdl.res_L[R], radius(mdl, R), s, sa, sb, sa0, sb0)


def term(mdl, par, k, p):
    sf, perm = mdl.term_sf[k], mdl.term_perm[k]
    if sf == W.SF_NONRES:
        return mp.mpc(1)
    r = [p[perm[i]] for i in range(4)]
    mf2 = [mp.mpf(mdl.m_final[perm[i]]) ** 2 for i in range(4)]
    R0, R1 = mdl.term_res[k]
    m0 = [mp.mpf(float(v)) for v in par.mass]
    g0 = [mp.mpf(float(v)) for v in par.width]
    rp = mp.mpf(mdl.r_parent)
    r0, r1 = radius(mdl, R0), radius(mdl, R1)
    if sf in (W.SF_VV_S, W.SF_VV_P, W.SF_VV_D):
        p1, q1, p2, q2 = madd(r[0], r[1]), msub(r[0], r[1]), madd(r[2], r[3]), msub(r[2], r[3])
        pD, qD = madd(p1, p2), msub(p1, p2)
        v1, v2, d = mL1(p1, q1), mL1(p2, q2), mL1(pD, qD)
        s1, s2, sD = mdot(p1, p1), mdot(p2, p2), mdot(pD, pD)
        if sf == W.SF_VV_S:
            S = mdot(v1, v2)
        elif sf == W.SF_VV_P:
            S = meps(pD, qD, v1, v2)
        else:
            S = mdot(d, v1) * mdot(d, v2) - mdot(d, d) / 3 * (mdot(v1, v2) - mdot(pD, v1) * mdot(pD, v2) / sD)
        Fp = (F(LD[sf], (kallen_q(sD, s1, s2) * rp) ** 2) * F(mdl.res_L[R0], (kallen_q(s1, mf2[0], mf2[1]) * r0) ** 2)
              * F(mdl.res_L[R1], (kallen_q(s2, mf2[2], mf2[3]) * r1) ** 2))
        T = (lineshape(mdl, R0, m0, g0, s1, mf2[0], mf2[1], mf2[0], mf2[1])
             * lineshape(mdl, R1, m0, g0, s2, mf2[2], mf2[3], mf2[2], mf2[3]))
        return S * Fp * T
    pV, qV = madd(r[0], r[1]), msub(r[0], r[1])
    pX, qX = madd(pV, r[2]), msub(pV, r[2])
    pD, qD = madd(pX, r[3]), msub(pX, r[3])
    v, d, t = mL1(pV, qV), mL1(pD, qD), mL1(pX, qX)
    sV, sX, sD = mdot(pV, pV), mdot(pX, pX), mdot(pD, pD)
    if sf == W.SF_AP_S:
        S = -(mdot(d, v) - mdot(pX, d) * mdot(pX, v) / sX)
    elif sf == W.SF_AP_D:
        S = mdot(d, t) * mdot(t, v) - mdot(t, t) / 3 * (mdot(d, v) - mdot(pX, d) * mdot(pX, v) / sX)
    else:
        S = mdot(d, t) * meps(d, t, pX, v) + mdot(d, d) / 3 * mdot(pD, t) / sD * meps(pD, t, pX, v)
    Fp = (F(LD[sf], (kallen_q(sD, sX, mf2[3]) * rp) ** 2) * F(mdl.res_L[R0], (kallen_q(sX, sV, mf2[2]) * r0) ** 2)
          * F(mdl.res_L[R1], (kallen_q(sV, mf2[0], mf2[1]) * r1) ** 2))
    T = (lineshape(mdl, R0, m0, g0, sX, sV, mf2[2], m0[R1] ** 2, mf2[2])
         * lineshape(mdl, R1, m0, g0, sV, mf2[0], mf2[1], mf2[0], mf2[1]))
    return S * Fp * T


def amplitudes(mdl, par, p):
    A = Ab = mp.mpc(0)
    for k in range(mdl.n_terms):
        a = term(mdl, par, k, p)
        kap = mdl.term_coupling[k]
        A += mp.mpc(complex(par.c[kap])) * a
        Ab += mp.mpc(complex(par.cbar[kap])) * a
    return A, Ab


def brute_nll(mdl, par, p4, t, p4n, wn):
    x, y, tau = mp.mpf(par.x), mp.mpf(par.y), mp.mpf(par.tau)
    Gam = 1 / tau
    T1, T2, T3, T4 = tau / (1 - y * y), tau / (1 + x * x), tau * y / (1 - y * y), tau * x / (1 + x * x)

    def ev(arr, i):
        return [[mp.mpf(float(arr[4 * a + c, i])) for c in range(4)] for a in range(4)]

    N = mp.mpf(0)
    for j in range(p4n.shape[1]):
        A, Ab = amplitudes(mdl, par, ev(p4n, j))
        aa, bb, cr = abs(A) ** 2, abs(Ab) ** 2, A * mp.conj(Ab)
        N += mp.mpf(float(wn[j])) * (T1 * (aa + bb) + T2 * (aa - bb) - 2 * T3 * mp.re(cr) - 2 * T4 * mp.im(cr))
    N /= p4n.shape[1]
    nll, P = mp.mpf(0), []
    for i in range(p4.shape[1]):
        A, Ab = amplitudes(mdl, par, ev(p4, i))
        aa, bb, cr = abs(A) ** 2, abs(Ab) ** 2, A * mp.conj(Ab)
        ti = mp.mpf(float(t[i]))
        B = ((aa + bb) * mp.cosh(y * Gam * ti) + (aa - bb) * mp.cos(x * Gam * ti)
             - 2 * mp.re(cr) * mp.sinh(y * Gam * ti) - 2 * mp.im(cr) * mp.sin(x * Gam * ti))
        Pi = mp.exp(-Gam * ti) * B / N
        P.append(Pi)
        nll -= mp.log(Pi)
    return nll, N, P


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_ten_event_brute_force(cfg):
    mdl = W.config(cfg).model
    par = W.initial_params(mdl)
    par.x, par.y = 0.31, 0.12                     # large mixing so that every term of eq. (1) matters
    p4, t, w, _ = oracle.candidates(mdl, par.tau, 1234 + cfg, 0, 0, 35)
    data, td = p4[:, :10].copy(), t[:10] * 3.0
    nrm, wn = p4[:, 10:].copy(), w[10:] * 30.0
    nll_o, N_o, P_o, st = oracle.nll(mdl, par, data, td, nrm, wn)
    assert st == 0
    nll_b, N_b, P_b = brute_nll(mdl, par, data, td, nrm, wn)
    assert float(abs(N_o - N_b) / N_b) < 1e-12
    for po, pb in zip(P_o, P_b):
        assert float(abs(po - pb) / pb) < 1e-11
    assert float(abs(nll_o - nll_b)) < 1e-11 * max(1.0, float(abs(nll_b)))


def blocks_model():
    """Every further building block of SURVEY.md 8(f) NEXT-2 in one model: the axial D-wave cascade (chain 9), a
    constant-width lineshape, resonance radii different from the model's."""
    mdl = W.build_model([1, 3, 9, 2], bose=True)
    mdl.res_r[mdl.res_names.index("K*(892)0")] = 3.0
    mdl.res_r[mdl.res_names.index("K1(1400)[D]")] = 2.2
    mdl.res_lineshape[mdl.res_names.index("a1(1260)")] = W.LS_CONSTANT
    return mdl


def test_ten_event_brute_force_further_building_blocks():
    mdl = blocks_model()
    par = W.initial_params(mdl)
    par.x, par.y = 0.31, 0.12
    p4, t, w, _ = oracle.candidates(mdl, par.tau, 4321, 0, 0, 35)
    data, td = p4[:, :10].copy(), t[:10] * 3.0
    nrm, wn = p4[:, 10:].copy(), w[10:] * 30.0
    nll_o, N_o, P_o, st = oracle.nll(mdl, par, data, td, nrm, wn)
    assert st == 0
    nll_b, N_b, P_b = brute_nll(mdl, par, data, td, nrm, wn)
    assert float(abs(N_o - N_b) / N_b) < 1e-12
    for po, pb in zip(P_o, P_b):
        assert float(abs(po - pb) / pb) < 1e-11
    assert float(abs(nll_o - nll_b)) < 1e-11 * max(1.0, float(abs(nll_b)))
    S, Fb, a = oracle.terms(mdl, par, data)
    for i in range(5):
        p = [[mp.mpf(float(data[4 * b + c, i])) for c in range(4)] for b in range(4)]
        for k in range(mdl.n_terms):
            ref = complex(term(mdl, par, k, p))
            assert abs(a[k, i] - ref) <= 1e-11 * abs(ref)


def test_brute_force_per_term():
    """Every term amplitude of the 16-term model, 5 events, to 1e-11 of the term's modulus."""
    mdl = W.config(3).model
    par = W.initial_params(mdl)
    p4, *_ = oracle.candidates(mdl, par.tau, 555, 0, 0, 5)
    S, Fb, a = oracle.terms(mdl, par, p4)
    for i in range(5):
        p = [[mp.mpf(float(p4[4 * b + c, i])) for c in range(4)] for b in range(4)]
        for k in range(mdl.n_terms):
            ref = complex(term(mdl, par, k, p))
            assert abs(a[k, i] - ref) <= 1e-11 * abs(ref)
