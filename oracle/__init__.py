"""ctypes front end of the CPU oracle (oracle/tddp4_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, bench.py's cpu_baseline / `--impl reference` legs and __graft_entry__.smoke() may import
this package.  It never imports the CUDA binding, and the CUDA binding never imports it.

The arithmetic lives in the C file (fp64, written from the paper; see its header).  This file only
builds it with gcc, marshals numpy arrays, and adds the decay-time-resolution layer of O-8 (config 5),
which needs the complex error function: scipy.special.wofz / erfc serve as library primitives there.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tddp4_oracle.c")
_LIB = os.path.join(_HERE, "libtddp4_oracle.so")

MAX_RES, MAX_TERMS, MAX_COUPLINGS = 16, 64, 32


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (no FMA contraction: every product and sum rounds once) -fopenmp."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Model(C.Structure):
    _fields_ = [("m_parent", C.c_double), ("m_final", C.c_double * 4), ("r_res", C.c_double),
                ("r_parent", C.c_double), ("t_lo", C.c_double), ("t_hi", C.c_double),
                ("n_res", C.c_int), ("res_L", C.c_int * MAX_RES), ("n_terms", C.c_int),
                ("term_sf", C.c_int * MAX_TERMS), ("term_res", (C.c_int * 2) * MAX_TERMS),
                ("term_perm", (C.c_int * 4) * MAX_TERMS), ("term_coupling", C.c_int * MAX_TERMS),
                ("n_couplings", C.c_int), ("res_r", C.c_double * MAX_RES), ("res_kind", C.c_int * MAX_RES)]


class _Params(C.Structure):
    _fields_ = [("c", (C.c_double * 2) * MAX_COUPLINGS), ("cbar", (C.c_double * 2) * MAX_COUPLINGS),
                ("mass", C.c_double * MAX_RES), ("width", C.c_double * MAX_RES),
                ("x", C.c_double), ("y", C.c_double), ("tau", C.c_double)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        L.orc_sum.restype = C.c_double
        L.orc_breakup.restype = C.c_double
        L.orc_breakup.argtypes = [C.c_double] * 3
        L.orc_breakup_excess.restype = C.c_double
        L.orc_breakup_excess.argtypes = [C.c_double] * 4
        L.orc_barrier.restype = C.c_double
        L.orc_barrier.argtypes = [C.c_int, C.c_double]
        L.orc_dot.restype = C.c_double
        L.orc_eps4.restype = C.c_double
        L.orc_spin_factor.restype = C.c_double
        L.orc_bracket.restype = C.c_double
        L.orc_bracket.argtypes = [_dp, _dp, C.c_double, C.c_double, C.c_double, C.c_double]
        L.orc_breit_wigner.argtypes = [C.c_double, C.c_double, C.c_int, C.c_double, C.c_double, C.c_double,
                                       C.c_double, C.c_double, C.c_double, _dp]
        L.orc_time_integrals.argtypes = [C.c_double] * 5 + [_dp]
        L.orc_uniform_pair.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, _dp]
        L.orc_candidates.argtypes = [C.c_void_p, C.c_double, C.c_uint64, C.c_uint32, C.c_uint64, C.c_int64,
                                     C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_candidates.restype = None
        L.orc_candidate_ratio.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint64, C.c_int64,
                                          C.c_void_p, C.c_void_p]
        L.orc_generate.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_int64, C.c_int64,
                                   C.c_double, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                   C.POINTER(C.c_int64), C.POINTER(C.c_int64), _dp]
        L.orc_terms.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_amplitudes.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_norm.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, _dp, _dp]
        L.orc_rate.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_nll.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p,
                              C.c_void_p, _dp, _dp, C.c_void_p]
    return _lib


def threads() -> int:
    return int(lib().orc_threads())


# ---------------------------------------------------------------------------------------------
# marshalling of the plain-data model / parameter descriptions (workloads.Model / workloads.Params)
def c_model(mdl) -> _Model:
    m = _Model()
    m.m_parent = mdl.m_parent
    for i in range(4):
        m.m_final[i] = mdl.m_final[i]
    m.r_res, m.r_parent, m.t_lo, m.t_hi = mdl.r_res, mdl.r_parent, mdl.t_lo, mdl.t_hi
    m.n_res = mdl.n_res
    for i, L in enumerate(mdl.res_L):
        m.res_L[i] = L
    for i, r in enumerate(getattr(mdl, "res_r", []) or []):
        m.res_r[i] = r
    for i, k in enumerate(getattr(mdl, "res_lineshape", []) or []):
        m.res_kind[i] = k
    m.n_terms = mdl.n_terms
    for k in range(mdl.n_terms):
        m.term_sf[k] = mdl.term_sf[k]
        m.term_res[k][0], m.term_res[k][1] = mdl.term_res[k]
        for r in range(4):
            m.term_perm[k][r] = mdl.term_perm[k][r]
        m.term_coupling[k] = mdl.term_coupling[k]
    m.n_couplings = mdl.n_couplings
    return m


def c_params(par) -> _Params:
    p = _Params()
    for k, z in enumerate(par.c):
        p.c[k][0], p.c[k][1] = z.real, z.imag
    for k, z in enumerate(par.cbar):
        p.cbar[k][0], p.cbar[k][1] = z.real, z.imag
    for r, v in enumerate(par.mass):
        p.mass[r] = v
    for r, v in enumerate(par.width):
        p.width[r] = v
    p.x, p.y, p.tau = par.x, par.y, par.tau
    return p


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.c_void_p)


def _ref(s):
    return C.cast(C.byref(s), C.c_void_p)


# ---------------------------------------------------------------------------------------------
# scalar building blocks (used by the pins)
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def uniform_pair(seed, index, block, stream):
    u = (C.c_double * 2)()
    lib().orc_uniform_pair(seed, index, block, stream, u)
    return u[0], u[1]


def breakup(M, ma, mb):
    return lib().orc_breakup(M, ma, mb)


def barrier(L, z):
    return lib().orc_barrier(L, z)


def breit_wigner(m0, gamma0, L, r, s, ma, mb, ma0=None, mb0=None):
    out = (C.c_double * 2)()
    st = lib().orc_breit_wigner(m0, gamma0, L, r, s, ma, mb, ma if ma0 is None else ma0,
                                mb if mb0 is None else mb0, out)
    if st:
        raise ValueError("pole below threshold")
    return complex(out[0], out[1])


def breit_wigner_constant(m0, gamma0, s):
    out = (C.c_double * 2)()
    lib().orc_breit_wigner_constant(C.c_double(m0), C.c_double(gamma0), C.c_double(s), out)
    return complex(out[0], out[1])


def spin_factor(sf, perm, p):
    """p: [4 particles][4 components] of ONE event."""
    a, _ = _f64(p)
    pm = (C.c_int * 4)(*perm)
    return lib().orc_spin_factor(sf, pm, a.ctypes.data_as(_dp))


def bracket(A, Abar, x, y, Gamma, t):
    a = (C.c_double * 2)(A.real, A.imag)
    b = (C.c_double * 2)(Abar.real, Abar.imag)
    return lib().orc_bracket(a, b, x, y, Gamma, t)


def time_integrals(x, y, tau, t_lo=0.0, t_hi=math.inf):
    T = (C.c_double * 4)()
    lib().orc_time_integrals(x, y, tau, t_lo, t_hi, T)
    return np.array(T[:])


# ---------------------------------------------------------------------------------------------
# batch entry points
def candidates(mdl, tau, seed, stream, first, n):
    """Raubold-Lynch candidates first..first+n-1 -> p4[16][n], t[n], w[n], u_acc[n] (O-9)."""
    m = c_model(mdl)
    p4 = np.empty((16, n)); t = np.empty(n); w = np.empty(n); ua = np.empty(n)
    lib().orc_candidates(_ref(m), tau, seed, stream, first, n, p4.ctypes.data, t.ctypes.data,
                         w.ctypes.data, ua.ctypes.data)
    return p4, t, w, ua


def candidates_at(mdl, tau, seed, stream, index):
    """Candidates with the given indices (int64 array) -> p4[16][n], t, w, u_acc."""
    m = c_model(mdl)
    index = np.ascontiguousarray(index, dtype=np.int64)
    n = len(index)
    p4 = np.empty((16, n)); t = np.empty(n); w = np.empty(n); ua = np.empty(n)
    lib().orc_candidates_at(_ref(m), C.c_double(tau), C.c_uint64(seed), C.c_uint32(stream), C.c_int64(n),
                            index.ctypes.data_as(C.c_void_p), p4.ctypes.data_as(C.c_void_p),
                            t.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p), ua.ctypes.data_as(C.c_void_p))
    return p4, t, w, ua


def candidate_ratio(mdl, par, seed, stream, first, n):
    m, p = c_model(mdl), c_params(par)
    rho = np.empty(n); ua = np.empty(n)
    st = lib().orc_candidate_ratio(_ref(m), _ref(p), seed, stream, first, n, rho.ctypes.data, ua.ctypes.data)
    if st:
        raise ValueError("pole below threshold")
    return rho, ua


def generate(mdl, par, seed, stream, n_candidates, n_pilot, envelope_scale, capacity):
    """Accept-reject generation (O-9, G1-G6).  Returns dict(p4[16][n_acc], t, index, n_accepted,
    n_overflow, envelope)."""
    m, p = c_model(mdl), c_params(par)
    p4 = np.empty((16, capacity)); t = np.empty(capacity); idx = np.empty(capacity, dtype=np.int64)
    na, no, env = C.c_int64(), C.c_int64(), C.c_double()
    st = lib().orc_generate(_ref(m), _ref(p), seed, stream, n_candidates, n_pilot, envelope_scale, capacity,
                            p4.ctypes.data, t.ctypes.data, idx.ctypes.data, C.byref(na), C.byref(no), C.byref(env))
    if st == 1:
        raise ValueError("pole below threshold")
    k = min(na.value, capacity)
    return dict(p4=np.ascontiguousarray(p4[:, :k]), t=t[:k].copy(), index=idx[:k].copy(), n_accepted=na.value,
                n_overflow=no.value, envelope=env.value, status=st)


def terms(mdl, par, p4):
    """Per-term spin factor S[k][n], barrier product F[k][n] and amplitude a[k][n] (complex)."""
    m, p = c_model(mdl), c_params(par)
    p4, pp = _f64(p4)
    n = p4.shape[1]
    S = np.empty((mdl.n_terms, n)); F = np.empty((mdl.n_terms, n)); a = np.empty((mdl.n_terms, n, 2))
    st = lib().orc_terms(_ref(m), _ref(p), n, pp, S.ctypes.data, F.ctypes.data, a.ctypes.data)
    if st:
        raise ValueError("pole below threshold")
    return S, F, a[..., 0] + 1j * a[..., 1]


def amplitudes(mdl, par, p4):
    m, p = c_model(mdl), c_params(par)
    p4, pp = _f64(p4)
    n = p4.shape[1]
    A = np.empty((n, 2)); Ab = np.empty((n, 2))
    st = lib().orc_amplitudes(_ref(m), _ref(p), n, pp, A.ctypes.data, Ab.ctypes.data)
    if st:
        raise ValueError("pole below threshold")
    return A[:, 0] + 1j * A[:, 1], Ab[:, 0] + 1j * Ab[:, 1]


def norm(mdl, par, p4_norm, w=None):
    """N = (1/N_n) sum_j w_j int R dt and (S_1..S_4) (O-8)."""
    m, p = c_model(mdl), c_params(par)
    p4, pp = _f64(p4_norm)
    wp = None
    if w is not None:
        w, wp = _f64(w)
    out = C.c_double(); S = (C.c_double * 4)()
    st = lib().orc_norm(_ref(m), _ref(p), p4.shape[1], pp, wp, C.byref(out), S)
    if st:
        raise ValueError("pole below threshold")
    return out.value, np.array(S[:])


def rate(mdl, par, p4, t):
    """R_i = e^{-Gamma t_i} B_i and B_i (eq. 1)."""
    m, p = c_model(mdl), c_params(par)
    p4, pp = _f64(p4); t, tp = _f64(t)
    n = p4.shape[1]
    R = np.empty(n); B = np.empty(n)
    st = lib().orc_rate(_ref(m), _ref(p), n, pp, tp, R.ctypes.data, B.ctypes.data)
    if st:
        raise ValueError("pole below threshold")
    return R, B


def nll(mdl, par, p4, t, p4_norm, w_norm=None, want_prob=True):
    """NLL = -sum_i log(R_i / N) (step 7); returns (nll, N, P[n] or None, status)."""
    m, p = c_model(mdl), c_params(par)
    p4, pp = _f64(p4); t, tp = _f64(t); p4n, pnp = _f64(p4_norm)
    wp = None
    if w_norm is not None:
        w_norm, wp = _f64(w_norm)
    n = p4.shape[1]
    prob = np.empty(n) if want_prob else None
    out, nrm = C.c_double(), C.c_double()
    st = lib().orc_nll(_ref(m), _ref(p), n, pp, tp, p4n.shape[1], pnp, wp, C.byref(out), C.byref(nrm),
                       prob.ctypes.data if want_prob else None)
    return out.value, nrm.value, prob, st
