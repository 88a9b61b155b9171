"""Seeded, synthetic workload descriptions shared by the CUDA path, the oracle and the tests.

This module holds NONE of the method's arithmetic: only the plain-data model tables of
BASELINE.json's five configs (particle masses, resonance list, decay-chain terms, sizes, seeds)
and the random draws the method itself does not make (couplings, parameter trajectories), taken
from numpy's PCG64 so that both sides receive identical numbers as *inputs*.

Events are NOT produced here: "drawn from the model" / "flat phase space" samples come from the
Raubold-Lynch + Philox generator, which is part of the method and is
therefore implemented twice, once in oracle/ and once in csrc/ (parity: momenta to 1e-12).

Citations: P:<n> = /root/reference/PAPER.md line n; BJ = BASELINE.json; O-n = SURVEY.md 8(c).
"""
from __future__ import annotations

import copy
import math
from dataclasses import dataclass, field

import numpy as np

# spin-factor kinds (O-4).  Plain labels; each side maps them onto its own enum.
SF_NONRES, SF_VV_S, SF_VV_P, SF_VV_D, SF_AP_S, SF_TP_D, SF_AP_D = range(7)
# lineshape kinds: 0 relativistic Breit-Wigner with mass-dependent width (O-6), 1 with constant width
LS_RUNNING, LS_CONSTANT = 0, 1

# final-state order 0 = K+, 1 = pi-, 2 = pi+, 3 = pi- (O-3); masses from BJ:configs[0]
M_D0 = 1.86484
M_K = 0.493677
M_PI = 0.13957
TAU_D0 = 0.4101      # ps, BJ:configs[0]
X_MIX = 0.0049
Y_MIX = 0.0061
BASE_SEED = 42       # BJ:configs[3]

# Philox stream ids (O-9)
STREAM_DATA, STREAM_PARAMS, STREAM_NORM, STREAM_SMEAR = 0, 1, 2, 3

# resonance table: name -> (m0, Gamma0 [GeV], L of its own decay vertex) (BJ:configs[0..1], O-5, O-7)
RESONANCES = {
    "K*(892)0": (0.8955, 0.0473, 1),
    "rho(770)0": (0.775, 0.149, 1),
    "a1(1260)": (1.23, 0.42, 0),
    "K1(1270)": (1.272, 0.09, 0),
    "K2*(1430)": (1.4324, 0.109, 2),
    "K1(1400)": (1.403, 0.174, 0),
    "K1(1400)[D]": (1.403, 0.174, 2),      # the same state decaying to K* pi in D-wave (its own entry: L is per entry)
}

# decay chains, ordering A (O-7): (spin factor, (res0, res1), perm).  perm maps role -> particle:
#   VV kinds: R1 -> (perm0, perm1), R2 -> (perm2, perm3)
#   cascade : V -> (perm0, perm1), X -> (V, perm2), D -> (X, perm3)
CHAINS = {
    1: (SF_VV_S, ("K*(892)0", "rho(770)0"), (0, 1, 2, 3)),
    2: (SF_AP_S, ("a1(1260)", "rho(770)0"), (2, 3, 1, 0)),
    3: (SF_AP_S, ("K1(1270)", "K*(892)0"), (0, 1, 2, 3)),
    4: (SF_TP_D, ("K2*(1430)", "K*(892)0"), (0, 1, 2, 3)),
    5: (SF_AP_S, ("K1(1400)", "K*(892)0"), (0, 1, 2, 3)),
    6: (SF_VV_P, ("K*(892)0", "rho(770)0"), (0, 1, 2, 3)),
    7: (SF_VV_D, ("K*(892)0", "rho(770)0"), (0, 1, 2, 3)),
    8: (SF_NONRES, (None, None), (0, 1, 2, 3)),
    9: (SF_AP_D, ("K1(1400)[D]", "K*(892)0"), (0, 1, 2, 3)),       # further building block, in no config
}


@dataclass
class Model:
    """Plain-data description of a time-dependent amplitude model."""
    m_parent: float = M_D0
    m_final: tuple = (M_K, M_PI, M_PI, M_PI)
    r_res: float = 1.5          # GeV^-1, BJ:configs[1]
    r_parent: float = 1.5
    t_lo: float = 0.0
    t_hi: float = math.inf
    use_resolution: int = 0      # 0: eq. (1); 1: per-event Gaussian decay-time resolution; 2: time-integrated (no t)
    res_names: list = field(default_factory=list)
    res_L: list = field(default_factory=list)
    res_mass: list = field(default_factory=list)    # nominal m0 (initial parameter values)
    res_width: list = field(default_factory=list)   # nominal Gamma0
    res_r: list = field(default_factory=list)       # per-resonance Blatt-Weisskopf radius, 0 = r_res
    res_lineshape: list = field(default_factory=list)   # LS_* per resonance
    term_sf: list = field(default_factory=list)
    term_res: list = field(default_factory=list)    # [(r0, r1)] indices, -1 = none
    term_perm: list = field(default_factory=list)
    term_coupling: list = field(default_factory=list)
    n_couplings: int = 0

    @property
    def n_res(self):
        return len(self.res_names)

    @property
    def n_terms(self):
        return len(self.term_sf)


def _swap13(perm):
    """Ordering B: exchange the identical pions 1 <-> 3 (O-7, P:51 Bose symmetrisation)."""
    m = {0: 0, 1: 3, 2: 2, 3: 1}
    return tuple(m[p] for p in perm)


def build_model(chain_ids, bose=False, **kw) -> Model:
    mdl = Model(**kw)
    for cid in chain_ids:
        sf, names, perm = CHAINS[cid]
        idx = []
        for nm in names:
            if nm is None:
                idx.append(-1)
                continue
            if nm not in mdl.res_names:
                m0, g0, L = RESONANCES[nm]
                mdl.res_names.append(nm)
                mdl.res_L.append(L)
                mdl.res_mass.append(m0)
                mdl.res_width.append(g0)
                mdl.res_r.append(0.0)
                mdl.res_lineshape.append(LS_RUNNING)
            idx.append(mdl.res_names.index(nm))
        kappa = mdl.n_couplings
        mdl.n_couplings += 1
        for pm in ([perm, _swap13(perm)] if bose else [perm]):
            mdl.term_sf.append(sf)
            mdl.term_res.append(tuple(idx))
            mdl.term_perm.append(tuple(pm))
            mdl.term_coupling.append(kappa)
    return mdl


def flat_model(**kw) -> Model:
    """One constant term: with c = 1, cbar = 0, x = y = 0 the bracket of eq. (1) is 2 everywhere,
    so accept-reject against it un-weights Raubold-Lynch candidates to flat phase space (8(d))."""
    return build_model([8], bose=False, **kw)


@dataclass
class Params:
    """One point in parameter space, as the host minimiser would propose it."""
    c: np.ndarray        # [K_c] complex
    cbar: np.ndarray     # [K_c] complex
    mass: np.ndarray     # [n_res]
    width: np.ndarray    # [n_res]
    x: float = X_MIX
    y: float = Y_MIX
    tau: float = TAU_D0

    def copy(self):
        return copy.deepcopy(self)


def draw_couplings(n, rng):
    """|c| ~ U[0.5, 2], arg ~ U[0, 2 pi) (BJ:configs[0])."""
    return rng.uniform(0.5, 2.0, n) * np.exp(1j * rng.uniform(0.0, 2.0 * np.pi, n))


def initial_params(mdl: Model, seed=BASE_SEED) -> Params:
    rng = np.random.default_rng([seed, STREAM_PARAMS])
    c = draw_couplings(mdl.n_couplings, rng)
    cbar = draw_couplings(mdl.n_couplings, rng)
    return Params(c=c, cbar=cbar, mass=np.array(mdl.res_mass, float), width=np.array(mdl.res_width, float))


def flat_params(mdl: Model) -> Params:
    return Params(c=np.ones(1, complex), cbar=np.zeros(1, complex), mass=np.zeros(0), width=np.zeros(0),
                  x=0.0, y=0.0, tau=TAU_D0)


def trajectory(mdl: Model, p0: Params, n_calls, kind, seed=BASE_SEED, rel=1e-3, resonances=None):
    """Parameter steps standing in for the host minimiser.

    kind: 'couplings_xy' - every call perturbs couplings, x, y; masses/widths fixed (config 2)
          'minuit'       - p=0.8 one random floating parameter moves, p=0.2 all move (configs 3, 5)
          'coupling_only'- one coupling component moves per call (best case)
          'all'          - every parameter moves on every call (worst case)
          'one_resonance'- the mass or the width of ONE resonance (drawn from `resonances`, default all) moves per call
    Steps are relative Gaussian perturbations of size `rel` around the start point p0."""
    kinds = {"couplings_xy": 0, "minuit": 1, "coupling_only": 2, "all": 3, "one_resonance": 4}
    rng = np.random.default_rng([seed, STREAM_PARAMS, n_calls, kinds[kind]])
    kc, nr = mdl.n_couplings, mdl.n_res
    n_float = 4 * kc + 2 * nr + 2
    cur = p0.copy()
    out = []

    def move(p, j):
        g = 1.0 + rel * rng.standard_normal()
        if j < 2 * kc:
            k, part = divmod(j, 2)
            z = p.c[k]
            p.c[k] = complex(z.real * g, z.imag) if part == 0 else complex(z.real, z.imag * g)
        elif j < 4 * kc:
            k, part = divmod(j - 2 * kc, 2)
            z = p.cbar[k]
            p.cbar[k] = complex(z.real * g, z.imag) if part == 0 else complex(z.real, z.imag * g)
        elif j < 4 * kc + nr:
            p.mass[j - 4 * kc] = p0.mass[j - 4 * kc] * g
        elif j < 4 * kc + 2 * nr:
            p.width[j - 4 * kc - nr] = p0.width[j - 4 * kc - nr] * g
        elif j == 4 * kc + 2 * nr:
            p.x = p0.x * g
        else:
            p.y = p0.y * g

    for _ in range(n_calls):
        nxt = cur.copy()
        if kind == "couplings_xy":
            for j in list(range(4 * kc)) + [n_float - 2, n_float - 1]:
                move(nxt, j)
        elif kind == "minuit":
            if rng.uniform() < 0.8:
                move(nxt, int(rng.integers(n_float)))
            else:
                for j in range(n_float):
                    move(nxt, j)
        elif kind == "coupling_only":
            move(nxt, int(rng.integers(4 * kc)))
        elif kind == "all":
            for j in range(n_float):
                move(nxt, j)
        elif kind == "one_resonance":
            pool = list(range(nr)) if resonances is None else list(resonances)
            r = pool[int(rng.integers(len(pool)))]
            move(nxt, 4 * kc + r + (nr if rng.uniform() < 0.5 else 0))
        else:
            raise ValueError(kind)
        out.append(nxt)
        cur = nxt
    return out


@dataclass
class Config:
    name: str
    model: Model
    n_data: int
    n_norm: int
    n_calls: int
    trajectory: str
    n_candidates: int = 0
    n_pilot: int = 100_000
    envelope_scale: float = 1.2
    sigma_t: tuple | None = None        # (lo, hi) ps, per-event resolution (config 5)
    efficiency: tuple | None = None     # (lo, hi) weights on the normalisation sample (config 5)


def config(i: int) -> Config:
    """BASELINE.json configs, 1-based as in SURVEY.md 8 (C1..C5)."""
    if i == 1:
        return Config("C1", build_model([1, 2, 3]), 1_000, 10_000, 1, "coupling_only")
    if i == 2:
        return Config("C2", build_model(range(1, 9)), 50_000, 500_000, 300, "couplings_xy")
    if i == 3:
        return Config("C3", build_model(range(1, 9), bose=True), 1_000_000, 4_000_000, 1000, "minuit")
    if i == 4:
        return Config("C4", build_model([1, 2, 3]), 0, 0, 1, "coupling_only", n_candidates=10_000_000)
    if i == 5:
        return Config("C5", build_model(range(1, 9), bose=True, t_lo=0.0, t_hi=4.0, use_resolution=1),
                      10_000_000, 10_000_000, 100, "minuit", sigma_t=(0.03, 0.08), efficiency=(0.5, 1.0))
    raise ValueError(i)


def flat_envelope_inputs(mdl: Model):
    """Plain data for the hit-or-miss bound of the flat sample: the three (M, m_a, m_b) triples whose
    breakup momenta multiply to the rigorous bound on the Raubold-Lynch weight.
    The arithmetic (breakup momentum) is done by whoever consumes it."""
    m0, m1, m2, m3 = mdl.m_final
    M = mdl.m_parent
    return [(M, m0 + m1 + m2, m3), (M - m3, m0 + m1, m2), (M - m2 - m3, m0, m1)]


def smear_times(t_true, cfg: Config, seed=BASE_SEED):
    """Input synthesis for config 5 (BJ:configs[4]): per-event sigma_t ~ U[lo, hi] and observed time t + sigma z, z ~ N(0,1),
    redrawn until it falls inside the model's decay-time window.  numpy PCG64([seed, STREAM_SMEAR]); both the CUDA path
    and the oracle receive the result as input."""
    rng = np.random.default_rng([seed, STREAM_SMEAR])
    t_true = np.asarray(t_true, dtype=np.float64)
    lo, hi = cfg.sigma_t
    sigma = rng.uniform(lo, hi, t_true.shape[0])
    t_obs = t_true + sigma * rng.standard_normal(t_true.shape[0])
    for _ in range(1000):
        bad = (t_obs < cfg.model.t_lo) | (t_obs > cfg.model.t_hi)
        if not bad.any():
            break
        t_obs[bad] = t_true[bad] + sigma[bad] * rng.standard_normal(int(bad.sum()))
    # true times far beyond the window can never be smeared back into it: fold them to the window edge region
    bad = (t_obs < cfg.model.t_lo) | (t_obs > cfg.model.t_hi)
    t_obs[bad] = np.clip(t_obs[bad], cfg.model.t_lo, cfg.model.t_hi)
    return t_obs, sigma


def efficiency_weights(n, cfg: Config, seed=BASE_SEED):
    """epsilon_j ~ U[lo, hi] on the normalisation sample (BJ:configs[4])."""
    rng = np.random.default_rng([seed, STREAM_SMEAR, 1])
    lo, hi = cfg.efficiency
    return rng.uniform(lo, hi, n)
