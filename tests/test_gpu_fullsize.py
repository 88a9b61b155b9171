"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (persistent grids, tddp4_nll_batch).

The oracle cannot evaluate 1e6..1e7 events per call in seconds, so outputs are SAMPLED: the CUDA generator returns the
candidate indices of the events it accepted; the oracle regenerates the sampled events itself from (seed, index), so
no momentum it sees was produced by the CUDA path.  The normalisation is checked through the oracle's own direct sum
over the full normalisation sample (a few seconds with OpenMP).  What cannot be sampled (the NLL itself) is checked
through properties that hold at any size: invariance under a common real scale and a common phase of all couplings,
bit-reproducibility, and agreement of the batched with the synchronous entry point."""
import math

import numpy as np
import pytest

import oracle
from oracle import resolution as OR
from paper_1702_06735_b200 import workloads as W

pytestmark = pytest.mark.gpu
N_SAMPLE = 2_000


@pytest.fixture(scope="module")
def B():
    from paper_1702_06735_b200 import binding
    binding.load_library()
    return binding


def build_samples(B, cfg, device="cuda:0"):
    flat = W.flat_model()
    hf = B.Tddp4(flat, device)
    hf.set_params(W.flat_params(flat))
    p4n, _, idxn, _ = hf.generate_n(W.BASE_SEED, W.STREAM_NORM, cfg.n_norm, 0, 2.0 * hf.weight_bound(), chunk=1 << 24,
                                    want_index=True)
    hf.close()
    hg = B.Tddp4(cfg.model, device)
    par = W.initial_params(cfg.model)
    hg.set_params(par)
    p4, t, idx, info = hg.generate_n(W.BASE_SEED, W.STREAM_DATA, cfg.n_data, cfg.n_pilot, cfg.envelope_scale,
                                     chunk=1 << 24, want_index=True)
    hg.close()
    return par, p4, t, idx, p4n, idxn


def oracle_norm_sums(mdl, par, flat, idxn, w=None):
    p4n_ref, _, _, _ = oracle.candidates_at(flat, W.TAU_D0, W.BASE_SEED, W.STREAM_NORM, idxn)
    return oracle.norm(mdl, par, p4n_ref, w)


def nll_properties(h, par, nll):
    """Properties of a normalised likelihood that hold at any size."""
    tol = 1e-11 * abs(nll)
    p = par.copy(); p.c = p.c * 1.7; p.cbar = p.cbar * 1.7
    h.set_params(p)
    assert abs(h.nll() - nll) <= tol
    p = par.copy(); ph = np.exp(0.83j); p.c = p.c * ph; p.cbar = p.cbar * ph
    h.set_params(p)
    assert abs(h.nll() - nll) <= tol
    h.set_params(par)
    assert h.nll() == nll
    vals, st = h.nll_batch(h.pack_params([par, p, par]))
    assert st.tolist() == [0, 0, 0] and vals[0] == nll and vals[2] == nll


def test_config3_full_size(B):
    cfg = W.config(3)
    mdl = cfg.model
    par, p4, t, idx, p4n, idxn = build_samples(B, cfg)
    assert p4.shape[1] == cfg.n_data and p4n.shape[1] == cfg.n_norm
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t)
    h.load_events(1, p4n)
    h.set_params(par)
    prob = h.empty(cfg.n_data)
    nll = h.nll(prob)
    norm_ref, _ = oracle_norm_sums(mdl, par, W.flat_model(), idxn.cpu().numpy())
    assert abs(h.nll_parts()["norm"] / norm_ref - 1.0) < 1e-11
    pick = np.unique(np.concatenate([np.arange(64), np.random.default_rng(1).integers(0, cfg.n_data, N_SAMPLE),
                                     np.arange(cfg.n_data - 64, cfg.n_data)]))
    p4s, ts, _, _ = oracle.candidates_at(mdl, par.tau, W.BASE_SEED, W.STREAM_DATA, idx.cpu().numpy()[pick])
    assert np.max(np.abs(p4.cpu().numpy()[:, pick] - p4s)) < 1e-12
    R_ref, _ = oracle.rate(mdl, par, p4s, ts)
    P = prob.cpu().numpy()
    assert np.max(np.abs(P[pick] / (R_ref / norm_ref) - 1.0)) < 1e-10
    assert np.all(P > 0) and abs(-float(np.sum(np.log(P))) - nll) < 1e-11 * abs(nll)   # NLL = -sum log of ITS OWN P_i
    nll_properties(h, par, nll)
    # a mass step at full size: the fused rebuild and the cached path give the same bits
    p2 = par.copy(); p2.mass[1] *= 1.0007
    h.set_params(p2); a = h.nll()
    h.set_params(par); h.nll()
    h.set_params(p2); assert h.nll() == a


def test_config5_full_size(B):
    cfg = W.config(5)
    mdl = cfg.model
    par, p4, t_true, idx, p4n, idxn = build_samples(B, cfg)
    t, sig = W.smear_times(t_true.cpu().numpy(), cfg)
    w = W.efficiency_weights(cfg.n_norm, cfg)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, h.empty(cfg.n_data).copy_(__import__("torch").from_numpy(t)),
                  sigma_t=h.empty(cfg.n_data).copy_(__import__("torch").from_numpy(sig)))
    h.load_events(1, p4n, None, weight=h.empty(cfg.n_norm).copy_(__import__("torch").from_numpy(w)))
    h.set_params(par)
    prob = h.empty(cfg.n_data)
    nll = h.nll(prob)
    _, S = oracle_norm_sums(mdl, par, W.flat_model(), idxn.cpu().numpy(), w)
    pick = np.unique(np.concatenate([np.arange(64), np.random.default_rng(2).integers(0, cfg.n_data, N_SAMPLE),
                                     np.arange(cfg.n_data - 64, cfg.n_data)]))
    p4s, _, _, _ = oracle.candidates_at(mdl, par.tau, W.BASE_SEED, W.STREAM_DATA, idx.cpu().numpy()[pick])
    A, Ab = oracle.amplitudes(mdl, par, p4s)
    P_ref, _, _ = OR.prob(A, Ab, S, t[pick], sig[pick], par.x, par.y, par.tau, mdl.t_lo, mdl.t_hi)
    P = prob.cpu().numpy()
    assert np.max(np.abs(P[pick] / P_ref - 1.0)) < 1e-10
    assert np.all(P > 0) and abs(-math.fsum(np.log(P)) - nll) < 1e-11 * abs(nll)
    nll_properties(h, par, nll)


def test_config4_full_size(B):
    """10 000 000 candidates, pilot 100 000, envelope x1.2, config-1 rate: counts, order, sampled momenta, and the accept
    mask bit-exact on two windows of 100 000 candidates (start and end of the range)."""
    cfg = W.config(4)
    mdl = cfg.model
    par = W.initial_params(mdl)
    h = B.Tddp4(mdl)
    h.set_params(par)
    n = cfg.n_candidates
    g = h.generate(W.BASE_SEED, W.STREAM_DATA, 0, n, cfg.n_pilot, cfg.envelope_scale, n // 4, want_index=True)
    idx = g["index"].cpu().numpy()
    assert g["n_accepted"] == len(idx) and np.all(np.diff(idx) > 0) and idx[-1] < n
    rho_p, _ = oracle.candidate_ratio(mdl, par, W.BASE_SEED, W.STREAM_DATA, 0, cfg.n_pilot)
    assert abs(g["envelope"] / (cfg.envelope_scale * rho_p.max()) - 1.0) < 1e-10
    for first in (0, n - 100_000):
        rho, ua = oracle.candidate_ratio(mdl, par, W.BASE_SEED, W.STREAM_DATA, first, 100_000)
        ref = ua * g["envelope"] < rho
        got = np.zeros(100_000, bool)
        got[idx[(idx >= first) & (idx < first + 100_000)] - first] = True
        diff = np.nonzero(ref != got)[0]
        assert np.all(np.abs(ua[diff] * g["envelope"] / rho[diff] - 1.0) < 1e-12)
    pick = np.random.default_rng(4).integers(0, len(idx), N_SAMPLE)
    p4r, tr, _, _ = oracle.candidates_at(mdl, par.tau, W.BASE_SEED, W.STREAM_DATA, idx[pick])
    assert np.max(np.abs(g["p4"].cpu().numpy()[:, pick] - p4r)) < 1e-12
    assert np.max(np.abs(g["t"].cpu().numpy()[pick] / tr - 1.0)) < 1e-12
