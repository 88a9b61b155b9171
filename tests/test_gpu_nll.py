"""GPU parity: the NLL path (steps 0-7 of SURVEY.md 8(a)) through the C-ABI against the CPU oracle.

Tolerances are BASELINE.json's north_star: relative 1e-10 per event probability, 1e-11 on the NLL
(relative to max(|NLL|, 1e-3 sum |log P_i|)).  Inputs come from the oracle's own generator
(tests/samples.py); nothing the oracle sees was produced by the CUDA path."""
import math

import numpy as np
import pytest

import oracle
from paper_1702_06735_b200 import workloads as W

import samples

pytestmark = pytest.mark.gpu

TOL_P = 1e-10
TOL_NLL = 1e-11
TOL_LAYER = 1e-11


@pytest.fixture(scope="module")
def B():
    from paper_1702_06735_b200 import binding
    binding.load_library()
    return binding


def nll_close(got, ref, logs):
    scale = max(abs(ref), 1e-3 * float(np.sum(np.abs(logs))))
    return abs(got - ref) <= TOL_NLL * scale


def run_case(B, mdl, par, p4, t, p4n, w=None, from_host=True):
    import torch
    h = B.Tddp4(mdl)
    if from_host:
        h.load_events(0, p4, t)
        h.load_events(1, p4n, None, weight=w)
    else:
        dev = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()
        h.load_events(0, dev(p4), dev(t))
        h.load_events(1, dev(p4n), None, weight=dev(w))
    h.set_params(par)
    prob = h.empty(max(1, p4.shape[1]))
    nll = h.nll(prob)
    return h, nll, prob[:p4.shape[1]].cpu().numpy()


def check_against_oracle(B, mdl, par, p4, t, p4n, w=None, from_host=True):
    ref_nll, ref_norm, ref_P, st = oracle.nll(mdl, par, p4, t, p4n, w)
    assert st == 0
    h, nll, P = run_case(B, mdl, par, p4, t, p4n, w, from_host)
    assert samples.rel_err(P, ref_P) < TOL_P
    assert abs(h.nll_parts()["norm"] / ref_norm - 1.0) < 1e-12
    assert nll_close(nll, ref_nll, np.log(ref_P))
    assert h.nll() == nll                      # without prob_out: same value bit for bit
    return h


def test_config1_full(B):
    """BASELINE config 1 at full size: 1 000 model-drawn events, 10 000 flat events, K = 3."""
    cfg = W.config(1)
    p4, t, _ = samples.data_sample(("C", 1), cfg.n_data)
    p4n, _ = samples.flat_sample(cfg.n_norm)
    check_against_oracle(B, cfg.model, W.initial_params(cfg.model), p4, t, p4n)


@pytest.mark.parametrize("from_host", [True, False])
def test_config2_model_ragged(B, from_host):
    """8 chains (all six spin-factor kinds); sizes that span several tiles and leave a ragged tail."""
    mdl = samples.model_of(("C", 2))
    p4, t, _ = samples.data_sample(("C", 2), 4_133)
    p4n, _ = samples.flat_sample(20_011)
    check_against_oracle(B, mdl, W.initial_params(mdl), p4, t, p4n, from_host=from_host)


def test_config3_model_bose_weights(B):
    """16 Bose-symmetrised terms on 8 couplings, efficiency weights on the normalisation sample."""
    mdl = samples.model_of(("C", 3))
    p4, t, _ = samples.data_sample(("C", 3), 3_001)
    p4n, _ = samples.flat_sample(10_007)
    w = np.random.default_rng(7).uniform(0.5, 1.0, p4n.shape[1])
    check_against_oracle(B, mdl, W.initial_params(mdl), p4, t, p4n, w)


def test_layers(B):
    """Per-layer parity: s-values, static factors S_k F, per-term amplitudes, columns."""
    import torch
    mdl = samples.model_of(("C", 3))
    par = W.initial_params(mdl)
    p4, _, _, _ = oracle.candidates(mdl, par.tau, 42, 5, 0, 2_077)     # raw candidates: whole phase space
    t = np.full(p4.shape[1], 0.3)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t)
    h.set_params(par)
    S, F, a = oracle.terms(mdl, par, p4)
    lay = h.layout()
    s_gpu = h.get(0, B.GET_S).cpu().numpy()
    P = p4.reshape(4, 4, -1)
    for row, mask in enumerate(lay["sys_mask"]):
        q = sum(P[i] for i in range(4) if mask >> i & 1)
        s_ref = q[0] ** 2 - q[1] ** 2 - q[2] ** 2 - q[3] ** 2
        assert samples.rel_err(s_gpu[row], s_ref) < 1e-13
    f_gpu = h.get(0, B.GET_STATIC).cpu().numpy()
    scale = np.abs(S * F).max(axis=1, keepdims=True)
    assert np.max(np.abs(f_gpu - S * F) / scale) < TOL_LAYER
    a_gpu = h.get(0, B.GET_TERMS).cpu().numpy()
    scale = np.abs(a).max(axis=1, keepdims=True)
    assert np.max(np.abs(a_gpu - a) / scale) < TOL_LAYER
    col = h.get(0, B.GET_COLUMNS).cpu().numpy()
    ref_col = np.zeros_like(col)
    for k, kap in enumerate(mdl.term_coupling):
        ref_col[kap] += a[k]
    scale = np.abs(ref_col).max(axis=1, keepdims=True)
    assert np.max(np.abs(col - ref_col) / scale) < TOL_LAYER


def test_further_building_blocks(B):
    """SURVEY.md 8(f) NEXT-2 / PAPER.md line 51: the axial D-wave cascade, per-resonance radii and a constant-width
    lineshape in one Bose-symmetrised model: static factors, per-term amplitudes, P_i, N, the NLL, the gradient, and a
    mass/width step on the constant-width and on the re-sized resonance (dirty tracking through the new code paths)."""
    from test_oracle_bruteforce import blocks_model
    from oracle import gradient as OG
    mdl = blocks_model()
    par = W.initial_params(mdl)
    p4, _, _, _ = oracle.candidates(mdl, par.tau, 42, 5, 0, 1_555)      # raw candidates: whole phase space
    t = np.random.default_rng(3).exponential(par.tau, p4.shape[1])
    p4n, _ = samples.flat_sample(4_001)
    h = check_against_oracle(B, mdl, par, p4, t, p4n)
    S, F, a = oracle.terms(mdl, par, p4)
    f_gpu = h.get(0, B.GET_STATIC).cpu().numpy()
    assert np.max(np.abs(f_gpu - S * F) / np.abs(S * F).max(axis=1, keepdims=True)) < TOL_LAYER
    a_gpu = h.get(0, B.GET_TERMS).cpu().numpy()
    assert np.max(np.abs(a_gpu - a) / np.abs(a).max(axis=1, keepdims=True)) < TOL_LAYER
    ref, _ = OG.nll_gradient(mdl, par, p4, t, p4n)
    _, g = h.nll_grad()
    assert np.max(np.abs(g - ref)) <= 1e-10 * np.abs(ref).max()
    for name in ("a1(1260)", "K*(892)0", "K1(1400)[D]"):
        step = par.copy()
        r = mdl.res_names.index(name)
        step.mass[r] *= 1.003; step.width[r] *= 0.98
        h.set_params(step)
        ref = oracle.nll(mdl, step, p4, t, p4n)
        assert nll_close(h.nll(), ref[0], np.log(ref[2]))
    # generation with the same blocks: candidate ratios against the oracle
    h.set_params(par)
    _, _, _, rho, _ = h.candidates(77, 0, 0, 3_000)
    rho_ref, _ = oracle.candidate_ratio(mdl, par, 77, 0, 0, 3_000)
    assert samples.rel_err(rho.cpu().numpy(), rho_ref, floor=np.abs(rho_ref).max() * 1e-12) < 1e-10


def test_trajectory_dirty_tracking(B):
    """Parameter steps as the minimiser would make them: every call is checked against a from-scratch oracle
    evaluation, so stale caches (lineshapes not refreshed, Gram matrix not rebuilt) cannot hide."""
    mdl = samples.model_of(("C", 3))
    p0 = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 3), 1_500)
    p4n, _ = samples.flat_sample(6_000)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t)
    h.load_events(1, p4n)
    steps = W.trajectory(mdl, p0, 12, "minuit", rel=1e-2) + W.trajectory(mdl, p0, 4, "coupling_only") + \
        W.trajectory(mdl, p0, 3, "all", rel=1e-2)
    prob = h.empty(p4.shape[1])
    for par in [p0] + steps:
        h.set_params(par)
        nll = h.nll(prob)
        ref_nll, ref_norm, ref_P, st = oracle.nll(mdl, par, p4, t, p4n)
        assert st == 0
        assert samples.rel_err(prob.cpu().numpy(), ref_P) < TOL_P
        assert nll_close(nll, ref_nll, np.log(ref_P))


def test_bit_reproducible_and_async_slots(B):
    mdl = samples.model_of(("C", 2))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 2), 4_133)
    p4n, _ = samples.flat_sample(20_011)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t)
    h.load_events(1, p4n)
    h.set_params(par)
    first = h.nll()
    assert all(h.nll() == first for _ in range(5))
    steps = W.trajectory(mdl, par, 8, "couplings_xy")
    sync = []
    for p in steps:
        h.set_params(p)
        sync.append(h.nll())
    for s, p in enumerate(steps):              # pipelined: enqueue all, then collect
        h.set_params(p)
        h.nll_async(s)
    assert [h.nll_result(s) for s in range(len(steps))] == sync
    h2 = B.Tddp4(mdl)                          # a second handle gives the same bits
    h2.load_events(0, p4, t)
    h2.load_events(1, p4n)
    h2.set_params(par)
    assert h2.nll() == first


@pytest.mark.parametrize("n", [1, 31, 32, 33, 255, 257, 1025])
def test_ragged_sizes(B, n):
    mdl = samples.model_of(("C", 1))
    p4, t, _ = samples.data_sample(("C", 1), 1_025)
    p4n, _ = samples.flat_sample(777)
    check_against_oracle(B, mdl, W.initial_params(mdl), p4[:, :n].copy(), t[:n].copy(), p4n[:, :max(1, n // 2)].copy())


def test_strided_device_input(B):
    """load_events with ld > n: rows of a larger device buffer are read in place."""
    import torch
    mdl = samples.model_of(("C", 1))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 1), 600)
    p4n, _ = samples.flat_sample(777)
    big = torch.zeros(16, 1000, dtype=torch.float64, device="cuda")
    big[:, :600] = torch.from_numpy(p4).cuda()
    h = B.Tddp4(mdl)
    h.load_events(0, big[:, :600], torch.from_numpy(t).cuda())
    h.load_events(1, p4n)
    h.set_params(par)
    ref = oracle.nll(mdl, par, p4, t, p4n)
    assert nll_close(h.nll(), ref[0], np.log(ref[2]))


def test_empty_data_sample(B):
    mdl = samples.model_of(("C", 1))
    p4n, _ = samples.flat_sample(777)
    h = B.Tddp4(mdl)
    h.load_events(0, np.zeros((16, 0)), np.zeros(0))
    h.load_events(1, p4n)
    h.set_params(W.initial_params(mdl))
    assert h.nll() == 0.0                       # empty sum


def test_special_cases_of_eq1(B):
    """x = y = 0 -> P independent of cbar; common global phase and common real scale leave the NLL unchanged."""
    mdl = samples.model_of(("C", 2))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 2), 2_000)
    p4n, _ = samples.flat_sample(5_000)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t)
    h.load_events(1, p4n)
    h.set_params(par)
    base = h.nll()
    q = par.copy(); q.c = par.c * np.exp(0.7j); q.cbar = par.cbar * np.exp(0.7j)
    h.set_params(q)
    assert abs(h.nll() - base) < 1e-9 * abs(base)
    q = par.copy(); q.c = par.c * 3.0; q.cbar = par.cbar * 3.0
    h.set_params(q)
    assert abs(h.nll() - base) < 1e-9 * abs(base)
    q = par.copy(); q.x = 0.0; q.y = 0.0
    h.set_params(q)
    a = h.nll()
    q.cbar = par.cbar[::-1].copy() * 0.3
    h.set_params(q)
    assert abs(h.nll() - a) < 1e-10 * abs(a)


def test_errors(B):
    mdl = samples.model_of(("C", 1))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 1), 100)
    p4n, _ = samples.flat_sample(777)
    h = B.Tddp4(mdl)
    with pytest.raises(B.Tddp4Error) as e:
        h.nll()
    assert e.value.code == B.ERR_STATE
    h.load_events(0, p4, t)
    h.set_params(par)
    with pytest.raises(B.Tddp4Error) as e:      # normalisation sample missing
        h.nll()
    assert e.value.code == B.ERR_STATE
    h.load_events(1, p4n)
    bad = par.copy(); bad.mass = par.mass.copy(); bad.mass[0] = 0.3     # K* pole below the K pi threshold
    with pytest.raises(B.Tddp4Error) as e:
        h.set_params(bad)
    assert e.value.code == B.ERR_DOMAIN
    zero = par.copy(); zero.c = par.c * 0; zero.cbar = par.cbar * 0    # rate vanishes: P_i = 0/0
    h.set_params(zero)
    with pytest.raises(B.Tddp4Error) as e:
        h.nll()
    assert e.value.code == B.ERR_NONFINITE
    assert h.nll(strict=False) == math.inf
    h.set_params(par)                           # the handle recovers
    ref = oracle.nll(mdl, par, p4, t, p4n)
    assert nll_close(h.nll(), ref[0], np.log(ref[2]))


def test_gram_matches_direct_normalisation(B):
    """Step 6 both ways: N from the Gram matrix (GPU) equals the direct sum over the sample (oracle), and the
    Gram matrix itself equals sum_j w_j a_k conj(a_l) built from the oracle's per-term amplitudes."""
    mdl = samples.model_of(("C", 3))
    par = W.initial_params(mdl)
    p4n, _ = samples.flat_sample(10_007)
    w = np.random.default_rng(3).uniform(0.5, 1.0, p4n.shape[1])
    h = B.Tddp4(mdl)
    h.load_events(1, p4n, None, weight=w)
    h.set_params(par)
    G, n = h.gram()
    assert n == p4n.shape[1]
    _, _, a = oracle.terms(mdl, par, p4n)
    col = np.zeros((mdl.n_couplings, p4n.shape[1]), complex)
    for k, kap in enumerate(mdl.term_coupling):
        col[kap] += a[k]
    G_ref = (col * w) @ col.conj().T
    assert np.max(np.abs(G - G_ref)) < 1e-12 * np.abs(G_ref).max()
    ref_norm, _ = oracle.norm(mdl, par, p4n, w)
    assert abs(h.norm() / ref_norm - 1.0) < 1e-12


def test_sharded_evaluation_adds_up(B):
    """SURVEY.md 8(e) on one GPU: two handles hold halves of both samples; summing their Gram matrices and
    their (sum log B, sum t) parts in rank order reproduces the single-handle NLL."""
    mdl = samples.model_of(("C", 2))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 2), 4_133)
    p4n, _ = samples.flat_sample(20_011)
    one = B.Tddp4(mdl)
    one.load_events(0, p4, t); one.load_events(1, p4n); one.set_params(par)
    full = one.nll()
    cut, cutn = 2_000, 9_000
    hs = [B.Tddp4(mdl), B.Tddp4(mdl)]
    hs[0].load_events(0, p4[:, :cut].copy(), t[:cut].copy()); hs[0].load_events(1, p4n[:, :cutn].copy())
    hs[1].load_events(0, p4[:, cut:].copy(), t[cut:].copy()); hs[1].load_events(1, p4n[:, cutn:].copy())
    Gs = []
    for h in hs:
        h.set_params(par)
        Gs.append(h.gram())
    G = Gs[0][0] + Gs[1][0]
    n = Gs[0][1] + Gs[1][1]
    sum_log_b = sum_t = 0.0
    for h in hs:
        h.gram_override(G, n)
        h.nll(strict=True)
        parts = h.nll_parts()
        sum_log_b += parts["sum_log_B"]; sum_t += parts["sum_t"]
        norm = parts["norm"]
    nll = sum_t / par.tau - sum_log_b + p4.shape[1] * math.log(norm)
    assert abs(nll - full) < 1e-12 * abs(full)


def test_dbar_tagged_sample(B):
    """SURVEY.md 8(f) NEXT-2, D0bar-tagged sample: a handle holding the D0bar-tagged events is fed the two coupling vectors
    exchanged (binding: set_params(par, dbar=True)); the oracle writes the D0bar rate and its normalisation out
    explicitly (oracle/tagged.py).  Both tags share one normalisation sample and one parameter point."""
    from oracle import tagged as OT
    mdl = samples.model_of(("C", 2))
    par = W.initial_params(mdl)
    par.x, par.y = 0.21, 0.13                       # large mixing: the cos and sin terms, which change sign, matter
    p4, t, _ = samples.data_sample(("C", 2), 4_133)
    p4n, _ = samples.flat_sample(20_011)
    tag = np.where(np.random.default_rng(9).uniform(size=p4.shape[1]) < 0.5, 1, -1)
    ref_nll, ref_P = OT.nll_tagged(mdl, par, p4, t, tag, p4n)
    total, P = 0.0, np.empty(p4.shape[1])
    for sign in (1, -1):
        sel = np.nonzero(tag == sign)[0]
        h = B.Tddp4(mdl)
        h.load_events(0, np.ascontiguousarray(p4[:, sel]), t[sel].copy())
        h.load_events(1, p4n)
        h.set_params(par, dbar=sign < 0)
        prob = h.empty(len(sel))
        total += h.nll(prob)
        P[sel] = prob.cpu().numpy()
    assert samples.rel_err(P, ref_P) < TOL_P
    assert nll_close(total, ref_nll, np.log(ref_P))


def test_large_mixing_phases_use_the_full_range_functions(B):
    """x, y far from the small-phase regime: the kernels switch from Taylor polynomials to exp / sincos."""
    mdl = samples.model_of(("C", 2))
    par = W.initial_params(mdl)
    par.x, par.y = 0.83, -0.41
    p4, t, _ = samples.data_sample(("C", 2), 2_000)
    p4n, _ = samples.flat_sample(5_000)
    h = check_against_oracle(B, mdl, par, p4, t, p4n)
    step = par.copy(); step.mass = par.mass * 1.001          # same regime through the fused columns+NLL kernel
    h.set_params(step)
    ref = oracle.nll(mdl, step, p4, t, p4n)
    assert nll_close(h.nll(), ref[0], np.log(ref[2]))
    # just below / above the switch-over (|phase| = 1/4 at the largest decay time) both agree with the oracle
    for scale in (0.999, 1.001):
        q = par.copy(); q.y = 0.0061; q.x = scale * 0.25 * par.tau / t.max()
        h.set_params(q)
        ref = oracle.nll(mdl, q, p4, t, p4n)
        assert nll_close(h.nll(), ref[0], np.log(ref[2]))


@pytest.mark.parametrize("chains", [(1, 2, 3, 4, 5, 6, 7, 8, 1, 3), (1, 2, 3, 4, 5, 6, 7, 8, 2, 3, 4, 5, 6)])
def test_more_than_eight_couplings(B, chains):
    """K_c = 10 and 13: the Gram kernel's 3- and 4-block tensor-core tilings and the wide NLL kernels."""
    mdl = samples.model_of(("chains", chains, False))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 2), 1_111)
    p4n, _ = samples.flat_sample(3_333)
    h = check_against_oracle(B, mdl, par, p4, t, p4n)
    step = par.copy(); step.width = par.width * 1.01
    h.set_params(step)
    ref = oracle.nll(mdl, step, p4, t, p4n)
    assert nll_close(h.nll(), ref[0], np.log(ref[2]))


def test_sharded_wrapper_on_one_rank(B):
    """sharded.ShardedNLL around the CUDA handle, world size 1: same value as the handle's own NLL to rounding of the
    recombination (Gamma sum t - sum log B + n log N is formed on the host here, on the device there)."""
    from paper_1702_06735_b200 import sharded
    mdl = samples.model_of(("C", 2))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 2), 2_049)
    p4n, _ = samples.flat_sample(10_001)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t); h.load_events(1, p4n)
    h.set_params(par)
    direct = h.nll()
    sh = sharded.ShardedNLL(h)
    sh.set_params(par)
    assert abs(sh.nll() - direct) <= 1e-13 * abs(direct)
    p2 = par.copy(); p2.mass[1] *= 1.0005
    h.set_params(p2); direct2 = h.nll()
    sh.set_params(p2)
    assert abs(sh.nll() - direct2) <= 1e-13 * abs(direct2)


def test_in_kernel_timing_of_the_coupling_only_kernel(B):
    """tddp4_profile_in_kernel: counted once per coupling-only launch while profiling, positive, below the CUDA-event
    duration of the same launches, and off (no count) when profiling is off; the NLL bits do not depend on it."""
    mdl = samples.model_of(("C", 2))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 2), 4_133)
    p4n, _ = samples.flat_sample(10_001)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t); h.load_events(1, p4n)
    h.set_params(par)
    ref = h.nll()
    plain = [h.nll() for _ in range(3)]
    assert h.profile_in_kernel() == (0.0, 0)
    h.profile(True); h.profile_reset()
    timed = [h.nll() for _ in range(5)]
    us, n = h.profile_in_kernel()
    ev_ms, ev_n, _ = h.profile_read()["nll"]
    h.profile(False)
    assert plain == [ref] * 3 and timed == [ref] * 5
    assert n == 5 and ev_n == 5 and 0.0 < us < 1e3 * ev_ms
    h.profile_reset()
    assert h.profile_in_kernel() == (0.0, 0)


def test_in_kernel_timing_of_the_gradient_kernel(B):
    """tddp4_profile_in_kernel_of(TDDP4_K_GRAD): one count per tddp4_nll_grad launch while profiling, positive, below the
    CUDA-event duration of the same launches; the coupling-only counter is a separate one; NLL and gradient bits do not
    depend on the stamps; other kernel ids are rejected."""
    mdl = samples.model_of(("C", 2))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 2), 4_133)
    p4n, _ = samples.flat_sample(10_001)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t); h.load_events(1, p4n)
    h.set_params(par)
    ref_nll, ref_grad = h.nll_grad()
    assert h.profile_in_kernel_of(B.K_GRAD) == (0.0, 0)
    h.profile(True); h.profile_reset()
    timed = [h.nll_grad() for _ in range(4)]
    h.nll()
    us, n = h.profile_in_kernel_of(B.K_GRAD)
    us_nll, n_nll = h.profile_in_kernel_of(B.K_NLL)
    ev_ms, ev_n, _ = h.profile_read()["nll_grad"]
    h.profile(False)
    assert all(v == ref_nll and np.array_equal(g, ref_grad) for v, g in timed)
    assert n == 4 and ev_n == 4 and 0.0 < us < 1e3 * ev_ms
    assert n_nll == 1 and us_nll > 0.0 and (us_nll, n_nll) == h.profile_in_kernel()
    with pytest.raises(B.Tddp4Error):
        h.profile_in_kernel_of(B.K_GRAM)
    h.profile_reset()
    assert h.profile_in_kernel_of(B.K_GRAD) == (0.0, 0)


def test_incremental_gram_has_the_bits_of_a_full_pass(B):
    """with tddp4_set_gram_mode(1) the normalisation columns are kept and a move of few columns
    rebuilds only those; along a trajectory of single-resonance, all-parameter and coupling-only moves G and the NLL must
    be bit-identical to a handle that runs full passes, and incremental passes must actually have happened."""
    mdl = samples.model_of(("C", 3))
    p4, t, _ = samples.data_sample(("C", 3), 1_031)
    p4n, _ = samples.flat_sample(20_011)
    par = W.initial_params(mdl)
    full, inc = B.Tddp4(mdl), B.Tddp4(mdl)
    assert inc.set_gram_mode(1) == 0
    for h in (full, inc):
        h.load_events(0, p4, t); h.load_events(1, p4n)
    traj = W.trajectory(mdl, par, 60, "minuit", seed=77)
    for k, p in enumerate(traj):
        full.set_params(p); inc.set_params(p)
        assert full.nll() == inc.nll(), k
        if k % 7 == 0:
            Gf, nf = full.gram(); Gi, ni = inc.gram()
            assert nf == ni and np.array_equal(Gf, Gi), k
    n_inc = inc.set_gram_mode(-1)
    assert 0 < n_inc < 60
    # a reload drops the stored columns' validity; switching the mode off frees them
    inc.load_events(1, p4n)
    inc.set_params(traj[3]); full.set_params(traj[3])
    assert inc.nll() == full.nll()
    inc.set_gram_mode(0)
    inc.set_params(traj[5]); full.set_params(traj[5])
    assert inc.nll() == full.nll()


def test_sharded_device_path_issues_nccl_collectives(B):
    """The NCCL calls of the sharded device path on ONE rank (the pool has one GPU per box): a one-rank NCCL process group,
    collectives forced, every exchange runs on the handle's stream -- same NLL as the handle alone, exchanges counted."""
    import socket
    import torch
    import torch.distributed as dist
    from paper_1702_06735_b200 import sharded
    if dist.is_initialized():
        pytest.skip("a process group exists already")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1,
                            device_id=torch.device("cuda:0"))
    try:
        mdl = samples.model_of(("C", 2))
        par = W.initial_params(mdl)
        p4, t, _ = samples.data_sample(("C", 2), 2_049)
        p4n, _ = samples.flat_sample(10_001)
        h = B.Tddp4(mdl)
        h.load_events(0, p4, t); h.load_events(1, p4n)
        h.set_params(par)
        direct = h.nll()
        sh = sharded.ShardedNLL(h, always_collective=True)
        sh.set_params(par)
        assert abs(sh.nll() - direct) <= 1e-13 * abs(direct)
        assert sh.exchanges == 2                              # Gram sums + result words (the count exchange is not counted)
        p2 = par.copy(); p2.c[0] *= 1.01
        h.set_params(p2); direct2 = h.nll()
        sh.set_params(p2)                                     # couplings only: the global Gram matrix stays in force
        assert abs(sh.nll() - direct2) <= 1e-13 * abs(direct2)
        assert sh.exchanges == 3
        p3 = par.copy(); p3.mass[1] *= 1.0005
        h.set_params(p3); direct3 = h.nll()
        sh.set_params(p3)
        assert abs(sh.nll() - direct3) <= 1e-13 * abs(direct3)
        assert sh.exchanges == 5
    finally:
        dist.destroy_process_group()


def test_maximum_model_size(B):
    """The limits of include/tddp4.h: 16 couplings, 32 terms (all eight chains twice, both Bose orderings), and a model
    with odd instance and term counts (5 instances, 5 terms)."""
    mdl = W.build_model(list(range(1, 9)) * 2, bose=True)
    assert mdl.n_couplings == 16 and mdl.n_terms == 32
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 3), 777)
    p4n, _ = samples.flat_sample(2_222)
    w = np.random.default_rng(5).uniform(0.5, 1.0, 2_222)
    h = check_against_oracle(B, mdl, par, p4, t, p4n, w)
    from oracle import gradient as OG
    ref, _ = OG.nll_gradient(mdl, par, p4, t, p4n, w)
    _, g = h.nll_grad()
    assert np.max(np.abs(g - ref)) <= 1e-10 * np.abs(ref).max()
    odd = W.build_model([1, 2, 3, 8, 4], bose=False)             # 5 couplings, 5 terms, 6 lineshape instances
    par = W.initial_params(odd)
    check_against_oracle(B, odd, par, p4, t, p4n, w)
    with pytest.raises(B.Tddp4Error):
        B.Tddp4(W.build_model(list(range(1, 9)) * 2 + [1], bose=True))   # 17 couplings / 34 terms: refused at create


def many_instance_model():
    """24 de-duplicated lineshape instances on 10 particle systems (the limits of the tables are 24 and 12): two copies of
    the resonance list under different names, the second copy's K* rho chain on the systems (0,2), (1,3)."""
    mdl = W.Model()
    names = ["K*(892)0", "rho(770)0", "a1(1260)", "K1(1270)", "K2*(1430)", "K1(1400)"]
    for copy in (0, 1):
        for nm in names:
            m0, g0, L = W.RESONANCES[nm]
            mdl.res_names.append(f"{nm}#{copy}"); mdl.res_L.append(L)
            mdl.res_mass.append(m0 * (1.0 + 0.01 * copy)); mdl.res_width.append(g0 * (1.0 + 0.1 * copy))
            mdl.res_r.append(0.0); mdl.res_lineshape.append(W.LS_RUNNING)
    for copy, chains in ((0, (1, 2, 3, 4, 5)), (1, (1, 2, 3, 4))):
        for cid in chains:
            sf, res, perm = W.CHAINS[cid]
            if copy == 1 and cid == 1:
                perm = (0, 2, 1, 3)
            idx = tuple(names.index(r) + 6 * copy for r in res)
            for pm in (perm, W._swap13(perm)):
                mdl.term_sf.append(sf); mdl.term_res.append(idx); mdl.term_perm.append(tuple(pm))
                mdl.term_coupling.append(mdl.n_couplings)
            mdl.n_couplings += 1
    return mdl


def test_many_lineshape_instances(B):
    """n_sys + n_inst = 34: the kinematics kernel needs more than 48 KB of dynamic shared memory (opt-in attribute)."""
    mdl = many_instance_model()
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 3), 515)
    p4n, _ = samples.flat_sample(1_301)
    h = check_against_oracle(B, mdl, par, p4, t, p4n)
    lay = h.layout()
    assert len(lay["inst_res"]) == 24 and len(lay["sys_mask"]) == 10


def test_stale_column_tracking(B):
    """Only the stored columns whose lineshapes moved are rewritten after a mass/width step (nothing is recomputed
    that did not change -- here: nothing is re-stored).  After single-resonance moves, several moves without an
    evaluation in between, and a move back, the stored columns equal the oracle's and the NLL equals, bit for bit,
    that of a fresh handle."""
    mdl = samples.model_of(("C", 3))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 3), 1_537)
    p4n, _ = samples.flat_sample(4_001)
    h = B.Tddp4(mdl)
    h.load_events(0, p4, t); h.load_events(1, p4n)
    h.set_params(par); h.nll()
    names = mdl.res_names

    def columns_ok(p):
        _, _, a = oracle.terms(mdl, p, p4)
        ref = np.zeros((mdl.n_couplings, p4.shape[1]), complex)
        for k, kap in enumerate(mdl.term_coupling):
            ref[kap] += a[k]
        col = h.get(0, B.GET_COLUMNS).cpu().numpy()
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert np.max(np.abs(col - ref) / scale) < TOL_LAYER

    def fresh(p):
        g = B.Tddp4(mdl)
        g.load_events(0, p4, t); g.load_events(1, p4n)
        g.set_params(p)
        return g.nll()

    cur = par.copy()
    for res, what in [("a1(1260)", "mass"), ("K*(892)0", "width"), ("K2*(1430)", "mass"), ("rho(770)0", "mass")]:
        r = names.index(res)
        if what == "mass":
            cur.mass[r] *= 1.002
        else:
            cur.width[r] *= 0.99
        h.set_params(cur)
        assert h.nll() == fresh(cur)
        columns_ok(cur)
    two = cur.copy(); two.mass[names.index("K1(1270)")] *= 1.001
    h.set_params(two)                                            # no evaluation: the stale set must accumulate
    three = two.copy(); three.width[names.index("K1(1400)")] *= 1.01
    h.set_params(three)
    assert h.nll() == fresh(three)
    columns_ok(three)
    h.set_params(par)                                            # all the way back
    assert h.nll() == fresh(par)
    columns_ok(par)


@pytest.mark.parametrize("n,nn", [(300, 900), (70_000, 150_000)])
def test_overlapped_launches_match_synchronous_calls(B, n, nn):
    """The per-call kernels overlap through programmatic dependent launch (a successor becomes resident while its
    predecessors drain).  A batched minuit-like trajectory (kernels back to back, every ordering of NLL / Gram / fused
    kernels) must give, bit for bit, what one synchronous call per point gives -- on a grid that leaves SMs free for
    early successors (small n) and on one that fills the GPU."""
    mdl = samples.model_of(("C", 3))
    par = W.initial_params(mdl)
    if n <= 1000:
        p4, t, _ = samples.data_sample(("C", 3), n)
        p4n, _ = samples.flat_sample(nn)
    else:                                                        # any physical events will do: raw candidates
        p4, t, _, _ = oracle.candidates(mdl, par.tau, 7, 0, 0, n)
        p4n, _, _, _ = oracle.candidates(mdl, par.tau, 7, 2, 0, nn)
    traj = W.trajectory(mdl, par, 150, "minuit")
    hb, hs = B.Tddp4(mdl), B.Tddp4(mdl)
    for h in (hb, hs):
        h.load_events(0, p4, t); h.load_events(1, p4n)
    for rep in range(3):
        vals, st = hb.nll_batch(hb.pack_params(traj))
        assert not st.any()
        if rep == 0:
            ref = []
            for p in traj:
                hs.set_params(p)
                ref.append(hs.nll())
            ref = np.array(ref)
        assert np.array_equal(vals, ref)
