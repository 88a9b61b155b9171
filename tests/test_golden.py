"""The oracle against the stored fixtures of tests/golden/ (see its README for where each value comes from)."""
import importlib.util
import math
import os

import numpy as np
import pytest

import oracle
from paper_1702_06735_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def closed_forms():
    rows = []
    with open(os.path.join(GOLD, "closed_forms.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if line:
                rows.append(line)
    return rows


def make_golden():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(GOLD, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_lineshape_pole_values():
    """T_R(m0^2) = i/(m0 Gamma0) (O-6): the oracle's Breit-Wigner at s = m0^2 against the typed-in values."""
    seen = 0
    for row in closed_forms():
        if row[0] != "bw_pole_im":
            continue
        name, m0, g0, want, tol = row[1], float(row[2]), float(row[3]), float(row[4]), float(row[5])
        m0_tab, g0_tab, L = W.RESONANCES[name]
        assert (m0_tab, g0_tab) == (m0, g0)
        # two-body daughters: K pi for the K-type resonances, pi pi otherwise (three-body ones: a light stand-in pair;
        # the pole value does not depend on the daughters)
        ma, mb = (W.M_K, W.M_PI) if name.startswith("K") else (W.M_PI, W.M_PI)
        T = oracle.breit_wigner(m0, g0, L, 1.5, m0 * m0, ma, mb)
        assert abs(T.real) < 1e-9 * abs(T.imag)
        assert abs(T.imag / want - 1.0) < tol
        seen += 1
    assert seen == 4


def test_massless_volume_and_weight_bound():
    rows = {r[0]: r for r in closed_forms()}
    M, want, tol = (float(v) for v in rows["massless_volume_n4"][1:4])
    assert abs(math.pi ** 3 * M ** 4 / 96.0 / want - 1.0) < tol
    # the generator's mean weight reproduces that volume (massless final state): (2^2 pi^3 T^2 / (M 2!)) <w>
    mdl = W.flat_model(m_parent=M, m_final=(0.0, 0.0, 0.0, 0.0))
    _, _, w, _ = oracle.candidates(mdl, 1.0, 7, 0, 0, 400_000)
    vol = 4.0 * math.pi ** 3 * M ** 2 / (M * 2.0) * float(np.mean(w))
    assert abs(vol / want - 1.0) < 4e-3                          # MC error of 4e5 samples ~ 1.2e-3
    bound, btol = float(rows["rl_weight_bound"][1]), float(rows["rl_weight_bound"][2])
    got = math.prod(oracle.breakup(*tr) for tr in W.flat_envelope_inputs(W.flat_model()))
    assert abs(got / bound - 1.0) < btol


def test_paper_mixing_parameters():
    rows = {r[0]: r for r in closed_forms()}
    assert W.X_MIX == float(rows["paper_x"][1]) and W.Y_MIX == float(rows["paper_y"][1])


def read_fixture():
    vals, rows = {}, []
    with open(os.path.join(GOLD, "oracle_c1_10events.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            p = line.split()
            if p[0] in ("nll", "norm"):
                vals[p[0]] = float(p[1])
            else:
                rows.append([float(v) for v in p[1:]])
    return vals, np.array(rows)


def test_oracle_reproduces_its_fixture():
    """Regression: today's oracle gives the stored values (1e-13: libm may differ in the last bits between boxes)."""
    vals, rows = read_fixture()
    r = make_golden().compute()
    assert abs(r["nll"] - vals["nll"]) < 1e-12 * abs(vals["nll"])
    assert abs(r["norm"] / vals["norm"] - 1) < 1e-13
    got = np.stack([r["p4"][0], r["t"], r["w"], r["A"].real, r["A"].imag, r["Ab"].real, r["Ab"].imag, r["P"]], axis=1)
    assert np.max(np.abs(got - rows) / np.maximum(np.abs(rows), 1e-3)) < 1e-12


@pytest.mark.gpu
def test_cuda_path_reproduces_the_oracle_fixture():
    """The stored oracle values against the CUDA path through the C-ABI (generator candidates, weights, P_i, NLL)."""
    from paper_1702_06735_b200 import binding
    mg = make_golden()
    vals, rows = read_fixture()
    mdl = W.config(1).model
    par = W.initial_params(mdl)
    h = binding.Tddp4(mdl)
    h.set_params(par)
    p4, t, _, _, _ = h.candidates(W.BASE_SEED, W.STREAM_DATA, 0, mg.N_DATA)
    p4n, _, wn, _, _ = h.candidates(W.BASE_SEED, W.STREAM_NORM, mg.FIRST_NORM, mg.N_NORM)
    h.load_events(0, p4, t)
    h.load_events(1, p4n, None, weight=wn)
    prob = h.empty(mg.N_DATA)
    nll = h.nll(prob)
    assert np.max(np.abs(p4[0].cpu().numpy() - rows[:, 0])) < 1e-12
    assert np.max(np.abs(t.cpu().numpy() / rows[:, 1] - 1)) < 1e-12
    assert np.max(np.abs(prob.cpu().numpy() / rows[:, 7] - 1)) < 1e-10
    assert abs(nll - vals["nll"]) < 1e-11 * max(abs(vals["nll"]), 1e-3 * float(np.sum(np.abs(np.log(rows[:, 7])))))
