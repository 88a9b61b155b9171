"""A thin host fit loop around the C-ABI: the minimiser stays on the host (BASELINE.json north_star; the paper drives its
fits with a MINUIT-type minimiser).  Every objective evaluation is ONE `tddp4_nll_grad` call
(NLL and analytic gradient from one pass over the cached columns); nothing of the likelihood is computed here.

Floating parameters: any subset of the couplings (Re/Im of c_k, cbar_k) and the mixing parameters x, y; masses, widths
and tau stay at the values of `par0` (their derivatives are not provided by the library; float them with a
derivative-free outer loop and `tddp4_nll_batch` if needed).  The overall phase and scale of all couplings are null
directions of a normalised likelihood: fix at least one complex coupling (the default fixes c_0).

    res = fit(handle, par0, free_couplings="all_but_first", free_xy=True)
    res.par, res.nll, res.errors["x"], res.n_calls
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
from scipy import optimize


@dataclass
class FitResult:
    par: object
    nll: float
    n_calls: int
    success: bool
    message: str
    free: np.ndarray                     # indices into the gradient layout [4 K_c + 2] that floated
    covariance: np.ndarray | None = None
    errors: dict = field(default_factory=dict)


def _theta(par):
    return np.concatenate([np.asarray(par.c, complex).view(float), np.asarray(par.cbar, complex).view(float),
                           [par.x, par.y]])


def _with_theta(par, th):
    kc = len(par.c)
    p = par.copy()
    p.c = th[:2 * kc].view(complex).copy()
    p.cbar = th[2 * kc:4 * kc].view(complex).copy()
    p.x, p.y = float(th[4 * kc]), float(th[4 * kc + 1])
    return p


def free_indices(kc, free_couplings="all_but_first", free_xy=True):
    """Indices of the floating entries in the layout of tddp4_nll_grad."""
    idx = []
    if free_couplings == "all_but_first":
        idx += list(range(2, 4 * kc))
    elif free_couplings == "all":
        idx += list(range(4 * kc))
    elif free_couplings not in (None, "none"):
        idx += [int(i) for i in free_couplings]
    if free_xy:
        idx += [4 * kc, 4 * kc + 1]
    return np.array(sorted(set(idx)), dtype=int)


def fit(handle, par0, free_couplings="all_but_first", free_xy=True, hesse=True, gtol=1e-6, maxiter=500):
    """Minimise the NLL of `handle` (data and normalisation samples loaded) over the chosen parameters with
    scipy's BFGS and the analytic gradient; `hesse`: covariance from a central-difference Hessian of the gradient at
    the minimum (two gradient calls per floating parameter)."""
    kc = len(par0.c)
    free = free_indices(kc, free_couplings, free_xy)
    th0 = _theta(par0)
    scale = np.maximum(np.abs(th0[free]), 1e-3)          # BFGS in units of the start values: x, y ~ 5e-3, couplings ~ 1
    calls = [0]

    def objective(u):
        th = th0.copy()
        th[free] = u * scale
        handle.set_params(_with_theta(par0, th))
        nll, g = handle.nll_grad()
        calls[0] += 1
        return nll, g[free] * scale

    res = optimize.minimize(objective, th0[free] / scale, jac=True, method="BFGS", options={"gtol": gtol, "maxiter": maxiter})
    th = th0.copy()
    th[free] = res.x * scale
    best = _with_theta(par0, th)
    # BFGS stops with "precision loss" once the NLL (~1e3..1e6) no longer changes in its last digits: converged if the
    # scaled gradient is small against the size of the function
    converged = bool(res.success) or float(np.max(np.abs(res.jac))) < 1e-7 * max(1.0, abs(float(res.fun)))
    out = FitResult(par=best, nll=float(res.fun), n_calls=calls[0], success=converged, message=str(res.message), free=free)
    if hesse:
        n = len(free)
        H = np.empty((n, n))
        for j in range(n):
            h = 1e-4 * scale[j]
            up, dn = th.copy(), th.copy()
            up[free[j]] += h
            dn[free[j]] -= h
            handle.set_params(_with_theta(par0, up)); _, gu = handle.nll_grad()
            handle.set_params(_with_theta(par0, dn)); _, gd = handle.nll_grad()
            calls[0] += 2
            H[j] = (gu[free] - gd[free]) / (2 * h)
        H = 0.5 * (H + H.T)
        try:
            cov = np.linalg.inv(H)
            out.covariance = cov
            names = {4 * kc: "x", 4 * kc + 1: "y"}
            for j, i in enumerate(free):
                if i in names and cov[j, j] > 0:
                    out.errors[names[i]] = float(np.sqrt(cov[j, j]))
        except np.linalg.LinAlgError:
            pass
        out.n_calls = calls[0]
        handle.set_params(best)
    return out


def sensitivity_study(binding, model, par, sizes=(20_000, 50_000, 70_000), n_toys=50, n_norm=1_000_000, device="cuda:0",
                      seed=4242, flat_model=None, flat_par=None, n_pilot=100_000, envelope_scale=1.2):
    """The shape of the paper's Table 1 (statistical sensitivity to x and y against the number of
    events, model fixed, no resolution, no background): for every sample size an ensemble of `n_toys` independent
    pseudo-experiments, each generated with tddp4_generate from `model` at `par` (own Philox seed) and fitted for x and
    y with `fit` (couplings fixed).  Orchestration only: generation, kinematics, NLL and gradient run behind the C-ABI.

    Returns one dict per size: mean Hessian errors, the ensemble RMS of the fitted values and the mean pulls."""
    import numpy as _np
    stream_norm, stream_data = 2, 0
    if flat_model is not None:
        hf = binding.Tddp4(flat_model, device)
        hf.set_params(flat_par)
        p4n, _, _, _ = hf.generate_n(seed, stream_norm, n_norm, 0, 2.0 * hf.weight_bound(), chunk=1 << 24)
        hf.close()
    else:
        raise ValueError("a constant-amplitude model is needed to un-weight the normalisation sample")
    gen = binding.Tddp4(model, device)
    gen.set_params(par)
    h = binding.Tddp4(model, device)
    h.load_events(1, p4n)
    rows, toy = [], 0
    for n in sizes:
        xs, ys, sx, sy, calls = [], [], [], [], 0
        for _ in range(n_toys):
            toy += 1
            p4, t, _, _ = gen.generate_n(seed + toy, stream_data, n, n_pilot, envelope_scale, chunk=1 << 23)
            h.load_events(0, p4, t)
            res = fit(h, par, free_couplings=None, free_xy=True)
            calls += res.n_calls
            if res.success and "x" in res.errors and "y" in res.errors:
                xs.append(res.par.x); ys.append(res.par.y); sx.append(res.errors["x"]); sy.append(res.errors["y"])
        xs, ys, sx, sy = map(_np.asarray, (xs, ys, sx, sy))
        rows.append({"n_events": int(n), "n_toys": int(len(xs)), "sigma_x_hesse": float(sx.mean()), "sigma_y_hesse": float(sy.mean()),
                     "rms_x": float(xs.std(ddof=1)), "rms_y": float(ys.std(ddof=1)),
                     "pull_mean_x": float(((xs - par.x) / sx).mean()), "pull_mean_y": float(((ys - par.y) / sy).mean()),
                     "pull_rms_x": float(((xs - par.x) / sx).std(ddof=1)), "pull_rms_y": float(((ys - par.y) / sy).std(ddof=1)),
                     "nll_grad_calls_per_fit": calls / max(1, n_toys)})
    gen.close()
    h.close()
    return rows
