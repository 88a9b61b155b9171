"""Seeded input samples for the parity tests, produced by the ORACLE's generator only (never by the CUDA
path): "drawn from the model" = accepted events of the O-9 generator, "flat" = hit-or-miss on the
Raubold-Lynch weight against its rigorous bound.  Results are cached per process."""
import functools
import math

import numpy as np

import oracle
from paper_1702_06735_b200 import workloads as W

from helpers import breakup


def weight_bound(mdl):
    return math.prod(breakup(*tr) for tr in W.flat_envelope_inputs(mdl))


@functools.lru_cache(maxsize=None)
def flat_sample(n_events, seed=W.BASE_SEED, stream=W.STREAM_NORM):
    """First n_events flat phase-space events of (seed, stream): p4[16][n], candidate indices."""
    mdl = W.flat_model()
    par = W.flat_params(mdl)
    n_cand = int(n_events / 0.06) + 2000
    while True:
        g = oracle.generate(mdl, par, seed, stream, n_cand, 0, 2.0 * weight_bound(mdl), n_events)
        if g["n_accepted"] >= n_events:
            return g["p4"][:, :n_events].copy(), g["index"][:n_events].copy()
        n_cand *= 2


_MODELS = {}


def model_of(key):
    """key: ('C', i) for BASELINE config i, or ('chains', ids tuple, bose)."""
    if key not in _MODELS:
        if key[0] == "C":
            _MODELS[key] = W.config(key[1]).model
        else:
            _MODELS[key] = W.build_model(list(key[1]), bose=key[2])
    return _MODELS[key]


@functools.lru_cache(maxsize=None)
def data_sample(key, n_events, n_pilot=20_000, seed=W.BASE_SEED, stream=W.STREAM_DATA):
    """First n_events accepted events of the model at its initial parameters: p4, t, candidate indices."""
    mdl = model_of(key)
    par = W.initial_params(mdl)
    n_cand = max(4 * n_pilot, 40 * n_events)
    while True:
        g = oracle.generate(mdl, par, seed, stream, n_cand, n_pilot, 1.2, n_events)
        if g["n_accepted"] >= n_events:
            return g["p4"][:, :n_events].copy(), g["t"][:n_events].copy(), g["index"][:n_events].copy()
        n_cand *= 2


def rel_err(a, b, floor=0.0):
    """max |a-b| / max(|b|, floor) element-wise (b = oracle)."""
    a, b = np.asarray(a), np.asarray(b)
    if a.size == 0:
        return 0.0
    return float(np.max(np.abs(a - b) / np.maximum(np.abs(b), floor if floor > 0 else np.finfo(float).tiny)))
