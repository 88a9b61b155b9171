#!/usr/bin/env python
"""Writes tests/golden/oracle_c1_10events.txt: the oracle's own per-event results on a 10-event input of BASELINE config 1.

It calls ONLY `oracle/` (and the plain-data tables of workloads.py); nothing here comes from the CUDA path.  The file is a
regression fixture: it freezes the oracle's arithmetic (readings O-1..O-9 of DESIGN.md 3) so that a later change to it
is visible in review and has to name the passage that justifies it.  The values themselves are pinned independently by
tests/test_oracle_bruteforce.py (mpmath recomputation at 30 digits of the same kind of input).

    python tests/golden/make_golden.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "..", ".."))

import numpy as np  # noqa: E402

import oracle  # noqa: E402
from paper_1702_06735_b200 import workloads as W  # noqa: E402

N_DATA, N_NORM, FIRST_NORM = 10, 200, 1_000_000


def compute():
    mdl = W.config(1).model
    par = W.initial_params(mdl)
    # data: RL candidates 0..9 of stream 0 taken as they come (no accept step), norm: candidates of stream 2
    p4, t, w, _ = oracle.candidates(mdl, par.tau, W.BASE_SEED, W.STREAM_DATA, 0, N_DATA)
    p4n, _, wn, _ = oracle.candidates(mdl, par.tau, W.BASE_SEED, W.STREAM_NORM, FIRST_NORM, N_NORM)
    nll, norm, P, st = oracle.nll(mdl, par, p4, t, p4n, wn)      # RL weights as normalisation weights
    A, Ab = oracle.amplitudes(mdl, par, p4)
    assert st == 0
    return dict(p4=p4, t=t, w=w, A=A, Ab=Ab, P=P, nll=nll, norm=norm)


def main():
    r = compute()
    path = os.path.join(HERE, "oracle_c1_10events.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_golden.py (calls only oracle/); BASELINE config 1 model, seed 42\n")
        f.write("# data = Raubold-Lynch candidates 0..9 of Philox stream 0; normalisation = candidates 1000000..1000199 of\n")
        f.write("# stream 2 weighted by their phase-space weight.  eq. (1)/(2): PAPER.md lines 30-32, 46-49.\n")
        f.write(f"nll {r['nll']!r}\nnorm {r['norm']!r}\n")
        f.write("# i  E_K  t  w  ReA  ImA  ReAbar  ImAbar  P\n")
        for i in range(N_DATA):
            vals = [r["p4"][0, i], r["t"][i], r["w"][i], r["A"][i].real, r["A"][i].imag, r["Ab"][i].real,
                    r["Ab"][i].imag, r["P"][i]]
            f.write(f"{i} " + " ".join(repr(float(v)) for v in vals) + "\n")
    print(path)


if __name__ == "__main__":
    main()
