"""the N > 1 path on CPU.  Two processes (gloo, world_size 2) each own a contiguous shard of the data
and normalisation samples; `sharded.ShardedNLL` exchanges Gram sums and three scalars per call and must reproduce the
single-process NLL.  The per-rank evaluator here is a stand-in with the interface of `binding.Tddp4` built on the
oracle (this is a test: the product path has no CPU evaluator), so what is under test is the host logic: shard
ranges, the rank-ordered sums, when the Gram exchange happens, the NLL recombination, the +inf propagation."""
import math
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1702_06735_b200 import sharded, workloads as W

import samples


class OracleEvaluator:
    """gram / gram_override / nll / nll_parts of one shard, from oracle pieces only."""

    def __init__(self, mdl, p4, t, p4n):
        self.mdl, self.p4, self.t, self.p4n = mdl, p4, t, p4n
        self.n_data = p4.shape[1]
        self.gram_calls = 0

    def set_params(self, par):
        self.par = par

    def load_events(self, which, p4, t=None):
        if which == 0:
            self.p4, self.t, self.n_data = p4, t, p4.shape[1]
        else:
            self.p4n = p4

    def _columns(self, p4):
        if p4.shape[1] == 0:
            return np.zeros((self.mdl.n_couplings, 0), complex)
        a = oracle.terms(self.mdl, self.par, p4)[2]
        col = np.zeros((self.mdl.n_couplings, p4.shape[1]), complex)
        for k, kap in enumerate(self.mdl.term_coupling):
            col[kap] += a[k]
        return col

    def gram(self):
        self.gram_calls += 1
        col = self._columns(self.p4n)
        return col @ col.conj().T, self.p4n.shape[1]

    def gram_override(self, G, n):
        self.G, self.n_norm = G / n, n

    def nll(self, strict=True):
        par = self.par
        T = oracle.time_integrals(par.x, par.y, par.tau, self.mdl.t_lo, self.mdl.t_hi)
        c, cb, G = np.asarray(par.c), np.asarray(par.cbar), self.G
        nAA, nBB = (c @ G @ c.conj()).real, (cb @ G @ cb.conj()).real
        X = c @ G @ cb.conj()
        self.norm = T[0] * (nAA + nBB) + T[1] * (nAA - nBB) - 2 * T[2] * X.real - 2 * T[3] * X.imag
        if self.n_data:
            B = oracle.rate(self.mdl, par, self.p4, self.t)[1]
        else:
            B = np.zeros(0)
        self.bad = int(np.sum(~(B > 0)))
        self.slb = float(np.sum(np.log(B[B > 0])))
        return 0.0

    def nll_parts(self):
        st = float(np.sum(self.t))
        local = st / self.par.tau - self.slb + self.n_data * math.log(self.norm)   # with the GLOBAL normalisation
        return dict(sum_log_B=self.slb, sum_t=st, norm=self.norm, nll=local, n_bad=self.bad)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_data, n_norm, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mdl = samples.model_of(("C", 1))
        par = W.initial_params(mdl)
        p4, t, _ = samples.data_sample(("C", 1), n_data)
        p4n, _ = samples.flat_sample(n_norm)
        lo, hi = sharded.shard_range(n_data, rank, world)
        ln, hn = sharded.shard_range(n_norm, rank, world)
        ev = OracleEvaluator(mdl, p4[:, lo:hi].copy(), t[lo:hi].copy(), p4n[:, ln:hn].copy())
        sh = sharded.ShardedNLL(ev)
        vals = []
        sh.set_params(par)
        vals.append(sh.nll())
        p2 = par.copy(); p2.c[0] *= 1.01; p2.x *= 1.1            # coupling/x step: no Gram exchange
        sh.set_params(p2)
        vals.append(sh.nll())
        p3 = p2.copy(); p3.mass[0] *= 1.001                      # mass step: Gram exchange
        sh.set_params(p3)
        vals.append(sh.nll())
        counts = (ev.gram_calls, sh.exchanges)
        # a reloaded normalisation shard with unchanged masses/widths must trigger a new exchange
        half = (hn - ln) // 2
        sh.load_events(1, p4n[:, ln:ln + half].copy())
        sh.set_params(p3)
        vals.append(sh.nll())
        out[rank] = (vals, counts[0], counts[1], ev.gram_calls, (ln, ln + half))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_data,n_norm", [(301, 2_001), (1, 7)])
def test_world_size_2_matches_single_process(n_data, n_norm):
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), n_data, n_norm, out), nprocs=world, join=True)
    mdl = samples.model_of(("C", 1))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 1), n_data)
    p4n, _ = samples.flat_sample(n_norm)
    p2 = par.copy(); p2.c[0] *= 1.01; p2.x *= 1.1
    p3 = p2.copy(); p3.mass[0] *= 1.001
    ref = [oracle.nll(mdl, p, p4, t, p4n, want_prob=False)[0] for p in (par, p2, p3)]
    keep = np.concatenate([np.arange(*out[r][4]) for r in range(world)])      # the halved normalisation shards
    if len(keep):
        ref.append(oracle.nll(mdl, p3, p4, t, np.ascontiguousarray(p4n[:, keep]), want_prob=False)[0])
    assert out[0][0] == out[1][0]                                # same bits on both ranks
    for got, want in zip(out[0][0], ref):
        assert abs(got - want) <= 1e-11 * max(abs(want), 1.0)
    for r in range(world):
        assert out[r][1] == 2                                    # Gram rebuilt at the first call and at the mass step only
        assert out[r][2] == 2 + 3                                # 2 Gram exchanges + 3 scalar exchanges
        assert out[r][3] == 3                                    # ... and once more after the reload


def test_shard_ranges_partition_the_events():
    for n in (0, 1, 5, 1000, 1_000_003):
        for world in (1, 2, 3, 8):
            cuts = [sharded.shard_range(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def test_single_process_needs_no_process_group():
    mdl = samples.model_of(("C", 1))
    par = W.initial_params(mdl)
    p4, t, _ = samples.data_sample(("C", 1), 50)
    p4n, _ = samples.flat_sample(400)
    sh = sharded.ShardedNLL(OracleEvaluator(mdl, p4, t, p4n))
    sh.set_params(par)
    ref = oracle.nll(mdl, par, p4, t, p4n, want_prob=False)[0]
    assert abs(sh.nll() - ref) <= 1e-11 * abs(ref) and sh.exchanges == 0
