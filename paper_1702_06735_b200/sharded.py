"""Event-sharded NLL across ranks: host-side logic only, argument marshalling and one exchange.

Events are independent, so data and normalisation samples are split into contiguous index blocks, one per rank
(one process per GPU).  Per minimiser call the only data that must cross ranks is

  * the K_c x K_c Hermitian Gram sums of the normalisation shards (only when a mass or width moved), and
  * per rank of the data pass: its local NLL (evaluated with the GLOBAL normalisation), its event count and its number
    of bad events,

because with N (or, with per-event resolution, S_1..S_4) taken from the global Gram matrix the NLL is a plain sum over
events: -sum_i log P_i = sum over ranks of (Gamma sum t - sum log B + n_r log N)_r.  Both exchanges are
all-gathers of a few hundred bytes followed by a sum IN RANK ORDER on every rank, so every rank holds the same bits
and the result does not depend on arrival order.  (An all-reduce would be one call less; NCCL's reduction order is
not specified, and at 2 K_c^2 + 1 doubles the exchange is latency-bound either way.)

`evaluator` is anything with the four methods of `binding.Tddp4` used here (set_params, gram, gram_override, nll,
nll_parts): the CUDA handle in production, a stand-in in the CPU (gloo) tests.
"""
from __future__ import annotations

import math

import numpy as np


def shard_range(n: int, rank: int, world: int):
    """Contiguous block [lo, hi) of rank `rank` when n events are split over `world` ranks; sizes differ by at
    most one, earlier ranks take the larger blocks."""
    base, rem = divmod(int(n), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


class ShardedNLL:
    def __init__(self, evaluator, group=None):
        import torch.distributed as dist
        self.ev = evaluator
        self.dist = dist
        self.group = group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self._mw = None          # masses/widths the global Gram matrix in force was built for
        self.exchanges = 0       # all-gather calls issued (for tests / launch accounting)

    def _all_gather(self, vec: np.ndarray) -> np.ndarray:
        """[world][len(vec)] float64, identical on every rank."""
        if self.world == 1:
            return vec[None, :].copy()
        import torch
        mine = torch.from_numpy(np.ascontiguousarray(vec, dtype=np.float64))
        if self.dist.get_backend(self.group) == "nccl":          # NCCL moves device memory only
            mine = mine.cuda()
        out = [torch.empty_like(mine) for _ in range(self.world)]
        self.dist.all_gather(out, mine, group=self.group)
        self.exchanges += 1
        return np.stack([o.cpu().numpy() for o in out])

    def set_params(self, par):
        self.par = par
        self.ev.set_params(par)
        mw = (tuple(np.asarray(par.mass, float)), tuple(np.asarray(par.width, float)))
        if mw != self._mw:                      # normalisation shards changed: exchange the Gram sums once
            G, n = self.ev.gram()
            kc = G.shape[0]
            flat = np.concatenate([np.real(G).ravel(), np.imag(G).ravel(), [float(n)]])
            allv = self._all_gather(flat)
            tot = np.zeros_like(flat)
            for r in range(self.world):         # rank order: same bits everywhere
                tot = tot + allv[r]
            Gt = tot[:kc * kc].reshape(kc, kc) + 1j * tot[kc * kc:2 * kc * kc].reshape(kc, kc)
            self.ev.gram_override(Gt, int(round(tot[-1])))
            self._mw = mw

    def nll(self):
        """Global NLL, the same double on every rank; +inf if any rank saw a non-positive rate."""
        self.ev.nll(strict=False)
        p = self.ev.nll_parts()
        allv = self._all_gather(np.array([p["nll"], float(self.ev.n_data), p["n_bad"]]))
        total = bad = 0.0
        for r in range(self.world):             # rank order: same bits everywhere
            if allv[r, 1] > 0:
                total += allv[r, 0]
            bad += allv[r, 2]
        if bad > 0 or not math.isfinite(total):
            return math.inf
        return total
