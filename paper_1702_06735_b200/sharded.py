"""Event-sharded NLL across ranks: host-side logic only -- argument marshalling and one exchange.

Events are independent, so data and normalisation samples are split into contiguous index blocks, one per rank
(one process per GPU).  Per minimiser call the only data that must cross ranks is

  * the K_c x K_c Hermitian Gram sums of the normalisation shards (only when a mass or width moved), and
  * per rank of the data pass: its NLL term (evaluated with the GLOBAL normalisation) and its number of bad events,

because with N (or, with per-event resolution, S_1..S_4) taken from the global Gram matrix the NLL is a plain sum over
events: -sum_i log P_i = sum over ranks of (Gamma sum t - sum log B + n_r log N)_r.  Both exchanges are
all-gathers of a few hundred bytes followed by a sum IN RANK ORDER, so every rank holds the same bits and the result
does not depend on arrival order.  (An all-reduce would be one call less; NCCL's reduction order is not specified, and
at 2 K_c^2 + 1 doubles the exchange is latency-bound either way.)

Two paths, chosen from what the evaluator offers:

  * device path (the CUDA handle, `binding.Tddp4`): `gram_enqueue` -> all-gather -> `gram_reduce` and `nll_enqueue` ->
    all-gather run back to back on the handle's stream (the collective is issued under that stream, NCCL or none at
    world size 1); the rank-ordered Gram sum is one kernel of the library; the only synchronisation of a call is the
    read of the gathered world x 8 result words from a pinned buffer.  All buffers are allocated once.
  * host path (any object with set_params / gram / gram_override / nll / nll_parts: the stand-in of the CPU gloo tests).
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
    def __init__(self, evaluator, group=None, always_collective=False):
        """always_collective: issue the collectives even at world size 1 (a one-rank process group): the single-GPU check
        of the NCCL calls of the device path (tests, `bench.py --sharded`)."""
        import torch.distributed as dist
        self.ev = evaluator
        self.dist = dist
        self.group = group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.backend = dist.get_backend(group) if dist.is_initialized() else None
        self.exchanges = 0       # collectives issued (for tests / launch accounting)
        self._mw = None          # host path: masses/widths the global Gram matrix in force was built for
        self._n_norm_total = None
        self.device_path = hasattr(evaluator, "nll_enqueue") and (self.world == 1 or self.backend == "nccl")
        self.always_collective = bool(always_collective) and dist.is_initialized() and self.backend == "nccl"
        if self.device_path:
            import torch
            self.torch = torch
            ev = evaluator
            if getattr(ev, "stream", None) is None:          # the collective must run on the handle's stream
                ev.set_stream(torch.cuda.Stream(ev.device))
            self.stream = ev.stream
            glen = 2 * ev.kc * ev.kc + 1
            f64 = dict(dtype=torch.float64, device=ev.device)
            self.g_mine, self.g_all = torch.zeros(glen, **f64), torch.zeros(self.world, glen, **f64)
            self.r_mine, self.r_all = torch.zeros(8, **f64), torch.zeros(self.world, 8, **f64)
            self.r_host = torch.zeros(self.world, 8, dtype=torch.float64).pin_memory()

    # -- exchange primitives ----------------------------------------------------------------------
    def _all_gather_host(self, vec: np.ndarray) -> np.ndarray:
        """[world][len(vec)] float64, identical on every rank (host path)."""
        if self.world == 1:
            return vec[None, :].copy()
        import torch
        mine = torch.from_numpy(np.ascontiguousarray(vec, dtype=np.float64))
        if self.backend == "nccl":                            # NCCL moves device memory only
            mine = mine.cuda()
        out = [torch.empty_like(mine) for _ in range(self.world)]
        self.dist.all_gather(out, mine, group=self.group)
        self.exchanges += 1
        return np.stack([o.cpu().numpy() for o in out])

    def _all_gather_device(self, out, mine):
        """Enqueued on the current (= the handle's) stream; world size 1 needs no collective."""
        if self.world == 1 and not self.always_collective:
            out[0].copy_(mine)
        else:
            self.dist.all_gather_into_tensor(out, mine, group=self.group)
            self.exchanges += 1

    def _norm_total(self):
        """Sum of the ranks' normalisation sample sizes; exchanged once per loaded sample (host integers)."""
        if self._n_norm_total is None:
            n = float(self.ev.n[1])
            if self.world == 1 and not self.always_collective:
                self._n_norm_total = int(n)
            else:
                t = self.torch.tensor([n], dtype=self.torch.float64, device=self.ev.device)
                out = self.torch.zeros(self.world, dtype=self.torch.float64, device=self.ev.device)
                self.dist.all_gather_into_tensor(out, t, group=self.group)
                self._n_norm_total = int(round(float(out.sum().item())))
        return self._n_norm_total

    # -- the evaluator's interface, sharded --------------------------------------------------------
    def load_events(self, which, *args, **kw):
        """Forwarded to the evaluator; a new normalisation shard invalidates the global Gram matrix and the count."""
        self.ev.load_events(which, *args, **kw)
        if which == 1:
            self._mw = None
            self._n_norm_total = None

    def set_params(self, par):
        self.par = par
        self.ev.set_params(par)
        if self.device_path:
            valid, overridden = self.ev.gram_state()
            if valid and overridden:                        # the global matrix in force still matches the masses/widths
                return
            n_total = self._norm_total()
            with self.torch.cuda.stream(self.stream):
                self.ev.gram_enqueue(self.g_mine)
                self._all_gather_device(self.g_all, self.g_mine)
                self.ev.gram_reduce(self.g_all, self.world, n_total)
            return
        mw = (tuple(np.asarray(par.mass, float)), tuple(np.asarray(par.width, float)))
        state = getattr(self.ev, "gram_state", None)
        in_force = state is None or all(state())            # a reloaded sample or an explicit gram() drops the override
        if mw != self._mw or not in_force:                  # normalisation changed: exchange the Gram sums once
            G, n = self.ev.gram()
            kc = G.shape[0]
            flat = np.concatenate([np.real(G).ravel(), np.imag(G).ravel(), [float(n)]])
            allv = self._all_gather_host(flat)
            tot = np.zeros_like(flat)
            for r in range(self.world):         # rank order: same bits everywhere
                tot = tot + allv[r]
            Gt = tot[:kc * kc].reshape(kc, kc) + 1j * tot[kc * kc:2 * kc * kc].reshape(kc, kc)
            self.ev.gram_override(Gt, int(round(tot[-1])))
            self._mw = mw

    def nll(self):
        """Global NLL, the same double on every rank; +inf if any rank saw a non-positive rate."""
        if self.device_path:
            with self.torch.cuda.stream(self.stream):
                self.ev.nll_enqueue(self.r_mine)
                self._all_gather_device(self.r_all, self.r_mine)
                self.r_host.copy_(self.r_all, non_blocking=True)
            self.stream.synchronize()
            allv = self.r_host.numpy()
            total = bad = 0.0
            for r in range(self.world):         # rank order: same bits everywhere
                total += allv[r, 3]
                bad += allv[r, 4]
            return math.inf if bad > 0 or not math.isfinite(total) else float(total)
        self.ev.nll(strict=False)
        p = self.ev.nll_parts()
        allv = self._all_gather_host(np.array([p["nll"], float(self.ev.n_data), p["n_bad"]]))
        total = bad = 0.0
        for r in range(self.world):             # rank order: same bits everywhere
            if allv[r, 1] > 0:
                total += allv[r, 0]
            bad += allv[r, 2]
        if bad > 0 or not math.isfinite(total):
            return math.inf
        return total
