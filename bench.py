#!/usr/bin/env python
"""bench.py -- throughput of the hot path on BASELINE.json's headline workload (configs[2], "C3" in SURVEY.md 8):
1 000 000 data events, 4 000 000 flat normalisation events, 16 Bose-symmetrised terms on 8 couplings, masses and
widths floating, consecutive NLL evaluations along a seeded MINUIT-like parameter trajectory.

One "step" = one NLL evaluation (tddp4_set_params + tddp4_nll): lineshapes and coupling columns are refreshed for
whatever that step's parameter change made dirty, the Gram matrix of the normalisation sample is rebuilt if a
mass or width moved, then the amplitude-sum + rate + -log pass runs over the data sample.  Kinematics and spin
factors (step 1) run once per event set, at load, as the paper's de-duplication licence allows.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N = 1: the headline above plus the other configs, the generator, the fit-shaped extras.  N > 1 (the script re-launches
itself under torch.distributed.run when it was not started by a launcher): the EVENT-SHARDED evaluation of SURVEY.md
8(e) through `sharded.ShardedNLL` -- every rank holds a C3-sized shard (1 M + 4 M events) of an N times larger sample
(weak scaling), one Gram exchange per mass/width move and one 8-word exchange per call over NCCL on the handle's stream;
the strong-scaling figure of ONE C3 sample split N ways is reported next to it.

Prints ONE JSON line (see DESIGN.md "Measurement" for every key).  Metric: events x NLL evaluations per second.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1702_06735_b200 import workloads as W  # noqa: E402

METRIC = "nll_events_x_evals_per_s"
UNIT = "events*evals/s"
WORKLOAD = "C3"
TRAJECTORY = "minuit"


def csrc_sha16():
    """Hash of the CUDA sources: the committed ncu traffic figures are only quoted for the sources they were taken on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1702_06735_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".h")):
            with open(os.path.join(d, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def committed_table(name):
    """profiles/<name>.csv as {kernel: row dict}; rows whose csrc_sha16 differs from the current sources are dropped."""
    import csv
    path = os.path.join(ROOT, "profiles", name)
    if not os.path.exists(path):
        return {}, "absent"
    sha = csrc_sha16()
    with open(path) as f:
        rows = list(csv.DictReader(f))
    good = {r["kernel"]: r for r in rows if r.get("csrc_sha16", "") == sha}
    if rows and not good:
        return {}, f"stale: profiles/{name} was captured on csrc {rows[0].get('csrc_sha16')}, sources are now {sha}"
    return good, f"profiles/{name} (ncu capture on csrc {sha})"


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.01):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.sm, self.reasons, self.stop_flag = [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    NAMES = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
             0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}

    def run(self):
        if self.nv is None:
            return
        while not self.stop_flag:
            try:
                self.sm.append(self.nv.nvmlDeviceGetClockInfo(self.dev, self.nv.NVML_CLOCK_SM))
                r = self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev)
                for bit, name in self.NAMES.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        self.stop_flag = True
        if self.is_alive():
            self.join()
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


def build_workload(binding, cfg, device, seed):
    """Seeded synthetic samples of the config, produced on the device by the CUDA generator:
    flat normalisation sample = hit-or-miss on the Raubold-Lynch weight; data = accept-reject against the model."""
    flat = W.flat_model()
    hf = binding.Tddp4(flat, device)
    hf.set_params(W.flat_params(flat))
    p4n, _, idxn, _ = hf.generate_n(seed, W.STREAM_NORM, cfg.n_norm, 0, 2.0 * hf.weight_bound(), chunk=1 << 24, want_index=True)
    hf.close()
    hg = binding.Tddp4(cfg.model, device)
    hg.set_params(W.initial_params(cfg.model))
    p4, t, idx, info = hg.generate_n(seed, W.STREAM_DATA, cfg.n_data, cfg.n_pilot, cfg.envelope_scale, chunk=1 << 24, want_index=True)
    hg.close()
    info["index"], info["index_norm"], info["seed"] = idx, idxn, seed      # candidate indices: the oracle regenerates from them
    return p4, t, p4n, info


def kernel_table(prof, total_ms):
    hbm, which = peaks()
    out = {}
    for name, (ms, n, by) in prof.items():
        if n == 0:
            continue
        gbs = by / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
        out[name] = {"launches": n, "ms": round(ms, 4), "share": round(ms / total_ms, 4) if total_ms > 0 else None,
                     "us_per_launch": round(1e3 * ms / n, 3), "alg_MB_per_launch": round(by / n / 1e6, 3),
                     "achieved_GBs": round(gbs, 1), "frac": round(gbs / hbm, 4)}
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1702_06735_b200 import binding

    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if world > 1 or (args.sharded and "RANK" in os.environ):
        return run_sharded(args)
    device = f"cuda:{local}"
    torch.cuda.set_device(device)
    binding.load_library()          # fails loudly if the CUDA extension is missing: there is no fallback

    cfg = W.config(3)
    mdl = cfg.model
    N, Nn, KC = cfg.n_data, cfg.n_norm, mdl.n_couplings
    # tddp4_create specialises the two fused passes to the model and compiles them with NVRTC: first handle
    # of the process (opens NVRTC, compiles), second handle of the same model (per-process cache)
    torch.zeros(1, device=device)
    jit = {}
    for key in ("create_first_s", "create_cached_s"):
        t0 = time.perf_counter()
        binding.Tddp4(mdl, device).close()
        jit[key] = round(time.perf_counter() - t0, 4)
    p4, t, p4n, ginfo = build_workload(binding, cfg, device, W.BASE_SEED + rank)
    p0 = W.initial_params(mdl)
    traj = W.trajectory(mdl, p0, args.warmup + args.steps, TRAJECTORY)

    stream = torch.cuda.Stream(device)
    h = binding.Tddp4(mdl, device)
    h.set_stream(stream)
    h.load_events(0, p4, t)
    h.load_events(1, p4n)
    packed = h.pack_params(traj)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-timed region (headline): K steps enqueued back to back through tddp4_nll_batch, no per-kernel events ------
    h.set_params(p0)
    h.nll()
    h.nll_batch(packed[:args.warmup])
    launches0 = h.launch_count()
    sampler = ClockSampler(local)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    ev0.record(stream)
    nll_vals, _ = h.nll_batch(packed[args.warmup:])
    ev1.record(stream)
    barrier()
    clocks = sampler.summary()
    ms = ev0.elapsed_time(ev1)
    launches = h.launch_count() - launches0
    if world > 1:
        tms = torch.tensor([ms], device=device, dtype=torch.float64)
        dist.all_reduce(tms, op=dist.ReduceOp.MAX)
        ms = float(tms.item())
    value = world * N * args.steps / (ms * 1e-3)

    # ---- the same K steps again with CUDA events around every kernel (tddp4_profile): per-kernel durations for the
    #      roofline.  The events serialise consecutive kernels (no programmatic overlap), so this pass is slower. ------
    h.set_params(p0)
    h.nll_batch(packed[:args.warmup])
    h.profile(True)
    h.profile_reset()
    torch.cuda.synchronize()
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2.record(stream)
    nll_prof, _ = h.nll_batch(packed[args.warmup:])
    ev3.record(stream)
    torch.cuda.synchronize()
    ms_prof = ev2.elapsed_time(ev3)
    prof = h.profile_read()
    in_us, in_n = h.profile_in_kernel()      # the coupling-only kernel on the GPU's own clock (earliest block start -> result written)
    h.profile(False)
    assert np.array_equal(nll_prof, nll_vals), "profiled and unprofiled passes differ"

    # ---- sub-cases reported next to the mixture ---------------------------------------------
    sub = {}
    for kind in ("coupling_only", "all"):
        tr = h.pack_params(W.trajectory(mdl, p0, args.warmup + args.steps, kind))
        h.set_params(p0)
        h.nll_batch(tr[:args.warmup])
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        h.nll_batch(tr[args.warmup:])
        b.record(stream)
        torch.cuda.synchronize()
        m = a.elapsed_time(b)
        sub[kind] = {"ms_per_step": round(m / args.steps, 5), "value": N * args.steps / (m * 1e-3)}
        if kind == "coupling_only":     # one NLL kernel per step, launches overlapped: the steady-state stream rate
            gbs = N * (16.0 * KC + 8.0) * args.steps / (m * 1e-3) / 1e9
            sub[kind].update({"alg_MB_per_step": N * (16.0 * KC + 8.0) / 1e6, "achieved_GBs": round(gbs, 1),
                              "frac": round(gbs / peaks()[0], 4)})

    # ---- the synchronous coupling-only call, the quantity a sequential minimiser sees:
    #      tddp4_set_params + tddp4_nll round trips on the host clock, one at a time -------------------------------------
    ctraj = W.trajectory(mdl, p0, 220, "coupling_only")
    for par in ctraj[:20]:
        h.set_params(par); h.nll()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for par in ctraj[20:]:
        h.set_params(par); h.nll()
    sync_us = (time.perf_counter() - t0) / 200 * 1e6
    sub["coupling_only"]["sync_us_per_call"] = round(sync_us, 2)
    sub["coupling_only"]["note"] = ("ms_per_step: calls enqueued back to back (tddp4_nll_batch), consecutive kernels overlap head to "
                                    "tail and part of the 136 MB stream is still in the 126 MB L2, hence above the HBM peak; "
                                    "sync_us_per_call: one tddp4_set_params + tddp4_nll round trip at a time on the host clock "
                                    "(launch + kernel + polled result)")

    # ---- end to end through the C-ABI with HOST buffers: load both samples from pinned host memory, then K
    #      synchronous tddp4_set_params + tddp4_nll calls, all inside the timed region ------------------------
    host = [torch.empty(x.shape, dtype=torch.float64, pin_memory=True).copy_(x) for x in (p4, t, p4n)]
    hp4, ht, hp4n = [x.numpy() for x in host]
    torch.cuda.synchronize()
    h2 = binding.Tddp4(mdl, device)
    h2.load_events(0, hp4, ht)                 # untimed warm-up of the whole end-to-end path (allocations, first H2D copies)
    h2.load_events(1, hp4n)
    for par in traj[:args.warmup]:
        h2.set_params(par)
        h2.nll()
    barrier()
    t0 = time.perf_counter()
    h2.load_events(0, hp4, ht)
    h2.load_events(1, hp4n)
    t_load = time.perf_counter() - t0
    e2e_vals = []
    for par in traj[args.warmup:]:
        h2.set_params(par)
        e2e_vals.append(h2.nll())
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    if world > 1:
        tt = torch.tensor([t_e2e], device=device, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_e2e = float(tt.item())
    assert np.array_equal(np.asarray(e2e_vals), nll_vals), "batched and synchronous evaluations differ"
    load_bytes = hp4.nbytes + ht.nbytes + hp4n.nbytes
    e2e = {"value": world * N * args.steps / t_e2e, "unit": UNIT,
           "h2d_bytes_per_step": load_bytes / args.steps + h2.h2d_bytes_per_call, "d2h_bytes_per_step": 64,
           "load_events_ms": round(1e3 * t_load, 3), "ms_per_step_after_load": round(1e3 * (t_e2e - t_load) / args.steps, 5),
           "note": "timed region = tddp4_load_events of both samples from pinned host memory (648 MB over PCIe, one-time, "
                   "amortised over the K steps: at small K it dominates -- load_events_ms against K x ms_per_step_after_load) "
                   "+ K synchronous tddp4_set_params/tddp4_nll calls"}
    h2.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    total_kernel_ms = sum(v[0] for v in prof.values())
    ktab = kernel_table(prof, total_kernel_ms)
    dominant = max(ktab, key=lambda k: ktab[k]["ms"])
    hbm, which = peaks()
    roof = {"kernel": dominant, "bound": "hbm", "achieved": ktab[dominant]["achieved_GBs"], "peak": hbm, "unit": "GB/s",
            "frac": ktab[dominant]["frac"], "peak_source": which, "traffic": None,
            "alg_bytes_per_launch": ktab[dominant]["alg_MB_per_launch"] * 1e6, "us_per_launch": ktab[dominant]["us_per_launch"]}
    # dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture of the SAME sources
    # (ncu cannot run inside this timed program); dropped, with the reason, when the sources have changed since
    tr, tr_src = committed_table("traffic.csv")
    roof["traffic"] = float(tr[dominant]["dram_bytes_per_launch"]) if dominant in tr else None
    roof["traffic_source"] = tr_src
    for k in ktab:
        ktab[k]["traffic"] = float(tr[k]["dram_bytes_per_launch"]) if k in tr else None
        ktab[k]["frac_of_8TBs_nominal"] = round(ktab[k]["achieved_GBs"] / 8000.0, 4)
        if k in tr and tr[k].get("ncu_us_per_launch"):
            # context, not a bench value: the same kernel's gpu__time_duration in the committed ncu capture (one cold launch, no
            # launch gap between CUDA events).  For the data pass the captured launch rewrote one column, not the mixture's mean.
            ktab[k]["ncu_us_per_launch_committed"] = float(tr[k]["ncu_us_per_launch"])

    if "nll" in ktab and in_n:
        us = in_us / in_n
        ktab["nll"].update({"in_kernel_us_per_launch": round(us, 2), "in_kernel_launches": in_n,
                            "in_kernel_GBs": round(N * (16.0 * KC + 8.0) / (us * 1e-6) / 1e9, 1),
                            "in_kernel_frac": round(N * (16.0 * KC + 8.0) / (us * 1e-6) / 1e9 / hbm, 4),
                            "in_kernel_frac_of_8TBs_nominal": round(N * (16.0 * KC + 8.0) / (us * 1e-6) / 1e9 / 8000.0, 4),
                            "in_kernel_note": "%globaltimer from the earliest block start to the result written, same launches as "
                                              "us_per_launch: the CUDA-event figure also contains the launch gap of an isolated launch"})

    # ---- what a pair of CUDA events costs around a kernel that does nothing (a one-element torch add on the same stream):
    #      the floor under every per-launch figure of `kernels`, and under any "isolated call" figure on this machine ----
    try:
        tiny = torch.zeros(32, device=device)
        floor = {}
        with torch.cuda.stream(stream):
            for key, sync_each in (("back_to_back", False), ("after_host_sync", True)):
                pairs = []
                for k in range(120):
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream); tiny.add_(1.0); b.record(stream)
                    if sync_each:
                        stream.synchronize()
                    if k >= 20:
                        pairs.append((a, b))
                stream.synchronize()
                floor[key] = round(1e3 * sum(a.elapsed_time(b) for a, b in pairs) / len(pairs), 2)
        floor["note"] = ("us between two CUDA events around a one-element kernel: launch + completion latency that every "
                         "event-bracketed launch above contains; tddp4_profile_in_kernel (kernels.nll.in_kernel_*) excludes it")
        roof["event_floor_us"] = floor
    except Exception as e:
        roof["event_floor_us"] = {"error": repr(e)}

    # ---- the dominant kernel on its own, and the step as a whole.  Inside the mixture the CUDA events around a Gram launch
    #      also see the write-back of the column lines the preceding data pass left dirty in L2 (its 16 B per stale column are
    #      stored into L2 and reach DRAM while the NEXT kernel streams: DESIGN.md 7); `alone` times the same kernel in a loop
    #      of tddp4_set_params (one mass moved) + tddp4_gram, where no such lines exist, and `whole_step` divides the
    #      algorithmic bytes of ALL launches of the timed region by its duration (no per-kernel events) ---------------------
    try:
        h.profile(True)
        for k in range(30):
            if k == 5:
                h.profile_reset()
            q = p0.copy()
            q.mass[0] *= 1.0 + 1e-6 * (k + 1)
            h.set_params(q)
            h.gram()
        gms, gn, gby = h.profile_read()["gram"]
        h.profile(False)
        h.set_params(p0)
        a_gbs = gby / (gms * 1e-3) / 1e9
        roof["alone"] = {"us_per_launch": round(1e3 * gms / gn, 3), "launches": gn, "achieved": round(a_gbs, 1),
                         "frac": round(a_gbs / hbm, 4)}
        step_bytes = sum(v[2] for v in prof.values()) / args.steps
        s_gbs = step_bytes / (ms / args.steps * 1e-3) / 1e9
        roof["whole_step"] = {"alg_MB_per_step": round(step_bytes / 1e6, 1), "achieved": round(s_gbs, 1), "frac": round(s_gbs / hbm, 4),
                              "note": "algorithmic bytes of every launch of the timed region / its duration / peak"}
    except Exception as e:
        roof["alone"] = {"error": repr(e)}

    # ---- analytic gradient: one pass against the 2 (4 K_c + 2) NLL calls of a numerical gradient ----
    grad = {}
    try:
        h.set_params(p0)
        h.nll_grad()
        h.profile(True)
        h.profile_reset()
        for _ in range(20):
            h.nll_grad()
        gms, gn, gby = h.profile_read()["nll_grad"]
        gin_us, gin_n = h.profile_in_kernel_of(binding.K_GRAD)   # earliest block start -> gradient written, same launches
        h.profile(False)
        grad = {"us_per_call": round(1e3 * gms / gn, 3), "alg_MB_per_call": gby / gn / 1e6,
                "frac": round(gby / (gms * 1e-3) / 1e9 / peaks()[0], 4), "n_derivatives": 4 * KC + 2,
                "in_kernel_us_per_call": round(gin_us / gin_n, 2) if gin_n else None,
                "in_kernel_frac": round(gby / gn / (gin_us / gin_n * 1e-6) / 1e9 / peaks()[0], 4) if gin_n else None,
                "numerical_gradient_us": round(2 * (4 * KC + 2) * 1e3 * sub["coupling_only"]["ms_per_step"], 1)}
    except Exception as e:
        grad = {"error": repr(e)}
    # ---- incremental Gram update, measured on the same trajectory: the normalisation columns are
    #      kept (512 MB for C3) and a step that dirtied few columns rebuilds only those ------------------------------------
    inc = {}
    try:
        h.set_gram_mode(1)
        h.set_params(p0)
        h.nll_batch(packed[:args.warmup])
        n0 = h.set_gram_mode(-1)
        h.profile(True); h.profile_reset()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        nll_inc, _ = h.nll_batch(packed[args.warmup:])
        b.record(stream)
        torch.cuda.synchronize()
        m_ev = a.elapsed_time(b)
        pg = h.profile_read()["gram"]
        h.profile(False)
        n_inc = h.set_gram_mode(-1) - n0
        # the same pass without per-kernel events (as the headline)
        h.set_params(p0)
        h.nll_batch(packed[:args.warmup])
        torch.cuda.synchronize()
        a.record(stream)
        h.nll_batch(packed[args.warmup:])
        b.record(stream)
        torch.cuda.synchronize()
        inc = {"ms_per_step": round(a.elapsed_time(b) / args.steps, 5), "ms_per_step_full_passes": round(ms / args.steps, 5),
               "ms_per_step_with_kernel_events": round(m_ev / args.steps, 5),
               "gram_launches": pg[1], "incremental_passes": n_inc,
               "gram_us_per_launch": round(1e3 * pg[0] / max(1, pg[1]), 2), "gram_alg_MB_per_launch": round(pg[2] / max(1, pg[1]) / 1e6, 1),
               "stored_columns_MB": round(16.0 * KC * Nn / 1e6, 1), "bit_identical_nll": bool(np.array_equal(nll_inc, nll_vals))}
        # where it pays: a trajectory of one-column moves (mass or width of a1, K1(1270), K2*, K1(1400), each in ONE column)
        one = h.pack_params(W.trajectory(mdl, p0, args.warmup + 200, "one_resonance", resonances=[2, 3, 4, 5]))
        for mode, key in ((1, "ms_per_step"), (0, "ms_per_step_full_passes")):
            h.set_gram_mode(mode)
            h.set_params(p0)
            h.nll_batch(one[:args.warmup])
            torch.cuda.synchronize()
            a.record(stream)
            v, _ = h.nll_batch(one[args.warmup:])
            b.record(stream)
            torch.cuda.synchronize()
            inc.setdefault("one_column_moves", {"steps": 200})[key] = round(a.elapsed_time(b) / 200, 5)
            inc["one_column_moves"].setdefault("nll", []).append(float(v[-1]))
        nl = inc["one_column_moves"].pop("nll")
        inc["one_column_moves"]["bit_identical_nll"] = nl[0] == nl[1]
        h.set_gram_mode(0)
    except Exception as e:
        inc = {"error": repr(e)}
    cpu = cpu_baseline(mdl, p0, ginfo) if world == 1 else None      # the oracle is timed at N = 1 only
    fp64_peak = h.fp64_peak()
    h.close()
    others = other_configs(binding, device) if not args.headline_only else {}
    extras = {}
    if not args.headline_only:
        for key, fn in (("alu", lambda: alu_fractions(binding, device, fp64_peak)),
                        ("cpu_baseline_generate", cpu_baseline_generate),
                        ("validation_projections", lambda: validation_projections(binding, device, args.validation_events)),
                        ("table1_like", lambda: table1_like(binding, device))):
            try:
                extras[key] = fn()
            except Exception as e:                           # never lose the headline line over an extra
                extras[key] = {"error": repr(e)}
    try:      # the resolution time rows (config 5) against the same fp64 peak
        tr5 = others["C5"]["kernels"]["time_rows"]
        counts, _ = committed_table("alu_counts.csv")
        per = float(counts["time_rows"]["fp64_warp_inst_per_unit"])
        tr5.update({"bound": "alu", "fp64_warp_inst_per_unit": per,
                    "frac_fp64_peak": round(per * W.config(5).n_data / (tr5["us_per_launch"] * 1e-6) / (fp64_peak / 32.0), 4)})
    except Exception:
        pass
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "n_data": N, "n_norm": Nn, "n_terms": mdl.n_terms, "n_couplings": KC,
                       "trajectory": TRAJECTORY + " (p=0.8 one of 46 floating parameters moves, p=0.2 all move)",
                       "l2": "inputs larger than L2: a coupling-only step streams 136 MB, a dirty step 1.5+ GB; no flush",
                       "generation": {"data_candidates": ginfo["n_candidates"], "envelope": ginfo["envelope"]}},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "kernels": ktab,
            "ms_per_step_with_kernel_events": ms_prof / args.steps,
            "coupling_only": sub["coupling_only"], "all_dirty": sub["all"], "cpu_baseline": cpu,
            "nll_first_last": [float(nll_vals[0]), float(nll_vals[-1])], "gradient": grad, "other_configs": others,
            "fp64_peak_inst_per_s": fp64_peak, "jit": jit, "incremental_gram": inc, **extras}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def other_configs(binding, device, steps_c5=100):
    """The other BASELINE.json workloads next to the headline: C2 as calls/s (L2-resident), C4 as generated
    candidates/s and accepted events/s, C5 (per-event resolution, efficiency weights) as events x evals/s.  Reported keys
    only; the headline `value` is C3's."""
    import torch
    out = {}
    try:
        # ---- C4: 10 M Raubold-Lynch candidates, pilot 100 000, envelope x1.2, config-1 rate, compacted output ----------
        cfg = W.config(4)
        h = binding.Tddp4(cfg.model, device)
        h.set_params(W.initial_params(cfg.model))
        n = cfg.n_candidates
        h.generate(W.BASE_SEED, W.STREAM_DATA, 0, n // 10, cfg.n_pilot, cfg.envelope_scale, n // 40)      # warm-up
        best, g = float("inf"), None
        for _ in range(3):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            g = h.generate(W.BASE_SEED, W.STREAM_DATA, 0, n, cfg.n_pilot, cfg.envelope_scale, n // 4)
            torch.cuda.synchronize()
            best = min(best, time.perf_counter() - t0)
        out["C4"] = {"candidates": n, "accepted": g["n_accepted"], "overflow": g["n_overflow"], "ms": round(1e3 * best, 3),
                     "candidates_per_s": n / best, "accepted_per_s": g["n_accepted"] / best,
                     "note": "tddp4_generate end to end (pilot pass + ratio pass + scan + emit, host-synchronous), best of 3"}
        h.close()
        # ---- C2: 50 000 + 500 000 events, 8 terms, ~300 calls, couplings/x/y float ---------------------------------------
        for name, idx in (("C2", 2),):
            cfg = W.config(idx)
            p4, t, p4n, _ = build_workload(binding, cfg, device, W.BASE_SEED)
            h = binding.Tddp4(cfg.model, device)
            h.load_events(0, p4, t)
            h.load_events(1, p4n)
            p0 = W.initial_params(cfg.model)
            tr = h.pack_params(W.trajectory(cfg.model, p0, cfg.n_calls + 10, cfg.trajectory))
            h.set_params(p0)
            h.nll_batch(tr[:10])
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            h.nll_batch(tr[10:])
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            out[name] = {"calls": cfg.n_calls, "calls_per_s": cfg.n_calls / dt, "value": cfg.n_data * cfg.n_calls / dt,
                         "unit": UNIT, "us_per_call": round(1e6 * dt / cfg.n_calls, 3),
                         "note": "working set 6.8 MB per call: L2-resident, launch-latency bound"}
            h.close()
        # ---- the shape of the paper's Table 3: fit to 100 000 pseudo-events, model fixed, x and y floating, against
        #      the number of normalisation points (0.75 M .. 6 M); the config-2 model stands in for the paper's unpublished one.
        #      Context only: K40 0.6 / 1.0 / 1.7 / 3.2 s, 2 x Xeon (48 threads) 3.3 / 6.5 / 12.4 / 22.5 s.  -------------------------
        from paper_1702_06735_b200 import fit as F
        cfg = W.config(2)
        flat = W.flat_model()
        hf = binding.Tddp4(flat, device)
        hf.set_params(W.flat_params(flat))
        p4n6, _, _, _ = hf.generate_n(W.BASE_SEED, W.STREAM_NORM, 6_000_000, 0, 2.0 * hf.weight_bound(), chunk=1 << 24)
        hf.close()
        hg = binding.Tddp4(cfg.model, device)
        p0 = W.initial_params(cfg.model)
        hg.set_params(p0)
        p4d, td, _, _ = hg.generate_n(W.BASE_SEED, W.STREAM_DATA, 100_000, cfg.n_pilot, cfg.envelope_scale, chunk=1 << 23)
        hg.close()
        rows = []
        for n_norm in (750_000, 1_500_000, 3_000_000, 6_000_000):
            h = binding.Tddp4(cfg.model, device)
            h.load_events(0, p4d, td)
            h.load_events(1, p4n6[:, :n_norm].contiguous())
            start = p0.copy()
            start.x, start.y = 0.0, 0.0
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            res = F.fit(h, start, free_couplings=None, free_xy=True)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            rows.append({"n_norm": n_norm, "fit_s": round(dt, 5), "nll_grad_calls": res.n_calls, "converged": res.success,
                         "x": res.par.x, "y": res.par.y, "sigma_x": res.errors.get("x"), "sigma_y": res.errors.get("y")})
            h.close()
        out["table3_like"] = {"n_data": 100_000, "floating": ["x", "y"], "rows": rows,
                              "note": "fit wall time incl. the first call's column and Gram build and the Hessian; the "
                                      "normalisation enters only through the cached Gram matrix, so the time does not grow "
                                      "with n_norm beyond that one pass"}
        del p4n6
        # ---- C5: 10 M + 10 M events, per-event sigma_t, efficiency weights, minuit trajectory ----------------------------
        cfg = W.config(5)
        p4, t_true, p4n, _ = build_workload(binding, cfg, device, W.BASE_SEED)
        t_obs, sig = W.smear_times(t_true.cpu().numpy(), cfg)
        w = W.efficiency_weights(cfg.n_norm, cfg)
        dev = lambda a: torch.from_numpy(a).to(device)
        h = binding.Tddp4(cfg.model, device)
        h.load_events(0, p4, dev(t_obs), sigma_t=dev(sig))
        h.load_events(1, p4n, None, weight=dev(w))
        del p4, p4n
        p0 = W.initial_params(cfg.model)
        tr = h.pack_params(W.trajectory(cfg.model, p0, steps_c5 + 5, cfg.trajectory))
        h.set_params(p0)
        h.nll_batch(tr[:5])
        h.profile(True)
        h.profile_reset()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        vals, _ = h.nll_batch(tr[5:])
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        prof = h.profile_read()
        hbm, _ = peaks()
        kt = {k: {"launches": v[1], "us_per_launch": round(1e3 * v[0] / v[1], 2), "alg_MB_per_launch": round(v[2] / v[1] / 1e6, 1),
                  "frac_hbm": round(v[2] / (v[0] * 1e-3) / 1e9 / hbm, 4)} for k, v in prof.items() if v[1]}
        if "nll" in kt:      # SURVEY.md 8(d) counts 16 K_c + 16 = 144 B/event for this pass (t and sigma_t); the design streams
            # 16 K_c + 64 = 192 B/event (eight cached time rows instead of recomputing three convolutions per event)
            kt["nll"]["frac_hbm_at_144B_per_event"] = round(cfg.n_data * 144.0 / (kt["nll"]["us_per_launch"] * 1e-6) / 1e9 / hbm, 4)
            kt["nll"]["bytes_per_event_streamed"] = 192
        out["C5"] = {"calls": steps_c5, "ms_per_call": round(1e3 * dt / steps_c5, 4), "value": cfg.n_data * steps_c5 / dt,
                     "unit": UNIT, "kernels": kt, "nll_last": float(vals[-1]),
                     "note": "resolution mode: the NLL pass streams 16 K_c + 64 B per event (cached time rows), time rows are "
                             "rebuilt when x, y or tau move (ALU-bound)"}
        h.close()
    except Exception as e:                                   # never lose the headline line over an extra
        out["error"] = repr(e)
    return out


def alu_fractions(binding, device, fp64_peak):
    """The fp64-ALU-bound kernels (generator ratio pass, kinematics at load, resolution time rows) against the MEASURED fp64
    issue rate of this GPU (tddp4_fp64_peak: a dependent-free DFMA chain on every SM).  Achieved = fp64 warp instructions
    per launch -- counted by ncu (sm__inst_executed_pipe_fp64.sum) on the same sources, committed in
    profiles/alu_counts.csv as instructions per candidate / event -- divided by the CUDA-event duration measured here."""
    import torch
    counts, src = committed_table("alu_counts.csv")
    out = {"fp64_peak_inst_per_s": fp64_peak, "fp64_peak_warp_inst_per_s": fp64_peak / 32.0, "counts_source": src,
           "peak_source": "measured here (tddp4_fp64_peak)", "kernels": {}}

    def entry(name, units, ms):
        e = {"units": units, "us_per_launch": round(1e3 * ms, 2)}
        if name in counts:
            per_unit = float(counts[name]["fp64_warp_inst_per_unit"])
            e.update({"fp64_warp_inst_per_unit": per_unit, "bound": "alu",
                      "achieved_warp_inst_per_s": per_unit * units / (ms * 1e-3),
                      "frac": round(per_unit * units / (ms * 1e-3) / (fp64_peak / 32.0), 4)})
        out["kernels"][name] = e

    cfg = W.config(4)
    h = binding.Tddp4(cfg.model, device)
    h.set_params(W.initial_params(cfg.model))
    n = cfg.n_candidates
    g = h.generate(W.BASE_SEED, W.STREAM_DATA, 0, n, cfg.n_pilot, cfg.envelope_scale, n // 4)
    h.profile(True); h.profile_reset()
    h.generate(W.BASE_SEED, W.STREAM_DATA, 0, n, 0, g["envelope"], n // 4)     # envelope given: exactly one ratio launch
    pr = h.profile_read(); h.profile(False)
    entry("gen_ratio", n, pr["gen_ratio"][0] / max(1, pr["gen_ratio"][1]))
    h.close()
    cfg = W.config(3)
    p4, t, _, _ = build_data_only(binding, cfg, device)
    h = binding.Tddp4(cfg.model, device)
    h.load_events(0, p4, t)
    h.profile(True); h.profile_reset()
    h.load_events(0, p4, t)
    pr = h.profile_read(); h.profile(False)
    entry("kin", cfg.n_data, pr["kin"][0] / max(1, pr["kin"][1]))
    h.close()
    return out


def table1_like(binding, device):
    """The shape of the paper's Table 1: sigma(x), sigma(y) from toy ensembles at 20 000 / 50 000 /
    70 000 events, model fixed, x = 0.49 %, y = 0.61 %.  Context, not a target: the paper's model is unpublished (the
    config-2 model stands in), its numbers were 0.030/0.031, 0.019/0.019, 0.016/0.017 %."""
    from paper_1702_06735_b200 import fit as F
    mdl = W.config(2).model
    flat = W.flat_model()
    t0 = time.perf_counter()
    rows = F.sensitivity_study(binding, mdl, W.initial_params(mdl), sizes=(20_000, 50_000, 70_000), n_toys=50, n_norm=1_000_000,
                               device=device, flat_model=flat, flat_par=W.flat_params(flat))
    for r in rows:
        r["sigma_x_times_sqrtN"] = r["sigma_x_hesse"] * r["n_events"] ** 0.5
        r["sigma_y_times_sqrtN"] = r["sigma_y_hesse"] * r["n_events"] ** 0.5
    return {"rows": rows, "wall_s": round(time.perf_counter() - t0, 2), "paper_table1_percent": {"20000": [0.030, 0.031], "50000": [0.019, 0.019],
                                                                                               "70000": [0.016, 0.017]},
            "note": "150 toy fits (generate + load + BFGS with the analytic gradient + Hessian) in wall_s"}


def build_data_only(binding, cfg, device):
    hg = binding.Tddp4(cfg.model, device)
    hg.set_params(W.initial_params(cfg.model))
    p4, t, idx, info = hg.generate_n(W.BASE_SEED, W.STREAM_DATA, cfg.n_data, cfg.n_pilot, cfg.envelope_scale, chunk=1 << 24)
    hg.close()
    return p4, t, idx, info


def cpu_baseline_generate(n_candidates=10_000_000):
    """The oracle's generator (Philox + Raubold-Lynch + rate + accept-reject, one candidate at a time, OpenMP over
    candidates) on config 4 as it stands: 10 M candidates, pilot 100 000 (under a second on the box's host cores)."""
    import oracle
    cfg = W.config(4)
    par = W.initial_params(cfg.model)
    t0 = time.perf_counter()
    g = oracle.generate(cfg.model, par, W.BASE_SEED, W.STREAM_DATA, n_candidates, cfg.n_pilot, cfg.envelope_scale, n_candidates // 4)
    dt = time.perf_counter() - t0
    return {"value": n_candidates / dt, "unit": "candidates/s", "accepted_per_s": g["n_accepted"] / dt, "cores": oracle.threads(),
            "kind": "oracle", "sample": f"all {n_candidates} candidates of config 4 (+ its 100 000-candidate pilot), one oracle.generate "
                                        f"call ({dt:.2f} s)"}


def validation_projections(binding, device, n_events):
    """The paper's validation (Fig. 3): a pseudo-event sample of the model generated on the GPU against
    an independent one from the other implementation -- here the oracle's generator with another seed, standing in for
    MINT3 -- compared in the five projections m12, m34, cos12, cos34, phi: pulls, chi2/ndf and p-value per projection.
    The GPU sample is histogrammed by tddp4_project, the oracle's by oracle/projections.py.  The config-2 model stands in
    for the paper's unpublished one; the paper used 500 000 events (--validation-events)."""
    import oracle
    from oracle import projections as OP
    from scipy import stats
    mdl = W.config(2).model
    par = W.initial_params(mdl)
    n_bins = 50
    rng = OP.default_ranges(mdl.m_parent, mdl.m_final)
    h = binding.Tddp4(mdl, device)
    h.set_params(par)
    t0 = time.perf_counter()
    p4, _, _, info = h.generate_n(W.BASE_SEED, W.STREAM_DATA, n_events, 100_000, 1.2, chunk=1 << 24)
    hist_gpu, _ = h.project(p4, n_bins, rng)
    t_gpu = time.perf_counter() - t0
    h.close()
    t0 = time.perf_counter()
    n_cand = int(n_events / 0.0085) + 200_000
    while True:
        g = oracle.generate(mdl, par, W.BASE_SEED + 1000, W.STREAM_DATA, n_cand, 100_000, 1.2, n_events)
        if g["n_accepted"] >= n_events:
            break
        n_cand = int(n_cand * 1.5)
    hist_orc = OP.histograms(g["p4"][:, :n_events], n_bins, rng)
    t_orc = time.perf_counter() - t0
    out = {"n_events": n_events, "n_bins": n_bins, "gpu_generate_and_project_s": round(t_gpu, 4), "oracle_generate_and_project_s": round(t_orc, 2),
           "projections": {}}
    for k, name in enumerate(OP.NAMES):
        a, b = hist_gpu[k].astype(float), hist_orc[k].astype(float)
        use = a + b >= 20
        pulls = (a[use] - b[use]) / np.sqrt(a[use] + b[use])
        chi2, ndf = float(np.sum(pulls ** 2)), int(use.sum()) - 1
        out["projections"][name] = {"chi2": round(chi2, 2), "ndf": ndf, "p_value": float(stats.chi2.sf(chi2, ndf)),
                                    "pull_mean": round(float(pulls.mean()), 3), "pull_rms": round(float(pulls.std(ddof=1)), 3),
                                    "frac_within_2_sigma": round(float(np.mean(np.abs(pulls) < 2.0)), 3)}
    return out


def run_sharded(args):
    """N > 1, launched by torch.distributed.run (one process per GPU): the event-sharded evaluation of SURVEY.md 8(e).
    Weak scaling is the headline: every rank holds its own C3-sized shard (1 M data + 4 M normalisation events, own
    Philox seed) of ONE global sample of N x (1 M + 4 M) events, evaluated through sharded.ShardedNLL -- per call one
    all-gather of the Gram sums when a mass or width moved and one all-gather of 8 result words, NCCL on the handle's
    stream.  Strong scaling (the one C3 sample of rank 0's seed split N ways) is reported next to it."""
    import torch
    import torch.distributed as dist
    from paper_1702_06735_b200 import binding, sharded
    rank, world, local = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"]), int(os.environ.get("LOCAL_RANK", 0))
    device = f"cuda:{local}"
    torch.cuda.set_device(device)
    dist.init_process_group("nccl", device_id=torch.device(device))
    binding.load_library()
    cfg = W.config(3)
    mdl = cfg.model
    N, KC = cfg.n_data, mdl.n_couplings
    p0 = W.initial_params(mdl)
    traj = W.trajectory(mdl, p0, args.warmup + args.steps, TRAJECTORY)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    def timed(shnll, stream, pars):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        a.record(stream)
        vals = []
        for par in pars:
            shnll.set_params(par)
            vals.append(shnll.nll())
        b.record(stream)
        barrier()
        ms = torch.tensor([a.elapsed_time(b)], device=device, dtype=torch.float64)
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item()), vals

    results = {}
    sampler = None
    for mode in ("weak", "strong"):
        if mode == "weak":
            p4, t, p4n, _ = build_workload(binding, cfg, device, W.BASE_SEED + rank)
        else:
            p4, t, p4n, _ = build_workload(binding, cfg, device, W.BASE_SEED)
            lo, hi = sharded.shard_range(cfg.n_data, rank, world)
            ln, hn = sharded.shard_range(cfg.n_norm, rank, world)
            p4, t, p4n = p4[:, lo:hi].contiguous(), t[lo:hi].contiguous(), p4n[:, ln:hn].contiguous()
        stream = torch.cuda.Stream(device)
        h = binding.Tddp4(mdl, device)
        h.set_stream(stream)
        sh = sharded.ShardedNLL(h, always_collective=args.sharded)
        sh.load_events(0, p4, t)
        sh.load_events(1, p4n)
        timed(sh, stream, traj[:args.warmup])
        launches0, ex0 = h.launch_count(), sh.exchanges
        if mode == "weak":
            sampler = ClockSampler(local)
            sampler.start()
        ms, vals = timed(sh, stream, traj[args.warmup:])
        clocks = sampler.summary() if mode == "weak" else None
        events = N * world if mode == "weak" else N
        results[mode] = {"ms_per_step": ms / args.steps, "value": events * args.steps / (ms * 1e-3), "events_per_call": events,
                         "gpu_launches": h.launch_count() - launches0, "collectives": sh.exchanges - ex0,
                         "nll_first_last": [vals[0], vals[-1]]}
        if mode == "weak":
            results[mode]["clocks"] = clocks
        h.close()
        del p4, t, p4n
    if rank == 0:
        wk = results["weak"]
        line = {"metric": METRIC, "value": wk["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": wk["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic",
                "config": {"workload": WORKLOAD + " sharded", "n_data_per_gpu": N, "n_norm_per_gpu": cfg.n_norm, "n_terms": mdl.n_terms,
                           "n_couplings": KC, "trajectory": TRAJECTORY, "parallelism": f"event shards x{world}",
                           "exchange": "all-gather of 2 K_c^2 + 1 doubles per mass/width move and of 8 doubles per call (NCCL, on "
                                       "the handle's stream), rank-ordered sums",
                           "l2": "inputs larger than L2: a coupling-only step streams 136 MB per GPU, a dirty step 1.5+ GB; no flush"},
                "clocks": wk["clocks"], "gpu_launches": wk["gpu_launches"], "collectives_per_run": wk["collectives"],
                "e2e": {"value": wk["value"], "unit": UNIT, "h2d_bytes_per_step": 8.0 * (4 * KC + 2 * mdl.n_res + 3),
                        "d2h_bytes_per_step": 64.0 * world,
                        "note": "the sharded path IS the synchronous public API: every step sends its parameters from the host and "
                                "reads the gathered result words back; events are resident (loaded once, untimed)"},
                "roofline": None, "cpu_baseline": None, "strong_scaling": results["strong"], "nll_first_last": wk["nll_first_last"]}
        print(json.dumps(line))
    dist.destroy_process_group()


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` without a launcher: start N ranks on this node (127.0.0.1 rendezvous) and replace this
    process by the launcher."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def cpu_baseline(mdl, par, ginfo, n_data=100_000):
    """The oracle as it stands, timed on this box's host cores on a bounded sample of the same workload: the first events
    of both samples, which the oracle regenerates itself from their candidate indices (it is handed no CUDA output)."""
    import oracle
    n_norm = 4 * n_data
    flat = W.flat_model()
    a, b, _, _ = oracle.candidates_at(mdl, par.tau, ginfo["seed"], W.STREAM_DATA, ginfo["index"][:n_data].cpu().numpy())
    c, _, _, _ = oracle.candidates_at(flat, W.TAU_D0, ginfo["seed"], W.STREAM_NORM, ginfo["index_norm"][:n_norm].cpu().numpy())
    best = float("inf")
    for _ in range(3):
        t0 = time.perf_counter()
        oracle.nll(mdl, par, a, b, c, want_prob=False)
        best = min(best, time.perf_counter() - t0)
    return {"value": n_data / best, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle",
            "sample": f"first {n_data} data + {n_norm} normalisation events of the same samples, 1 full-recompute NLL "
                      f"evaluation, best of 3 ({best:.3f} s)"}


def run_reference(args):
    """`--impl reference`: the CPU oracle, as it stands, on this box's host cores; same metric, config and trajectory.
    Each step is one full-recompute NLL evaluation on a bounded sample of the workload (same 1:4 data:normalisation
    ratio, same model), sized from a calibration call so that the W + K steps end within a few minutes.  No CUDA."""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    import oracle
    import math
    cfg = W.config(3)
    mdl = cfg.model
    p0 = W.initial_params(mdl)
    traj = W.trajectory(mdl, p0, args.warmup + args.steps, TRAJECTORY)
    flat, fpar = W.flat_model(), W.flat_params(W.flat_model())
    bound = math.prod(oracle.breakup(*tr) for tr in W.flat_envelope_inputs(flat))

    def sample(n_data):
        n_norm = 4 * n_data
        g = oracle.generate(flat, fpar, W.BASE_SEED, W.STREAM_NORM, int(n_norm / 0.06) + 5000, 0, 2.0 * bound, n_norm)
        assert g["n_accepted"] >= n_norm
        n_cand = 80 * n_data + 20000
        while True:
            d = oracle.generate(mdl, p0, W.BASE_SEED, W.STREAM_DATA, n_cand, min(cfg.n_pilot, n_cand // 4), cfg.envelope_scale, n_data)
            if d["n_accepted"] >= n_data:
                return d["p4"][:, :n_data].copy(), d["t"][:n_data].copy(), g["p4"][:, :n_norm].copy()
            n_cand *= 2

    p4, t, p4n = sample(2000)
    t0 = time.perf_counter()
    oracle.nll(mdl, p0, p4, t, p4n, want_prob=False)
    rate = 2000 / (time.perf_counter() - t0)                    # data events per second of one evaluation
    budget_s = 90.0
    n_data = int(max(500, min(50_000, rate * budget_s / (args.warmup + args.steps))))   # cap bounds the (untimed) generation
    if n_data != 2000:
        p4, t, p4n = sample(n_data)
    for par in traj[:args.warmup]:
        oracle.nll(mdl, par, p4, t, p4n, want_prob=False)
    t0 = time.perf_counter()
    vals = [oracle.nll(mdl, par, p4, t, p4n, want_prob=False)[0] for par in traj[args.warmup:]]
    dt = time.perf_counter() - t0
    value = n_data * args.steps / dt
    samp = (f"{n_data} data + {4 * n_data} normalisation events per step (oracle-generated with the workload's recipe), "
            f"{args.steps} full-recompute NLL evaluations along the same trajectory")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "n_data": cfg.n_data, "n_norm": cfg.n_norm, "n_terms": mdl.n_terms,
                       "n_couplings": mdl.n_couplings, "trajectory": TRAJECTORY, "sample": samp},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle", "sample": samp},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "nll_first_last": [vals[0], vals[-1]]}
    print(json.dumps(line))


def writeback_study(args):
    """DESIGN.md 7, "Where the Gram pass's time in the mixture goes": the Gram kernel's CUDA-event duration (tddp4_profile)
    after different predecessors on the stream.  Prints one JSON line; not part of the bench contract."""
    import torch
    from paper_1702_06735_b200 import binding
    device = "cuda:0"
    torch.cuda.set_device(device)
    binding.load_library()
    cfg = W.config(3)
    p4, t, p4n, _ = build_workload(binding, cfg, device, W.BASE_SEED)
    p0 = W.initial_params(cfg.model)
    h = binding.Tddp4(cfg.model, device)
    h.load_events(0, p4, t)
    h.load_events(1, p4n)
    del p4, p4n
    torch.cuda.empty_cache()
    other = torch.zeros(128 * 1024 * 1024, dtype=torch.float64, device=device)      # 1 GiB of memory the kernels never touch
    h.set_params(p0)
    h.nll()

    def moved(k):                       # one mass moved: Gram matrix and data columns stale
        q = p0.copy(); q.mass[0] *= 1.0 + 1e-6 * (k + 1); return q

    def coupling(k, j):                 # the same masses, one coupling moved: a coupling-only call
        q = moved(k); q.c[0] *= 1.0 + 1e-6 * (j + 1); return q

    def gram_only(k):
        h.set_params(moved(k)); h.gram()

    def dirty_step(k):
        h.set_params(moved(k)); h.nll()

    def dirty_then_coupling_only(k):
        dirty_step(k)
        for j in range(3):
            h.set_params(coupling(k, j)); h.nll()

    def dirty_then_read_elsewhere(k):
        dirty_step(k); other.sum().item()

    def dirty_then_write_elsewhere(k):
        dirty_step(k); other.zero_(); torch.cuda.synchronize()

    rows = []
    for name, body in (("GRAM -> GRAM (tddp4_gram after one mass moved)", gram_only),
                       ("GRAM -> COLNLL -> GRAM (dirty steps)", dirty_step),
                       ("GRAM -> COLNLL -> 3 x NLL -> GRAM", dirty_then_coupling_only),
                       ("GRAM -> COLNLL -> 1 GiB read of other memory -> GRAM", dirty_then_read_elsewhere),
                       ("GRAM -> COLNLL -> 1 GiB write of other memory -> GRAM", dirty_then_write_elsewhere)):
        for k in range(5):
            body(k)
        h.profile(True); h.profile_reset()
        for k in range(args.steps):
            body(k + 5)
        pr = h.profile_read()
        h.profile(False)
        rows.append({"sequence": name, **{n: round(1e3 * v[0] / v[1], 2) for n, v in pr.items() if v[1]}})
        gram_mb = pr["gram"][2] / pr["gram"][1] / 1e6
    h.close()
    print(json.dumps({"writeback_study": rows, "unit": "us per launch between CUDA events", "repetitions": args.steps,
                      "gram_alg_MB": gram_mb}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)     # BASELINE.json configs[2]: 1 000 consecutive evaluations
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--headline-only", action="store_true", help="skip the C2/C4/C5 extras (profiling runs)")
    ap.add_argument("--sharded", action="store_true",
                    help="run the event-sharded path (the N > 1 mode) even with one rank: a single-GPU check of that code path, "
                         "launched under torch.distributed.run --nproc-per-node 1")
    ap.add_argument("--validation-events", type=int, default=100_000,
                    help="events per sample of the Fig. 3 comparison (the paper: 500 000; the oracle generates ~0.9 %% of its candidates)")
    ap.add_argument("--writeback-study", action="store_true",
                    help="instead of the bench: the Gram kernel's duration after different predecessors (DESIGN.md 7); --steps = repetitions")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3 if args.impl == "ours" else 0)
    if args.writeback_study:
        args.steps = min(args.steps, 200)
        writeback_study(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
