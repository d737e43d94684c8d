#!/usr/bin/env python
"""bench.py -- simulated requests/s on the replica sweep (BASELINE.json configs[2])
and priority-select GB/s on config 5 (configs[4]), on N B200s of one node.

  python bench.py --gpus 1 --steps 5 --warmup 3
  python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
      --master-port P bench.py --gpus N --steps K --warmup W
  python bench.py --impl reference        # the CPU oracle, as it stands, on the host cores

One step = one pass of the whole hot path over one batch: a1 generate the
32,768 traces -> a4/a5 simulate 98,304 replicas (a2/a3 inside the admit step)
-> a6 per-replica p50/p90 + throughput inputs.  The standalone batched select
(config 5) is timed in its own region of the same run.  Rank r of an N-GPU run
takes seeds [r*4096, (r+1)*4096) and its own 65,536 queues: weak scaling, no
data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "simulated requests/sec (replica sweep)"
UNIT = "requests/s"
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback
# issue-slot peak: 148 SMs x 4 schedulers x 1 warp-instruction/clk x 1.965 GHz
ALU_PEAK_WARP_INSTR_PER_S = 148 * 4 * 1.965e9


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def csrc_sha16():
    """hash of the kernel sources the committed ncu constants were captured from"""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2603_11273_b200", "csrc", "*.cu*"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def load_profile_constants():
    """per-launch DRAM traffic and instructions per request, from the committed ncu summaries.  They are
    counters of a capture under ncu (never of this run): the file carries the hash of the kernel sources it
    was taken from, and a run on other sources marks every figure derived from it as stale."""
    p = os.path.join(ROOT, "profiles", "roofline_constants.json")
    if os.path.exists(p):
        try:
            c = json.load(open(p))
            c["stale"] = c.get("csrc_sha16") != csrc_sha16()
            return c
        except Exception:
            pass
    return {"stale": True}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            try:
                self.proc.kill()
            except Exception:
                pass
        try:
            sm, mx, reasons = [], [], set()
            for line in open(self.path):
                t = [x.strip() for x in line.split(",")]
                if len(t) < 9:
                    continue
                try:
                    sm.append(float(t[1]))
                    mx.append(float(t[2]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"),
                                   t[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            if sm:
                out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                       "samples": len(sm)}
            os.unlink(self.path)
        except Exception:
            pass
        return out


# ---------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of the default run, and --impl reference)
# ---------------------------------------------------------------------------

def oracle_sweep_sample(n_replicas: int, n: int, seed0: int, threads: int, keep=None, n_seeds: int = 4096):
    """Run the oracle on `n_replicas` replicas spread evenly over the sweep
    (generate -> simulate -> p50/p90).  -> (requests, seconds).  `keep` (a dict) receives
    replica index -> the oracle's summary tuple, for the parity check after the timed legs."""
    import concurrent.futures as cf
    import oracle as orc
    cfg = wl.config3(n_seeds=n_seeds, n=n, seed0=seed0)
    ln_dur, exp_t = wl.ln_dur_table(), wl.exp_table()
    total = cfg["n_seeds"] * len(cfg["rates_mhz"]) * len(cfg["policies"])
    picks = np.unique(np.linspace(0, total - 1, min(n_replicas, total)).astype(np.int64))
    cm = orc.cost(*cfg["cost"])
    orc.lib()

    def one(r):
        t, pol = divmod(int(r), 3)
        s, ri = divmod(t, 8)
        dist = 1 if s >= cfg["n_seeds"] // 2 else 0
        tr = orc.gen_trace(seed0 + s, cfg["rates_mhz"][ri], dist, n, ln_dur, exp_t)
        lat, ttft, first, end = orc.simulate(tr, cfg["policies"][pol], cm, cfg["slots"])
        return (orc.percentile(lat, 50), orc.percentile(lat, 90), orc.percentile(ttft, 50), orc.percentile(ttft, 90),
                first, end, n)

    t0 = time.perf_counter()
    with cf.ThreadPoolExecutor(max_workers=threads) as ex:   # ctypes releases the GIL
        res = list(ex.map(one, picks))
    dt = time.perf_counter() - t0
    if keep is not None:
        keep.update((int(r), v) for r, v in zip(picks, res))
    return len(picks) * n, dt


def oracle_select_sample(n_queues: int, q_len: int, threads: int, keep=None):
    """the first n_queues queues of the config-5 stream, HRRN + SJF, sort everything and take k.
    `keep` (a dict) receives policy -> int32[n_queues, k] of the oracle's indices."""
    import concurrent.futures as cf
    import oracle as orc
    cfg = wl.config5(q_len=q_len)
    ln_dur = wl.ln_dur_table()
    qs = orc.gen_queue(cfg["seed"], 0, n_queues * q_len, cfg["now"], ln_dur).reshape(n_queues, q_len)

    def one(i):
        return [orc.select(qs[i], pol, cfg["now"], cfg["k"]) for pol in cfg["policies"]]

    t0 = time.perf_counter()
    with cf.ThreadPoolExecutor(max_workers=threads) as ex:
        res = list(ex.map(one, range(n_queues)))
    dt = time.perf_counter() - t0
    if keep is not None:
        for j, pol in enumerate(cfg["policies"]):
            keep[pol] = np.stack([r[j] for r in res]) if res else np.zeros((0, cfg["k"]), dtype=np.int32)
    return n_queues * q_len * 16 * len(cfg["policies"]) / dt / 1e9, dt


SUMMARY_FIELDS = ("p50_e2e_us", "p90_e2e_us", "p50_ttft_us", "p90_ttft_us", "first_arrival_us", "last_done_us",
                  "n_done")


def cpu_baseline(n: int, n_seeds: int, q_len: int, summ, idx_by_policy, target_s: float = 25.0):
    """The oracle as it stands, timed on the host cores over a bounded sample of the workload -- and, because
    those results are the oracle's answers for the very replicas and queues the timed launches processed,
    compared (after the clock has stopped) with the GPU's full-size outputs: `summ` = the per-replica summaries
    of the timed sweep, `idx_by_policy` = the index rows of the timed select launches.
    -> (cpu_baseline dict, parity_checked dict)"""
    cores = os.cpu_count() or 1
    total_rep = n_seeds * 8 * 3
    req, dt = oracle_sweep_sample(cores, n, 0, cores, n_seeds=n_seeds)          # pilot: one replica per core
    per_replica = dt / max(1, req // n) * cores
    count = int(max(cores, min(total_rep, target_s * cores / max(per_replica, 1e-6))))
    kept = {}
    req, dt = oracle_sweep_sample(count, n, 0, cores, keep=kept, n_seeds=n_seeds)
    _, pilot_dt = oracle_select_sample(cores * 4, q_len, cores)
    n_have = min(len(v) for v in idx_by_policy.values()) if idx_by_policy else 0
    n_sel = int(max(cores * 4, min(65536, 4.0 * cores * 4 / max(pilot_dt, 1e-6))))   # about 4 s
    kept_sel = {}
    sel_gbs, sel_dt = oracle_select_sample(n_sel, q_len, cores, keep=kept_sel)
    # ---- parity of the full-size launches against what the oracle just computed (untimed)
    bad_rep = [r for r, want in kept.items()
               if r < len(summ) and tuple(int(summ[r][f]) for f in SUMMARY_FIELDS) != tuple(int(x) for x in want)]
    n_q = min(n_sel, n_have)
    bad_q = {pol: int((np.asarray(idx_by_policy[pol][:n_q]) != kept_sel[pol][:n_q]).any(axis=1).sum())
             for pol in kept_sel if pol in idx_by_policy}
    parity = {"replicas": len([r for r in kept if r < len(summ)]), "replicas_total": int(len(summ)),
              "queues": int(n_q), "queues_total": int(n_have), "queue_policies": sorted(bad_q),
              "mismatches": len(bad_rep) + sum(bad_q.values()),
              "what": "oracle summaries (p50/p90 E2E, p50/p90 TTFT, first arrival, last completion, n_done) of the "
                      "sampled config-3 replicas vs the timed sweep's output; oracle top-k index rows of the first "
                      "queues of config 5 vs the timed select launches' output, per policy; tolerance 0"}
    if bad_rep:
        parity["first_bad_replicas"] = bad_rep[:8]
    base = {"value": req / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d of the %d config-3 replicas (evenly spaced over seeds x rates x policies, "
                      "n=%d each; generate+simulate+p50/p90), %.1f s wall on %d threads"
                      % (req // n, total_rep, n, dt, cores),
            "select_gbs": sel_gbs,
            "select_sample": "%d config-5 queues x %d, HRRN+SJF full sort, %.1f s" % (n_sel, q_len, sel_dt)}
    return base, parity


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    per_step = max(cores, args.ref_replicas)
    for _ in range(args.warmup):
        oracle_sweep_sample(cores, args.n, 0, cores)
    req_total, t_total = 0, 0.0
    for s in range(args.steps):
        req, dt = oracle_sweep_sample(per_step, args.n, 0, cores)
        req_total += req
        t_total += dt
    value = req_total / t_total
    sample = "%d config-3 replicas per step (evenly spaced over the sweep), n=%d" % (per_step, args.n)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / max(1, args.steps),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
            "data": "synthetic",
            "config": {"workload": "config3 replica sweep (sampled): seeds x 8 rates x 3 policies, "
                                   "%d requests per replica, 32 slots" % args.n, "timing": "host wall clock"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------

def side_configs(asr, dev, d_tables, reps=5):
    """BASELINE.json configs[0], [1] and [3] (the small and the deep-backlog cases): generate ->
    simulate with per-request outputs and summary, CUDA events, median of `reps` runs.  Not part of
    `value`; parity of all three is in tests/ (-m gpu)."""
    import torch
    out = {}

    def timed(fn, reps=reps, warm=True):
        ms = []
        if warm:
            fn()
        torch.cuda.synchronize()
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        return statistics.median(ms)

    for cfg, rates in ((wl.config1(), None), (wl.config2(), wl.config2()["rates_mhz"])):
        rates = rates or (cfg["rate_mhz"],)
        n, pols = cfg["n"], cfg["policies"]
        specs = np.zeros(len(rates), dtype=asr.SPEC_DTYPE)
        specs["seed"], specs["rate_mhz"], specs["dist"] = cfg["seed"], rates, cfg["dist"]
        n_rep = len(rates) * len(pols)
        rep = asr.make_replicas(np.repeat(np.arange(len(rates), dtype=np.int64) * n, len(pols)),
                                np.arange(n_rep, dtype=np.int64) * n, n,
                                np.tile(np.asarray(pols, dtype=np.int32), len(rates)), cfg["slots"], 0)
        d_specs, d_rep, d_cost = (asr.to_device(x, dev) for x in (specs, rep, asr.make_cost(*cfg["cost"])))
        d_tr = torch.empty(len(rates) * n * 16, dtype=torch.uint8, device=dev)
        d_lat = torch.empty(n_rep * n, dtype=torch.int64, device=dev)
        d_ttft = torch.empty(n_rep * n, dtype=torch.int64, device=dev)
        d_sum = torch.zeros(n_rep * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device=dev)

        def step():
            asr.gen_trace_batched(d_specs, len(rates), n, d_tables, out=d_tr)
            asr.simulate_batched(d_tr, d_rep, n_rep, d_cost, 1, n_rep * n, cfg["slots"], d_lat, d_ttft, d_sum)
        ms = timed(step)
        out[cfg["name"]] = {"replicas": n_rep, "requests_per_replica": n, "ms": ms,
                            "requests_per_s": n_rep * n / (ms / 1e3)}
    cfg = wl.config4()
    n = cfg["n"]
    cost = asr.make_cost(*cfg["cost"])
    d_tr = torch.empty(n * 16, dtype=torch.uint8, device=dev)
    n_pol = len(cfg["policies"])
    # the policies are two replicas of one batched call (they share the trace; one CTA each, side by side)
    rep4 = asr.make_replicas([0] * n_pol, [i * n for i in range(n_pol)], n, list(cfg["policies"]), cfg["slots"], 0)
    d_rep4, d_cm4 = asr.to_device(rep4), asr.to_device(cost)
    d_lat4 = torch.empty(n_pol * n, dtype=torch.int64, device=dev)
    d_ttft4 = torch.empty(n_pol * n, dtype=torch.int64, device=dev)
    d_sum4 = torch.zeros(n_pol * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device=dev)

    def step4():
        asr.gen_trace(cfg["seed"], cfg["rate_mhz"], cfg["dist"], n, d_tables, out=d_tr)
        asr.simulate_batched(d_tr, d_rep4, n_pol, d_cm4, 1, n_pol * n, cfg["slots"], d_lat4, d_ttft4, d_sum4)
    ms = timed(step4, reps=2, warm=False)   # about a second per run: kept short
    summ = d_sum4.cpu().numpy().view(asr.SUMMARY_DTYPE)
    assert all(int(x) == n for x in summ["n_done"]), "config 4 did not complete"
    out[cfg["name"]] = {"replicas": n_pol, "requests_per_replica": n, "ms": ms,
                        "requests_per_s": n_pol * n / (ms / 1e3),
                        "note": "one sequential replica per policy (HRRN, SJF: two CTAs of one batched call), "
                                "backlog ~2.3e5 waiting, per-request outputs and p50/p90 included"}
    return out


def overload_sweep(asr, dev, d_tables, reps=3, n_seeds=512, n=3000, check=True):
    """The contended regime of the BASE simulator (Table 1 rows 20-25 req/s):
    n_seeds seeds x 8 arrival rates 16..30 req/s x 3 policies x n lognormal requests, at 16 and at 32 slots,
    through plain asr_sched_simulate_batched (summary-only, default options).  Above ~20 (16 slots) / ~23
    (32 slots) req/s the queue grows and SJF/HRRN choose at every admission.  Reports requests/s, the split
    of the time over the thread / warp / CTA tiers.  With `check` (the cpu_baseline / parity leg of the run, never
    inside a timed region) a sample of replicas is compared with the oracle, tolerance 0."""
    import torch
    if check:
        import oracle as orc
    rates = np.arange(16000, 31000, 2000, dtype=np.int32)                       # mHz
    pols = (wl.FCFS, wl.SJF, wl.HRRN)
    n_tr, n_rep = n_seeds * len(rates), n_seeds * len(rates) * len(pols)
    specs = np.zeros(n_tr, dtype=asr.SPEC_DTYPE)
    specs["seed"] = np.repeat(np.arange(n_seeds, dtype=np.uint64) + np.uint64(7000), len(rates))
    specs["rate_mhz"] = np.tile(rates, n_seeds)
    specs["dist"] = wl.DIST_LOGNORMAL
    d_specs, d_cost = asr.to_device(specs, dev), asr.to_device(asr.make_cost(*wl.CONFIG_COST), dev)
    d_tr = torch.empty(n_tr * n * 16, dtype=torch.uint8, device=dev)
    asr.gen_trace_batched(d_specs, n_tr, n, d_tables, out=d_tr)
    d_sum = torch.zeros(n_rep * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    from paper_2603_11273_b200 import binding as B
    d_ws = torch.empty(asr.workspace_bytes(B.OP_SIMULATE, n_rep * n, n_rep, 1), dtype=torch.uint8, device=dev)
    out = {"workload": "%d seeds x 8 rates 16-30 req/s x 3 policies = %d replicas x %d lognormal requests, "
                       "config-1 cost model, summary-only simulate_batched" % (n_seeds, n_rep, n)}
    ln, ex = wl.ln_dur_table(), wl.exp_table()
    for slots in (16, 32):
        rep = asr.make_replicas(np.repeat(np.arange(n_tr, dtype=np.int64) * n, len(pols)),
                                np.arange(n_rep, dtype=np.int64) * n, n,
                                np.tile(np.asarray(pols, dtype=np.int32), n_tr), slots, 0)
        d_rep = asr.to_device(rep, dev)

        def step():
            asr.simulate_batched(d_tr, d_rep, n_rep, d_cost, 1, n_rep * n, slots, None, None, d_sum, workspace=d_ws)
        step()
        torch.cuda.synchronize()
        asr.timing_enable(True)
        asr.timing_reset()
        ms = []
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            step()
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        kt = asr.timing_read()
        asr.timing_enable(False)
        summ = d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)
        assert int((summ["n_done"] == n).sum()) == n_rep, "overload sweep: replicas did not finish"
        # parity sample: evenly spaced replicas against the oracle
        bad = 0
        picks = np.linspace(0, n_rep - 1, 48).astype(np.int64) if check else []
        for r in picks:
            tr_i, pol = int(r) // len(pols), pols[int(r) % len(pols)]
            tr = orc.gen_trace(int(specs["seed"][tr_i]), int(specs["rate_mhz"][tr_i]), orc.DIST_LOGNORMAL, n, ln, ex)
            rl, rt, first, end = orc.simulate(tr, pol, orc.cost(*wl.CONFIG_COST), slots)
            want = (orc.percentile(rl, 50), orc.percentile(rl, 90), orc.percentile(rt, 50), orc.percentile(rt, 90),
                    first, end, n)
            got = tuple(int(summ[r][f]) for f in ("p50_e2e_us", "p90_e2e_us", "p50_ttft_us", "p90_ttft_us",
                                                  "first_arrival_us", "last_done_us", "n_done"))
            bad += int(got != want)
        med = statistics.median(ms)
        out["slots%d" % slots] = {
            "ms": med, "requests_per_s": n_rep * n / (med / 1e3),
            "kernel_ms": {k: v[0] / reps for k, v in kt.items() if v[1]},
            "parity_sample": {"replicas": int(len(picks)), "mismatches": bad} if check else None}
    return out


def extension_lines(asr, dev, d_tables, hbm_peak, reps=5, consts=None):
    """SURVEY.md 8(f) rows, each timed alone (CUDA events through the library's per-kernel timers):
    the two HBM streams against the measured HBM peak, the extended simulator on an overloaded
    sweep with a KV budget that binds."""
    import torch
    out = {}
    cost_h = asr.make_cost(*wl.CONFIG_COST)
    # --- estimate + tpot on 2^26 records
    n = 1 << 26
    d_tr = asr.gen_queues(77, 0, n, 10**10, d_tables)
    d_lat = torch.randint(10**5, 10**7, (n,), dtype=torch.int64, device=dev)
    d_ttft = torch.randint(10**3, 10**5, (n,), dtype=torch.int64, device=dev)
    d_out = torch.empty(n, dtype=torch.int64, device=dev)
    d_lang = torch.randint(0, 4, (n,), dtype=torch.uint8, device=dev)
    for _ in range(2):
        asr.estimate(d_tr, n, [5000, 2500, 7300, 4100], d_lang)
        asr.tpot(d_tr, n, cost_h, d_lat, d_ttft, d_out)
    torch.cuda.synchronize()
    asr.timing_enable(True)
    asr.timing_reset()
    for _ in range(reps):
        asr.estimate(d_tr, n, [5000, 2500, 7300, 4100], d_lang)
        asr.tpot(d_tr, n, cost_h, d_lat, d_ttft, d_out)
    kt = asr.timing_read()
    for name, bytes_per in (("estimate_kernel", 16 + 1 + 4), ("tpot_kernel", 16 + 8 + 8 + 8)):
        ms, cnt = kt.get(name, (0.0, 0))
        if cnt:
            a = n * bytes_per / (ms / cnt / 1e3) / 1e9
            out[name] = {"bound": "hbm", "achieved": a, "peak": hbm_peak, "unit": "GB/s", "frac": a / hbm_peak,
                         "algorithmic_bytes_per_launch": n * bytes_per, "avg_launch_ms": ms / cnt, "records": n}
    del d_tr, d_lat, d_ttft, d_out, d_lang
    # --- extended simulator: 256 seeds x 8 overload rates x 3 policies, 3,000 requests, 16 slots, KV budget
    n_seeds, n_req, slots = 256, 3000, 16
    rates = [16000, 18000, 20000, 22000, 24000, 26000, 28000, 30000]        # PAPER.md:104 heavy range, mHz
    seeds = np.repeat(np.arange(n_seeds, dtype=np.uint64) + 5000, len(rates))
    specs = np.zeros(len(seeds), dtype=asr.SPEC_DTYPE)
    specs["seed"], specs["rate_mhz"], specs["dist"] = seeds, np.tile(rates, n_seeds), 0
    n_tr, n_rep = len(seeds), len(seeds) * 3
    rep = asr.make_replicas(np.repeat(np.arange(n_tr, dtype=np.int64) * n_req, 3),
                            np.arange(n_rep, dtype=np.int64) * n_req, n_req,
                            np.tile(np.asarray([0, 1, 2], dtype=np.int32), n_tr), slots, 0)
    d_specs, d_rep, d_cost = (asr.to_device(x, dev) for x in (specs, rep, cost_h))
    d_ext = asr.to_device(asr.make_ext(kv_budget=25 * slots, kv_base=20, kv_per_s=2), dev)
    d_trs = asr.gen_trace_batched(d_specs, n_tr, n_req, d_tables)
    d_sum = torch.zeros(n_rep * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    d_pre = torch.zeros(n_rep, dtype=torch.int64, device=dev)
    from paper_2603_11273_b200 import binding as B
    d_ws = torch.empty(asr.workspace_bytes(B.OP_SIMULATE_EX, n_rep * n_req, n_rep, 1), dtype=torch.uint8, device=dev)

    def step():
        asr.simulate_batched_ex(d_trs, d_rep, n_rep, d_cost, d_ext, 1, n_rep * n_req, slots, None, None, d_sum, d_pre,
                                workspace=d_ws)
    step()
    torch.cuda.synchronize()
    asr.timing_reset()
    for _ in range(reps):
        step()
    kt = asr.timing_read()
    asr.timing_enable(False)
    ms, cnt = kt.get("sim_ex_kernel", (0.0, 0))
    summ = d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)
    # --- inter-token latency of the same replicas (simulate with gap capture + weighted percentiles)
    asr.timing_enable(True)
    asr.timing_reset()
    d_ws_itl = torch.empty(asr.workspace_bytes(B.OP_ITL, n_rep * n_req, n_rep, 0), dtype=torch.uint8, device=dev)
    for _ in range(reps):
        d_itl = asr.itl_batched(d_trs, d_rep, n_rep, d_cost, 1, n_rep * n_req, slots, [50, 90], workspace=d_ws_itl)
    kt_itl = asr.timing_read()
    asr.timing_enable(False)
    ms_p, cnt_p = kt_itl.get("itl_percentiles_kernel", (0.0, 0))
    ms_s, cnt_s = kt_itl.get("sim_ex_kernel", (0.0, 0))
    if cnt_p and cnt_s:
        gaps = int(d_itl[:, 2].sum().item())
        out["itl"] = {"workload": "the same %d replicas, no KV budget; P50/P90 of %d inter-token gaps per pass" % (n_rep, gaps),
                      "sim_ex_kernel_ms": ms_s / cnt_s, "itl_percentiles_kernel_ms": ms_p / cnt_p,
                      "requests_per_s": n_rep * n_req / ((ms_s / cnt_s + ms_p / cnt_p) / 1e3)}
    if cnt:
        out["sim_ex_kernel"] = {"bound": "alu", "workload": "%d replicas x %d requests at 16-30 req/s, %d slots, KV budget %d "
                                "(base 20 + 2/s of audio + generated tokens)" % (n_rep, n_req, slots, 25 * slots),
                                "avg_launch_ms": ms / cnt, "requests_per_s": n_rep * n_req / (ms / cnt / 1e3),
                                "preemptions_per_request": float(d_pre.sum().item()) / (n_rep * n_req),
                                "replicas_done": int((summ["n_done"] == n_req).sum())}
        wi = (consts or {}).get("sim_ex_kernel_warp_instr_per_request")
        if wi:   # issue-slot roofline as for the base simulator (ncu counter from the committed capture)
            a = wi * n_rep * n_req / (ms / cnt / 1e3)
            out["sim_ex_kernel"].update({"achieved": a, "peak": ALU_PEAK_WARP_INSTR_PER_S, "unit": "warp-instr/s",
                                         "frac": a / ALU_PEAK_WARP_INSTR_PER_S, "warp_instr_per_request": wi,
                                         "constants_stale": bool((consts or {}).get("stale"))})
    return out


def run_ours(args):
    import torch
    import paper_2603_11273_b200 as asr
    from paper_2603_11273_b200 import dist as D

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    rank, world, local = D.init()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    hbm_peak, peak_src = load_peaks()
    consts = load_profile_constants()

    if args.side_configs_only:
        # configs 1, 2 and 4 alone (the warp- and CTA-per-replica tiers): the command the ncu captures of those
        # kernels are taken with; prints its own line, not the bench line
        d_tables = asr.to_device(asr.make_tables(wl.ln_dur_table(), wl.exp_table()), dev)
        if rank == 0:
            side = {} if args.overload_only else side_configs(asr, dev, d_tables, reps=args.steps)
            side["overload_sweep"] = overload_sweep(asr, dev, d_tables, reps=min(args.steps, 3),
                                                    check=not args.no_cpu_baseline)
            print(json.dumps({"configs": side}))
        D.finalize()
        return

    # ---- inputs, resident in HBM before any timed region ------------------
    cfg3 = wl.config3(n_seeds=args.seeds, n=args.n, seed0=D.seed_block(rank, args.seeds))
    seeds, rates, dist = wl.config3_traces(cfg3)
    n_traces, n, n_pol = len(seeds), cfg3["n"], len(cfg3["policies"])
    n_rep = n_traces * n_pol
    total = n_rep * n
    specs = np.zeros(n_traces, dtype=asr.SPEC_DTYPE)
    specs["seed"], specs["rate_mhz"], specs["dist"] = seeds, rates, dist
    rep = asr.make_replicas(np.repeat(np.arange(n_traces, dtype=np.int64) * n, n_pol),
                            np.arange(n_rep, dtype=np.int64) * n, n,
                            np.tile(np.asarray(cfg3["policies"], dtype=np.int32), n_traces), cfg3["slots"], 0)
    tables_h = asr.make_tables(wl.ln_dur_table(), wl.exp_table())
    cost_h = asr.make_cost(*cfg3["cost"])
    d_tables, d_specs, d_rep, d_cost = (asr.to_device(x, dev) for x in (tables_h, specs, rep, cost_h))
    d_traces = torch.empty(n_traces * n * 16, dtype=torch.uint8, device=dev)
    d_sum = torch.zeros(n_rep * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    from paper_2603_11273_b200 import binding as B
    d_ws = torch.empty(asr.workspace_bytes(B.OP_SIMULATE, total, n_rep, 1), dtype=torch.uint8, device=dev)

    def sweep_step():
        asr.gen_trace_batched(d_specs, n_traces, n, d_tables, out=d_traces)
        asr.simulate_batched(d_traces, d_rep, n_rep, d_cost, 1, total, cfg3["slots"], None, None, d_sum, workspace=d_ws)

    cfg5 = wl.config5(n_queues=args.queues)
    nq, ql, k5, now5 = cfg5["n_queues"], cfg5["q_len"], cfg5["k"], cfg5["now"]
    d_queues = asr.gen_queues(cfg5["seed"], rank * nq * ql, nq * ql, now5, d_tables)
    d_idx = torch.empty((nq, k5), dtype=torch.int32, device=dev)

    def select_step():
        for pol in cfg5["policies"]:
            asr.select_batched(d_queues, nq, ql, pol, now5, k5, out_idx=d_idx)

    torch.cuda.synchronize()
    for _ in range(args.warmup):
        sweep_step()
        select_step()
    torch.cuda.synchronize()

    # ---- timed regions ------------------------------------------------------
    sampler = ClockSampler(local)
    sampler.start()
    asr.timing_enable(True)
    asr.timing_reset()
    launches0 = asr.launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    D.barrier()
    torch.cuda.synchronize()
    ev[0].record()
    for _ in range(args.steps):
        sweep_step()
    ev[1].record()
    torch.cuda.synchronize()
    D.barrier()
    sweep_ms = D.max_over_ranks(ev[0].elapsed_time(ev[1]))
    D.barrier()
    torch.cuda.synchronize()
    ev[2].record()
    for _ in range(args.steps):
        select_step()
    ev[3].record()
    torch.cuda.synchronize()
    D.barrier()
    select_ms = D.max_over_ranks(ev[2].elapsed_time(ev[3]))
    launches = asr.launch_count() - launches0
    ktimes = asr.timing_read()
    asr.timing_enable(False)
    clocks = sampler.stop()
    # the wide select (32 < k <= 256) on the same queues: reported beside the headline k = 32
    wide = None
    if rank == 0:
        d_idx_w = torch.empty((nq, 256), dtype=torch.int32, device=dev)
        asr.select_batched(d_queues, nq, ql, cfg5["policies"][0], now5, 256, out_idx=d_idx_w)
        torch.cuda.synchronize()
        w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        w0.record()
        for pol in cfg5["policies"]:
            asr.select_batched(d_queues, nq, ql, pol, now5, 256, out_idx=d_idx_w)
        w1.record()
        torch.cuda.synchronize()
        wms = w0.elapsed_time(w1) / len(cfg5["policies"])
        wide = {"k": 256, "ms_per_launch": wms, "gbs": (nq * ql * 16 + nq * 256 * 4) / (wms / 1e3) / 1e9,
                "kernel": "select_wide_kernel (shared-memory sort; not the streaming design of k <= 32)"}
        del d_idx_w
    # the index rows of the same launches once more, per policy, for the parity check of the cpu_baseline leg
    idx_by_policy = {}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        for pol in cfg5["policies"]:
            asr.select_batched(d_queues, nq, ql, pol, now5, k5, out_idx=d_idx)
            torch.cuda.synchronize()
            idx_by_policy[pol] = d_idx.cpu().numpy().copy()

    summ = d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)
    assert int((summ["n_done"] == n).sum()) == n_rep, "replicas did not finish"

    value = world * total * args.steps / (sweep_ms / 1e3)
    sel_bytes = nq * ql * 16 + nq * k5 * 4
    select_gbs = world * sel_bytes * len(cfg5["policies"]) * args.steps / (select_ms / 1e3) / 1e9

    def per_launch(name):
        ms, cnt = ktimes.get(name, (0.0, 0))
        return (ms / cnt if cnt else None), cnt, ms

    sel_avg, sel_cnt, sel_tot = per_launch("select_topk_kernel")
    gen_avg, _, gen_tot = per_launch("gen_trace_kernel")
    # the percentile reduction of a summary-only sweep = the radix kernel on the seeds, the one-warp-per-stream
    # kernel, the radix kernel on what that left: per step (the radix kernel is timed twice per step)
    pf_avg, pf_cnt, pf_tot = per_launch("summary_stream_kernel")
    pr_avg, pr_cnt, pr_tot = per_launch("summary_percentiles_kernel")
    pct_tot = (pf_tot or 0.0) + (pr_tot or 0.0)
    pct_avg = pct_tot / (pf_cnt or pr_cnt) if (pf_cnt or pr_cnt) else None
    # the thread-per-replica tier = plan + units + repair + redo
    lane_parts = {k_: per_launch(k_) for k_ in ("sim_lane_kernel", "lane_plan_kernels", "sim_lane_kernel(repair)",
                                                 "sim_lane_kernel(redo)")}
    rooflines = {}
    if sel_avg:
        a = sel_bytes / (sel_avg / 1e3) / 1e9
        rooflines["select_topk_kernel"] = {
            "bound": "hbm", "achieved": a, "peak": hbm_peak, "unit": "GB/s", "frac": a / hbm_peak,
            "traffic": consts.get("select_dram_bytes_per_launch"), "peak_source": peak_src,
            "algorithmic_bytes_per_launch": sel_bytes, "avg_launch_ms": sel_avg, "frac_of_nominal_8TBs": a / 8000.0}
    stage_ms = {"gen_trace_kernel": gen_tot, "summary_stream_kernel": pct_tot}
    for kname in ("sim_lane_kernel", "sim_warp_kernel"):
        k_avg, k_cnt, k_tot = per_launch(kname)
        if not k_avg:
            continue
        stage_ms[kname] = k_tot
        if kname == "sim_lane_kernel":
            stage_ms[kname] = sum(v[2] or 0.0 for v in lane_parts.values())
        # ALU/issue-bound: achieved = warp instructions issued per second; the per-request instruction counts
        # are ncu counters committed in profiles/roofline_constants.json (stale = captured from other sources).
        # A kernel that executed MORE instructions per request would score higher on `frac`, so the line also
        # carries the thread-level figure: thread instructions (warp instructions x active threads) per second
        # against 32 threads per issue slot.
        full = n == 10000 and cfg3["slots"] == 32
        wi = consts.get(kname + "_warp_instr_per_request") if full else None
        ti = consts.get(kname + "_thread_instr_per_request") if full else None
        a = (wi * total / (k_avg / 1e3)) if wi else None
        at = (ti * total / (k_avg / 1e3)) if ti else None
        rooflines[kname] = {
            "bound": "alu", "achieved": a, "peak": ALU_PEAK_WARP_INSTR_PER_S, "unit": "warp-instr/s",
            "frac": (a / ALU_PEAK_WARP_INSTR_PER_S) if a else None,
            "traffic": consts.get(kname + "_dram_bytes_per_launch"),
            "warp_instr_per_request": wi, "thread_instr_per_request": ti,
            "threads_per_warp_instr": (ti / wi) if (wi and ti) else None,
            "frac_thread_level": (at / (32 * ALU_PEAK_WARP_INSTR_PER_S)) if at else None,
            "algorithmic_bytes_per_launch": (n_traces * n * 16 + 2 * total * 4) if kname == "sim_lane_kernel" else None,
            "avg_launch_ms": k_avg, "constants_stale": bool(consts.get("stale")),
            "tier_ms_per_step": ({k_: (v[2] or 0.0) / args.steps for k_, v in lane_parts.items()}
                                 if kname == "sim_lane_kernel" else None),
            "peak_source": "148 SMs x 4 schedulers x 1.965 GHz (DESIGN.md)"}
    if gen_avg:
        a = n_traces * n * 16 / (gen_avg / 1e3) / 1e9
        rooflines["gen_trace_kernel"] = {"bound": "hbm", "achieved": a, "peak": hbm_peak, "unit": "GB/s",
                                         "frac": a / hbm_peak, "traffic": consts.get("gen_trace_dram_bytes_per_launch"),
                                         "algorithmic_bytes_per_launch": n_traces * n * 16, "avg_launch_ms": gen_avg}
    if pct_avg:
        # summary-only sweeps hand the reduction uint32 values (the lane kernel proves < 2^32 us): 4 B per value
        pct_bytes = 2 * total * 4
        a = pct_bytes / (pct_avg / 1e3) / 1e9
        rooflines["summary_stream_kernel"] = {"bound": "hbm", "achieved": a, "peak": hbm_peak, "unit": "GB/s",
                                            "frac": a / hbm_peak,
                                            "traffic": consts.get("summary_percentiles_dram_bytes_per_launch"),
                                            "algorithmic_bytes_per_launch": pct_bytes,
                                            "avg_launch_ms": pct_avg,
                                            "note": "seed pass (radix kernel) + one warp per value stream + radix kernel on the segments it left, per step"}
    dominant = max(stage_ms, key=lambda k_: stage_ms[k_] or 0.0)
    roofline = dict(rooflines.get(dominant, {}), kernel=dominant,
                    share_of_step=(stage_ms[dominant] / sweep_ms) if sweep_ms else None)

    # ---- end to end through the host-buffer C-ABI calls ---------------------
    e2e = None
    if not args.no_e2e:
        pol_h = np.asarray(cfg3["policies"], dtype=np.int32)
        out_h = np.zeros(n_rep, dtype=asr.SUMMARY_DTYPE)
        asr.sweep_host(specs, n, tables_h, pol_h, cfg3["slots"], cost_h, out_h)      # warm-up
        D.barrier()
        t0 = time.perf_counter()
        e2e_steps = max(1, min(args.steps, 3))
        for _ in range(e2e_steps):
            asr.sweep_host(specs, n, tables_h, pol_h, cfg3["slots"], cost_h, out_h)
        e2e_s = D.max_over_ranks(time.perf_counter() - t0)
        assert np.array_equal(out_h.view(np.uint8), summ.view(np.uint8)), "host-buffer sweep disagrees"
        h2d = specs.nbytes + tables_h.nbytes + cost_h.nbytes + pol_h.nbytes
        e2e = {"value": world * total * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(out_h.nbytes), "steps": e2e_steps,
               "call": "asr_sched_sweep_host (host specs/tables in, host summaries out; device scratch from the "
                       "stream-ordered pool inside the call, cached between calls)"}
        # select with host records: pinned host keys in, host indices out
        try:
            h_keys = torch.empty(nq * ql * 16, dtype=torch.uint8, pin_memory=True)
            h_keys.copy_(d_queues)
            h_idx = torch.empty((nq, k5), dtype=torch.int32, pin_memory=True)
            torch.cuda.synchronize()
            asr.select_host(h_keys, nq, ql, cfg5["policies"][0], now5, k5, h_idx)   # warm-up
            t0 = time.perf_counter()
            for pol in cfg5["policies"]:
                asr.select_host(h_keys, nq, ql, pol, now5, k5, h_idx)
            dt = D.max_over_ranks(time.perf_counter() - t0)
            e2e["select_gbs"] = world * sel_bytes * len(cfg5["policies"]) / dt / 1e9
            e2e["select_h2d_bytes_per_call"] = int(nq * ql * 16)
            e2e["select_d2h_bytes_per_call"] = int(nq * k5 * 4)
            del h_keys
        except Exception as exc:  # pinned allocation can fail on a small host
            e2e["select_error"] = str(exc)[:200]

    side = ext_lines = None
    if rank == 0 and not args.no_side_configs:
        del d_traces, d_ws, d_queues
        torch.cuda.empty_cache()
        side = side_configs(asr, dev, d_tables)
        side["overload_sweep"] = overload_sweep(asr, dev, d_tables, check=not args.no_cpu_baseline)
        ext_lines = extension_lines(asr, dev, d_tables, hbm_peak, consts=consts)

    base = parity = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        base, parity = cpu_baseline(n, args.seeds, ql, summ, idx_by_policy)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sweep_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
            "config": {
                "workload": "config3 replica sweep: %d seeds x 8 rates x 3 policies = %d replicas x %d requests "
                            "per GPU, 32 slots, config-1 cost model; half lognormal, half uniform durations"
                            % (args.seeds, n_rep, n),
                "select_workload": "config5: %d queues x %d records, now=1e10, k=32, HRRN+SJF" % (nq, ql),
                "l2": "inputs_larger_than_l2 (traces %.2f GB, queues %.2f GB per GPU; L2 126 MB)"
                      % (n_traces * n * 16 / 1e9, nq * ql * 16 / 1e9),
                "parallelism": "replicas/queues sharded over %d GPU(s), no collective" % world,
                "step": "gen_trace_batched -> simulate_batched(summary-only: simulate + p50/p90)"},
            "select": {"metric": "priority-select GB/s vs HBM peak", "value": select_gbs, "unit": "GB/s",
                       "ms_per_step": select_ms / args.steps, "policies": ["hrrn", "sjf"],
                       "frac_of_measured_peak": select_gbs / world / hbm_peak,
                       "frac_of_nominal_8TBs": select_gbs / world / 8000.0, "wide": wide},
            "roofline": roofline, "rooflines": rooflines, "clocks": clocks, "e2e": e2e,
            "gpu_launches": int(launches), "cpu_baseline": base, "parity_checked": parity, "configs": side,
            "extensions": ext_lines,
            "kernel_ms_total": {k_: v[0] for k_, v in ktimes.items() if v[1]},
        }
        print(json.dumps(line), flush=True)
    D.finalize()
    ov_bad = 0
    if side and side.get("overload_sweep"):
        for v in side["overload_sweep"].values():
            if isinstance(v, dict) and v.get("parity_sample"):
                ov_bad += v["parity_sample"]["mismatches"]
    if ov_bad:
        print("bench.py: the overload sweep disagrees with the oracle on %d sampled replicas" % ov_bad, file=sys.stderr)
        return 3
    if parity is not None and parity["mismatches"] != 0:
        print("bench.py: the timed launches disagree with the oracle: %r" % parity, file=sys.stderr)
        return 3
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--seeds", type=int, default=4096, help="config-3 seeds per GPU (4096 = the full config)")
    ap.add_argument("--n", type=int, default=10000, help="requests per replica")
    ap.add_argument("--queues", type=int, default=65536, help="config-5 queues per GPU")
    ap.add_argument("--ref-replicas", type=int, default=256, help="--impl reference: replicas per step")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-side-configs", action="store_true", help="skip the config 1/2/4 timings")
    ap.add_argument("--side-configs-only", action="store_true", help="time configs 1, 2 and 4 and nothing else")
    ap.add_argument("--overload-only", action="store_true", help="with --side-configs-only: the overload sweep alone")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
