"""-m gpu: the CTA-per-replica simulator tier (deep backlogs, BASELINE.json configs[3]) against the
oracle, bit-exact.  The tier is reached by escalation from the warp kernel; ESCALATE_WINDOW = 0
sends every SJF/HRRN replica there as soon as the policy has to choose, so the stress traces
exercise its candidate pool in all its modes (complete pool, SJF threshold, HRRN threshold with
horizon, tie-heavy fallbacks)."""
import os

import numpy as np
import pytest

import oracle as orc
import workloads as wl
from gpu_util import check_replica, run_batched

pytestmark = pytest.mark.gpu
POL = (orc.FCFS, orc.SJF, orc.HRRN)
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config4_oracle.txt")


@pytest.fixture(scope="module")
def asr_mod():
    import torch
    assert torch.cuda.is_available()
    import paper_2603_11273_b200 as asr
    return asr


@pytest.fixture
def asr_cta(asr_mod):
    """warp kernel hands over at the first real choice"""
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_MIN_REPLICAS, 2**31 - 1)
    asr_mod.set_option(asr_mod.OPT_SIM_ESCALATE_WINDOW, 0)
    yield asr_mod
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_MIN_REPLICAS, 1024)
    asr_mod.set_option(asr_mod.OPT_SIM_ESCALATE_WINDOW, 4096)


def _cta_ms(asr):
    return asr.timing_read().get("sim_cta_kernel", (0.0, 0))[0]


@pytest.mark.parametrize("kind,rate,n", [("lognormal", 3.6, 2000), ("lognormal", 25.0, 3000), ("uniform", 12.0, 3000),
                                         ("burst", 1.0, 500), ("six", 14.0, 2500), ("equal_est", 25.0, 1500),
                                         ("clumped", 1.0, 1500), ("misest", 24.0, 2000)])
def test_stress_traces_through_the_cta_tier(asr_cta, kind, rate, n):
    asr = asr_cta
    tr = wl.stress_trace(kind, n, 7, rate_per_s=rate)
    reps = [(0, p, s) for s in (1, 16, 32) for p in POL]
    asr.timing_enable(True)
    asr.timing_reset()
    L, T, S = run_batched([tr], reps, wl.CONFIG_COST, 32)
    ms = _cta_ms(asr)
    asr.timing_enable(False)
    for i, (_, p, s) in enumerate(reps):
        check_replica(tr, p, s, wl.CONFIG_COST, L[i], T[i], S[i], "%s slots=%d pol=%d" % (kind, s, p))
    assert ms > 0.02, "the CTA tier did not run (%.4f ms)" % ms


@pytest.mark.parametrize("slots", [100, 256])
def test_wide_batches_through_the_cta_tier(asr_cta, slots):
    tr = wl.stress_trace("lognormal", 4000, 8, rate_per_s=90.0)
    br = wl.stress_trace("burst", 3000, 9)          # 3000 simultaneous arrivals: pool in threshold mode at once
    reps = [(0, p, slots) for p in POL] + [(1, p, slots) for p in POL]
    L, T, S = run_batched([tr, br], reps, wl.CONFIG_COST, slots)
    for i, (t, p, s) in enumerate(reps):
        check_replica([tr, br][t], p, s, wl.CONFIG_COST, L[i], T[i], S[i], "slots=%d rep=%d" % (slots, i))


@pytest.mark.parametrize("n", [20000, 60000])
def test_config4_recipe_reduced(asr_mod, tables, n):
    """config-4 recipe (seed 4, 35,408 mHz, 256 slots, HRRN and SJF) at a length the oracle finishes in
    seconds; default escalation: the backlog (up to ~0.23 n) outgrows the window limit on its own and the
    pool runs in threshold mode"""
    import torch
    asr = asr_mod
    cfg = wl.config4(n=n)
    d_tab = asr.tables_to_device(*tables)
    d_tr = asr.gen_trace(cfg["seed"], cfg["rate_mhz"], cfg["dist"], n, d_tab)
    torch.cuda.synchronize()
    tr = d_tr.cpu().numpy().view(asr.REQ_DTYPE)
    ref = orc.gen_trace(cfg["seed"], cfg["rate_mhz"], cfg["dist"], n, *tables)
    assert np.array_equal(tr.view(np.uint8), ref.view(np.uint8))
    asr.timing_enable(True)
    asr.timing_reset()
    reps = [(0, p, cfg["slots"]) for p in cfg["policies"]]
    L, T, S = run_batched([ref], reps, cfg["cost"], cfg["slots"])
    ms = _cta_ms(asr)
    asr.timing_enable(False)
    for i, (_, p, s) in enumerate(reps):
        check_replica(ref, p, s, cfg["cost"], L[i], T[i], S[i], "config4 n=%d pol=%d" % (n, p))
    assert ms > 0.5, "the deep backlog did not reach the CTA tier"


def test_tie_heavy_deep_backlog(asr_mod):
    """six distinct durations and a backlog of thousands: whole est classes tie, the
    histogram cannot separate them, the pool is refused and the exact window scan takes over"""
    asr = asr_mod
    tr = wl.stress_trace("six", 5000, 21, rate_per_s=40.0)
    eq = wl.stress_trace("equal_est", 5000, 22, rate_per_s=60.0)
    reps = [(0, orc.SJF, 32), (0, orc.HRRN, 32), (1, orc.HRRN, 16), (1, orc.SJF, 16)]
    asr.set_option(asr.OPT_SIM_ESCALATE_WINDOW, 1024)
    try:
        asr.timing_enable(True)
        asr.timing_reset()
        L, T, S = run_batched([tr, eq], reps, wl.CONFIG_COST, 32)
        ms = _cta_ms(asr)
        asr.timing_enable(False)
    finally:
        asr.set_option(asr.OPT_SIM_ESCALATE_WINDOW, 4096)
    for i, (t, p, s) in enumerate(reps):
        check_replica([tr, eq][t], p, s, wl.CONFIG_COST, L[i], T[i], S[i], "ties rep=%d" % i)
    assert ms > 0.5, "the CTA tier did not run"


def test_hrrn_pool_overflow_shrinks_the_horizon(asr_cta):
    """one early request, then thousands arriving within a few milliseconds: at the first threshold build every
    wait is a few tens of milliseconds, so the default one-second horizon lets nearly the whole backlog reach the
    threshold ratio; the pool overflows and the horizon has to shrink until it fits (the branch the Poisson traces
    never reach).  Later, with waits of many seconds, the same horizon fits again."""
    rng = np.random.Generator(np.random.PCG64(33))
    n = 5000
    arr = np.concatenate([[0], 1000 + np.arange(n, dtype=np.int64) * 3])
    dur = np.concatenate([[1000], np.clip(np.rint(np.exp(rng.normal(np.log(6000.0), 0.6, size=n))), 1000, 35000)])
    tr = np.zeros(n + 1, dtype=wl.REQ)
    tr["arrival_us"], tr["dur_ms"], tr["est"] = arr, dur.astype(np.int32), dur.astype(np.int32)
    reps = [(0, orc.HRRN, 64), (0, orc.SJF, 64), (0, orc.HRRN, 8)]
    L, T, S = run_batched([tr], reps, wl.CONFIG_COST, 64)
    for i, (_, p, s) in enumerate(reps):
        check_replica(tr, p, s, wl.CONFIG_COST, L[i], T[i], S[i], "overflow rep=%d" % i)


def _digests(v):
    u = v.astype(np.uint64)
    i = np.arange(len(u), dtype=np.uint64)
    with np.errstate(over="ignore"):
        s = int(u.sum(dtype=np.uint64))
        w = int(((i + np.uint64(1)) * u).sum(dtype=np.uint64))
        r = i % np.uint64(64)
        x = int(np.bitwise_xor.reduce((u << r) | (u >> ((np.uint64(64) - r) % np.uint64(64)))))
    return s, w, x


@pytest.mark.skipif(not os.path.exists(GOLDEN), reason="tests/golden/config4_oracle.txt not generated yet")
def test_config4_full_size_against_stored_oracle_results(asr_mod, tables):
    """BASELINE.json configs[3] at full size (10^6 requests).  Expected values were written by
    tests/golden/make_config4_golden.py from the oracle alone."""
    import torch
    asr = asr_mod
    lines = [l.split() for l in open(GOLDEN) if not l.startswith("#")]
    hdr = [l for l in open(GOLDEN) if l.startswith("# seed")][0].split()
    n, stride = int(hdr[hdr.index("n") + 1]), int(hdr[hdr.index("stride") + 1])
    assert int(hdr[hdr.index("tables_crc32") + 1]) == wl.table_checksum()
    cfg = wl.config4(n=n)
    d_tab = asr.tables_to_device(*tables)
    d_tr = asr.gen_trace(cfg["seed"], cfg["rate_mhz"], cfg["dist"], n, d_tab)
    cost = asr.make_cost(*cfg["cost"])
    want = {}
    cur = None
    for l in lines:
        if l[0] == "policy":
            cur = want.setdefault(int(l[1]), {})
        else:
            cur[l[0]] = [int(x) for x in l[1:]]
    for pol in cfg["policies"]:
        lat, ttft, summ = asr.simulate(d_tr, n, pol, cost, cfg["slots"])
        torch.cuda.synchronize()
        s = summ.cpu().numpy().view(asr.SUMMARY_DTYPE)[0]
        w = want[pol]
        got = [int(s[f]) for f in ("p50_e2e_us", "p90_e2e_us", "p50_ttft_us", "p90_ttft_us", "first_arrival_us",
                                   "last_done_us")]
        assert got == w["summary"], (pol, got, w["summary"])
        assert int(s["n_done"]) == n
        for name, arr in (("lat", lat), ("ttft", ttft)):
            v = arr.cpu().numpy()
            assert [int(x) for x in v[::stride]] == w[name + "_samples"], (pol, name)
            assert list(_digests(v)) == w[name + "_digest"], (pol, name)
