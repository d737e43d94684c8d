"""-m gpu: the time-split thread-per-replica tier (units, repair, redo) and the carried-window percentile
kernel of summary-only calls, against the oracle and against the same call with the split switched off.

DESIGN.md "time-split units": a lightly loaded replica is cut into segments that are simulated side by side
as traces of their own; boundaries are stitched at regeneration points (server empty at an arrival).  The
results must not depend on any of it (tolerance 0, PAPER.md:100 percentiles by nearest rank)."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl
from gpu_util import check_replica, run_batched

pytestmark = pytest.mark.gpu
POL = (orc.FCFS, orc.SJF, orc.HRRN)


@pytest.fixture()
def asr():
    import torch
    assert torch.cuda.is_available()
    import paper_2603_11273_b200 as asr_mod
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_MIN_REPLICAS, 1)
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_SPLIT, 1)
    yield asr_mod
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_MIN_REPLICAS, 1024)
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_SPLIT, 1)


def _trace(arr, dur, est=None):
    t = np.zeros(len(arr), dtype=orc.REQ)
    t["arrival_us"] = arr
    t["dur_ms"] = dur
    t["est"] = dur if est is None else est
    return t


def _oracle_summary(tr, pol, slots, cost):
    rl, rt, first, end = orc.simulate(tr, pol, orc.cost(*cost), slots)
    return (orc.percentile(rl, 50), orc.percentile(rl, 90), orc.percentile(rt, 50), orc.percentile(rt, 90),
            first, end, len(tr))


def _check_all(traces, reps, S, cost, tag):
    cache = {}
    for i, (t, p, s) in enumerate(reps):
        key = (t, p, s)
        if key not in cache:
            cache[key] = _oracle_summary(traces[t], p, s, cost)
        got = tuple(int(S[i][f]) for f in ("p50_e2e_us", "p90_e2e_us", "p50_ttft_us", "p90_ttft_us",
                                           "first_arrival_us", "last_done_us", "n_done"))
        assert got == cache[key], "%s: replica %d (trace %d policy %d slots %d): %r != %r" % (
            tag, i, t, p, s, got, cache[key])


def test_split_equals_unsplit_and_oracle(asr):
    """loads from 0.05 to ~8 Erlangs around the split threshold, several lengths (whole and ragged last
    segments), slots 4/16/32, every policy: split on == split off == oracle"""
    specs = [("lognormal", 2500, 0.4), ("lognormal", 4099, 2.0), ("lognormal", 6000, 6.0), ("lognormal", 3000, 11.0),
             ("uniform", 2600, 1.0), ("uniform", 5003, 3.5), ("uniform", 2500, 6.5), ("six", 2777, 4.0),
             ("lognormal", 2500, 26.0), ("misest", 3100, 8.0), ("equal_est", 2560, 9.0), ("lognormal", 2499, 3.0)]
    traces = [wl.stress_trace(k, n, 300 + i, rate_per_s=r) for i, (k, n, r) in enumerate(specs)]
    reps = [(t, p, s) for t in range(len(traces)) for p in POL for s in (4, 16, 32)]
    _, _, S1 = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    asr.set_option(asr.OPT_SIM_LANE_SPLIT, 0)
    _, _, S0 = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    assert np.array_equal(S1.view(np.uint8), S0.view(np.uint8)), "split on/off differ"
    _check_all(traces, reps, S1, wl.CONFIG_COST, "split")


def test_bursty_boundaries_and_unstitchable_replicas(asr):
    """segment boundaries that fall inside busy periods: (a) clustered arrivals at a low average load, so that
    most boundaries need a repair over many requests; (b) one huge burst in the middle of a light trace: the
    repair finds no common regeneration point inside the next segment and the replica is redone in one piece
    (SJF/HRRN then have to choose and go on to the warp kernel)"""
    rng = np.random.Generator(np.random.PCG64(77))
    traces = []
    for j in range(4):   # (a)
        n = 5200 + 37 * j
        sizes = rng.geometric(1.0 / (4 + 3 * j), size=n)
        gaps = rng.exponential(2.5e6 * (1 + j), size=n).astype(np.int64)
        arr, t = [], 0
        for sz, g in zip(sizes, gaps):
            t += int(g)
            arr.extend(t + np.sort(rng.integers(0, 200000, size=sz)))
            if len(arr) >= n:
                break
        traces.append(_trace(np.sort(np.asarray(arr[:n], dtype=np.int64)), rng.integers(1000, 20001, size=n)))
    for j in range(2):   # (b)
        n = 6400
        arr = np.cumsum(rng.exponential(1.5e6, size=n).astype(np.int64))
        arr[2000:2000 + 1500 * (j + 1)] = arr[2000]      # 1500 / 3000 requests at one instant
        arr = np.maximum.accumulate(arr)
        traces.append(_trace(arr, rng.integers(1000, 9001, size=n)))
    reps = [(t, p, s) for t in range(len(traces)) for p in POL for s in (8, 32)]
    _, _, S1 = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    asr.set_option(asr.OPT_SIM_LANE_SPLIT, 0)
    _, _, S0 = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    assert np.array_equal(S1.view(np.uint8), S0.view(np.uint8)), "split on/off differ"
    _check_all(traces, reps, S1, wl.CONFIG_COST, "bursty")


def test_pieces_in_32_bit_times(asr):
    """the 32-bit clock of the pieces (an offset from an epoch that moves at idle arrivals) and the limits that send a
    replica back to the 64-bit code: (a) gaps of 20 minutes to 3 hours between arrivals (epoch moves; arrivals 2^32 us
    past the epoch), a trace that starts before t = 0 and one far from it (2^45 us); (b) a cost model whose encoder
    pass or whose iteration is outside the 32-bit budget, one with 10^5 us iterations, one that costs nothing; (c) busy
    periods of more than 2^31 us, one with requests that wait longer than 2^30 us and one without"""
    rng = np.random.Generator(np.random.PCG64(123))
    n = 2600
    gaps = rng.exponential(2.0e6, size=n).astype(np.int64)
    gaps[::97] += rng.integers(1_200_000_000, 11_000_000_000, size=len(gaps[::97]))   # 20 min .. 3 h
    arr = np.cumsum(gaps)
    dur = rng.integers(1000, 35001, size=n)
    traces = [_trace(arr, dur), _trace(arr - 5_000_000_000, dur), _trace(arr + (1 << 45), dur)]
    reps = [(t, p, s) for t in range(len(traces)) for p in POL for s in (4, 32)]
    _, _, S1 = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    _check_all(traces, reps, S1, wl.CONFIG_COST, "gaps")
    # (b)
    light = [wl.stress_trace("lognormal", 2700, 500, rate_per_s=0.5), wl.stress_trace("uniform", 5000, 501, rate_per_s=0.2)]
    reps = [(t, p, 32) for t in range(len(light)) for p in POL]
    for cost in ((20000, 30000, 8000, 50, 1, 4), (1 << 30, 0, 8000, 50, 1, 4), wl.TOY_COST, (0, 0, 0, 0, 1, 0),
                 (20000, 2, 1 << 26, 50, 1, 4)):
        _, _, S1 = run_batched(light, reps, cost, 32, summary_only=True)
        _check_all(light, reps, S1, cost, "cost %r" % (cost,))
    # (c) 2,700 requests over 2,700 s, ~20 s of service each under the toy cost model: the server never empties
    busy = [_trace(np.arange(2700, dtype=np.int64) * 1_000_000, rng.integers(20000, 30001, size=2700))]
    reps = [(0, p, 32) for p in POL]
    _, _, S1 = run_batched(busy, reps, wl.TOY_COST, 32, summary_only=True)
    _check_all(busy, reps, S1, wl.TOY_COST, "busy")
    # the same arrivals with a cheap encoder: ~12 requests running at any time, nobody waits, the server never
    # empties for 45 minutes (the epoch moves while the server is busy)
    steady = (20000, 0, 100000, 0, 0, 5)
    _, _, S1 = run_batched(busy, reps, steady, 32, summary_only=True)
    _check_all(busy, reps, S1, steady, "steady")


def test_carried_window_percentiles(asr):
    """1,500 replicas in runs and alternations of very different traces (the carried window of the percentile
    kernel hits, misses either way, overflows its slots and re-seeds), all values equal, lengths that are
    not whole quads (radix path through the miss list)"""
    rng = np.random.Generator(np.random.PCG64(5))
    n = 2560
    spaced = np.arange(n, dtype=np.int64) * 40_000_000          # one request every 40 s: isolated requests
    traces = [
        _trace(spaced, np.full(n, 6000)),                                     # every latency identical
        _trace(spaced, rng.integers(1000, 1100, size=n)),                     # a few hundred distinct values
        _trace(spaced, rng.integers(1000, 35001, size=n)),                    # wide
        wl.stress_trace("lognormal", n, 401, rate_per_s=1.0),
        wl.stress_trace("lognormal", n, 402, rate_per_s=1.0),                 # a neighbour of the one before
        wl.stress_trace("uniform", n, 403, rate_per_s=3.0),
        wl.stress_trace("lognormal", 2558, 404, rate_per_s=2.0),              # not whole quads
        wl.stress_trace("six", n, 405, rate_per_s=0.3),                       # six durations: massive ties
        _trace(spaced[:2500], np.where(np.arange(2500) % 2 == 0, 1000, 35000)),   # two values, p50 on the edge
    ]
    order = []
    for rep_len in (40, 1, 7, 2):           # runs of a trace, then strict alternation, ...
        for t in range(len(traces)):
            order += [t] * rep_len
    order = (order * 4)[:1500]
    reps = [(t, POL[i % 3], 32) for i, t in enumerate(order)]
    _, _, S = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    _check_all(traces, reps, S, wl.CONFIG_COST, "windows")


def test_warp_tier_window_beyond_the_chunk_ring(asr):
    """the warp tier with escalation switched off: a burst leaves a window of 7,000 requests, more than the ring of
    chunk bounds covers (plain scans), which then shrinks back into the ring (bounds rebuilt, branch and bound),
    while new arrivals keep joining; SJF and HRRN, per-request outputs"""
    rng = np.random.Generator(np.random.PCG64(99))
    n = 9000
    arr = np.concatenate([np.zeros(7000, dtype=np.int64),
                          np.cumsum(rng.exponential(400000.0, size=n - 7000).astype(np.int64))])
    tr = _trace(arr, rng.integers(1000, 12001, size=n))
    big = 2**31 - 1
    asr.set_option(asr.OPT_SIM_LANE_MIN_REPLICAS, big)
    asr.set_option(asr.OPT_SIM_ESCALATE_WINDOW, big)
    try:
        reps = [(0, orc.SJF, 8), (0, orc.HRRN, 8), (0, orc.HRRN, 32)]
        L, T, S = run_batched([tr], reps, wl.CONFIG_COST, 32)
        for i, (t, p, s) in enumerate(reps):
            check_replica(tr, p, s, wl.CONFIG_COST, L[i], T[i], S[i], "rep %d" % i)
    finally:
        asr.set_option(asr.OPT_SIM_ESCALATE_WINDOW, 4096)


def test_cost_models_mixed_in_one_batch(asr):
    """replica.cm_id: neighbouring lanes of a warp run different cost models (one of them outside the 32-bit budget of
    the pieces, one invalid id) -- summary-only (time-split pieces) and per-request outputs (one thread / one warp per
    replica), against the oracle replica by replica"""
    import torch
    from gpu_util import dev_trace
    costs = [wl.CONFIG_COST, wl.MEDIUM_COST, (20000, 30000, 8000, 50, 1, 4), (5000, 1, 3000, 20, 2, 7), wl.TOY_COST]
    traces = [wl.stress_trace("lognormal", 2600, 700, rate_per_s=1.5), wl.stress_trace("uniform", 4100, 701, rate_per_s=3.0),
              wl.stress_trace("six", 2500, 702, rate_per_s=0.4), wl.stress_trace("lognormal", 3000, 703, rate_per_s=9.0)]
    reps = [(t, p, s, c) for t in range(len(traces)) for p in POL for s in (8, 32) for c in range(len(costs))]
    reps.insert(7, (1, orc.SJF, 32, len(costs)))   # cm_id out of range: n_done = -1, nothing else
    offs = np.concatenate([[0], np.cumsum([len(t) for t in traces])]).astype(np.int64)
    ns = np.array([len(traces[t]) for t, _, _, _ in reps], dtype=np.int64)
    out_off = np.concatenate([[0], np.cumsum(ns)]).astype(np.int64)
    total = int(out_off[-1])
    rep = asr.make_replicas([offs[t] for t, _, _, _ in reps], out_off[:-1], ns, [p for _, p, _, _ in reps],
                            [s for _, _, s, _ in reps], [c for _, _, _, c in reps])
    d_tr, d_rep = dev_trace(np.concatenate(traces)), asr.to_device(rep)
    d_cm = asr.to_device(np.concatenate([asr.make_cost(*c) for c in costs]))
    cache = {}

    def want(i):
        t, p, s, c = reps[i]
        if (t, p, s, c) not in cache:
            cache[(t, p, s, c)] = _oracle_summary(traces[t], p, s, costs[c])
        return cache[(t, p, s, c)]

    fields = ("p50_e2e_us", "p90_e2e_us", "p50_ttft_us", "p90_ttft_us", "first_arrival_us", "last_done_us", "n_done")
    for summary_only in (True, False):
        d_sum = torch.zeros(len(reps) * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        lat = None if summary_only else torch.full((total,), -7, dtype=torch.int64, device="cuda")
        ttft = None if summary_only else torch.full((total,), -7, dtype=torch.int64, device="cuda")
        asr.simulate_batched(d_tr, d_rep, len(reps), d_cm, len(costs), total, 32, lat, ttft, d_sum)
        torch.cuda.synchronize()
        S = d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)
        for i in range(len(reps)):
            if reps[i][3] >= len(costs):
                assert int(S[i]["n_done"]) == -1
                continue
            got = tuple(int(S[i][f]) for f in fields)
            assert got == want(i), "summary_only=%r replica %d %r: %r != %r" % (summary_only, i, reps[i], got, want(i))
        if not summary_only:
            L, T = lat.cpu().numpy(), ttft.cpu().numpy()
            for i in (0, 13, 31, 58, len(reps) - 1):
                t, p, s, c = reps[i]
                rl, rt, _, _ = orc.simulate(traces[t], p, orc.cost(*costs[c]), s)
                assert np.array_equal(L[out_off[i]:out_off[i + 1]], rl) and np.array_equal(T[out_off[i]:out_off[i + 1]], rt), i


def test_stream_percentiles_on_long_and_ragged_segments(asr):
    """summary_stream_kernel (one warp per value stream) on segments longer than the register-resident
    radix path takes (12,000 / 30,004 / 70,000 values: 12 to 69 chunks of 1,024 keys, ragged last chunks), a length that
    is not a multiple of four (radix path through the miss list) and short ones, enough replicas for several runs of
    24 work items with shared seeds"""
    specs = [("lognormal", 12000, 1.0), ("uniform", 30004, 2.0), ("lognormal", 30002, 0.7), ("six", 12000, 0.5),
             ("lognormal", 2500, 3.0), ("uniform", 1028, 1.0), ("lognormal", 70000, 1.5)]
    traces = [wl.stress_trace(k, n, 800 + i, rate_per_s=r) for i, (k, n, r) in enumerate(specs)]
    reps = [(t, p, s) for _ in range(12) for t in range(len(traces)) for p in POL for s in (16, 32)]
    _, _, S = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    _check_all(traces, reps, S, wl.CONFIG_COST, "long")


def test_stream_percentiles_tiny_segments_and_high_bit_values(asr):
    """(a) replicas of 4 ... 2,052 requests (segments shorter than a chunk of 1,024 keys, one key per lane or fewer) mixed
    in one batch; (b) FCFS replicas whose latencies run up to 3.1e9 us in a busy period just short of 2^32 us: uint32 keys with the high bit set (p90 above
    2^31, p50 below), several runs of them"""
    rng = np.random.Generator(np.random.PCG64(321))
    lens = [4, 8, 12, 100, 1000, 1024, 1028, 2048, 2052, 36]
    traces = [wl.stress_trace("lognormal", n, 900 + i, rate_per_s=1.0 + 0.3 * (i % 4)) for i, n in enumerate(lens)]
    reps = [(t, p, 32) for _ in range(6) for t in range(len(traces)) for p in POL]
    _, _, S = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    _check_all(traces, reps, S, wl.CONFIG_COST, "tiny")
    # (b) one request per second, ~16 s of service each, 4 slots: the last request waits 3,100 s
    slow = [_trace(np.arange(1000, dtype=np.int64) * 1_000_000, rng.integers(20000, 30001, size=1000)) for _ in range(3)]
    reps = [(t, orc.FCFS, 4) for _ in range(12) for t in range(len(slow))]
    _, _, S = run_batched(slow, reps, wl.TOY_COST, 32, summary_only=True)
    assert int(S[0]["p90_e2e_us"]) > 2**31 > int(S[0]["p50_e2e_us"]) > 0
    _check_all(slow, reps, S, wl.TOY_COST, "high bit")
