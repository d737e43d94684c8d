"""Pins of the oracle's SURVEY.md 8(f) extensions (-m "not gpu"): preemption under a KV budget
(PAPER.md:285), policy switching on queue depth, TPOT and the
duration-based estimator (Listing 1)."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl

POL = (orc.FCFS, orc.SJF, orc.HRRN)
UNIT = orc.cost(0, 0, 1000, 0, 0, 1)       # 1 ms per iteration, tokens = seconds of audio, no encoder


def test_extensions_off_is_the_base_simulator():
    for kind, n, rate in (("lognormal", 600, 24.0), ("burst", 200, 1.0), ("six", 500, 20.0)):
        tr = wl.stress_trace(kind, n, 7, rate_per_s=rate)
        for pol in POL:
            for slots in (1, 8):
                a = orc.simulate(tr, pol, orc.cost(*wl.CONFIG_COST), slots)
                b = orc.simulate_ex(tr, pol, orc.cost(*wl.CONFIG_COST), orc.ext(), slots)
                assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[2:] == b[2:4]
                assert b[4] == 0


def test_budget_that_never_binds_changes_nothing():
    tr = wl.stress_trace("lognormal", 500, 8, rate_per_s=24.0)
    cm = orc.cost(*wl.CONFIG_COST)
    for pol in POL:
        a = orc.simulate(tr, pol, cm, 8)
        b = orc.simulate_ex(tr, pol, cm, orc.ext(kv_budget=10**9, kv_base=1500, kv_per_s=50), 8)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and b[4] == 0


def test_hand_worked_preemption_fcfs():
    """two 4-token requests, 2 slots, budget 4 tokens: after two iterations (2+2 held) a third
    token each does not fit; FCFS evicts the later one (B), which restarts after A has finished."""
    tr = orc.make_trace([0, 0], [4000, 4000])
    lat, ttft, first, end, npre = orc.simulate_ex(tr, orc.FCFS, UNIT, orc.ext(kv_budget=4), 2)
    assert list(lat) == [4000, 8000] and list(ttft) == [1000, 1000]      # TTFT: first admission
    assert (first, end, npre) == (0, 8000, 1)


def test_hand_worked_preemption_sjf_evicts_the_largest_estimate():
    tr = orc.make_trace([0, 0], [4000, 3000])            # est = dur: A=4000, B=3000
    lat, ttft, _, end, npre = orc.simulate_ex(tr, orc.SJF, UNIT, orc.ext(kv_budget=4), 2)
    assert list(lat) == [7000, 3000] and list(ttft) == [1000, 1000] and (end, npre) == (7000, 1)


def test_hand_worked_preemption_hrrn_evicts_the_lowest_ratio():
    tr = orc.make_trace([0, 0], [4000, 4000], est=[4000, 2000])   # at t=2000: A 0.5, B 1.0 -> A goes
    lat, ttft, _, end, npre = orc.simulate_ex(tr, orc.HRRN, UNIT, orc.ext(kv_budget=4), 2)
    assert list(lat) == [8000, 4000] and list(ttft) == [1000, 1000] and (end, npre) == (8000, 1)


def test_encoder_cache_counts_and_head_of_line_blocks():
    """kv_base 2: a request holds 2 + generated.  Budget 7, two 3-token requests: A (2+0) admitted,
    B needs 2 + (A's 2) + 2 new tokens = 6 <= 7: admitted; after one iteration 3+3=6, one more token
    each = 8 > 7: evict B; A finishes at 3 ms; B restarts alone and finishes at 6 ms."""
    tr = orc.make_trace([0, 0], [3000, 3000])
    lat, ttft, _, end, npre = orc.simulate_ex(tr, orc.FCFS, UNIT, orc.ext(kv_budget=7, kv_base=2), 2)
    assert list(lat) == [3000, 6000] and list(ttft) == [1000, 1000] and npre == 1
    # kv_per_s: 1 unit per second of audio -> 3 + generated each: 3+3+2 = 8 > 7: B is not even admitted
    lat, ttft, _, end, npre = orc.simulate_ex(tr, orc.FCFS, UNIT, orc.ext(kv_budget=7, kv_per_s=1), 2)
    assert list(lat) == [3000, 6000] and list(ttft) == [1000, 4000] and npre == 0


def test_request_that_cannot_fit_alone_is_an_error():
    tr = orc.make_trace([0], [9000])
    with pytest.raises(ValueError):
        orc.simulate_ex(tr, orc.FCFS, UNIT, orc.ext(kv_budget=8), 1)


def test_pressure_invariants_on_a_stress_trace():
    tr = wl.stress_trace("lognormal", 400, 9, rate_per_s=30.0)
    cm = orc.cost(*wl.CONFIG_COST)
    for pol in POL:
        base = orc.simulate(tr, pol, cm, 16)
        lat, ttft, first, end, npre = orc.simulate_ex(tr, pol, cm, orc.ext(kv_budget=400, kv_base=20, kv_per_s=2), 16)
        assert npre > 0 and (lat > 0).all() and (ttft > 0).all() and (ttft <= lat).all()
        assert end >= base[3] and first == base[2]       # recomputation can only cost time
        iso = np.array([orc.enc_cost(cm, int(d)) + orc.tokens(cm, int(d)) * (8000 + 50) for d in tr["dur_ms"]])
        assert (lat >= iso).all()


def test_adaptive_policy_reduces_to_the_pure_policies():
    tr = wl.stress_trace("lognormal", 500, 10, rate_per_s=26.0)
    cm = orc.cost(*wl.CONFIG_COST)
    for pol in POL:
        want = orc.simulate(tr, pol, cm, 8)
        for e in (orc.ext(depth1=0, depth2=0, pol=(0, 0, pol)),               # always the deep branch
                  orc.ext(depth1=10**6, depth2=10**6, pol=(pol, 0, 0)),       # always the shallow branch
                  orc.ext(depth1=0, depth2=10**6, pol=(0, pol, 0)),
                  orc.ext(depth1=5, depth2=50, pol=(pol, pol, pol))):
            got = orc.simulate_ex(tr, orc.ADAPTIVE, cm, e, 8)
            assert np.array_equal(want[0], got[0]) and np.array_equal(want[1], got[1])
    # and a genuinely mixed rule differs from all three
    mixed = orc.simulate_ex(tr, orc.ADAPTIVE, cm, orc.ext(depth1=4, depth2=40, pol=(orc.FCFS, orc.SJF, orc.HRRN)), 8)
    assert all(not np.array_equal(mixed[0], orc.simulate(tr, pol, cm, 8)[0]) for pol in POL)


def test_tpot_closed_form_and_single_token():
    cm = orc.cost(*wl.CONFIG_COST)
    tr = orc.make_trace([0, 10**9, 2 * 10**9], [6000, 35000, 0])       # isolated requests; 0 ms -> 1 token
    lat, ttft, _, _ = orc.simulate(tr, orc.FCFS, cm, 4)
    tp = orc.tpot(tr, cm, lat, ttft)
    assert list(tp) == [8050, 8050, -1]          # alone: every further token costs 8,000 + 50*1 us
    assert (lat[0] - ttft[0]) == 24 * 8050


def test_estimator_fig1_tokens_and_floor():
    """8/4/2 s at kappa = 5 tokens/s -> 40, 20 and 10 tokens; max(1, int(.))"""
    tr = orc.make_trace([0, 0, 0, 0, 0], [8000, 4000, 2000, 100, 399], est=[7, 7, 7, 7, 7])
    out = orc.estimate(tr, [5000])
    assert list(out["est"]) == [40, 20, 10, 1, 1]
    assert list(out["dur_ms"]) == [8000, 4000, 2000, 100, 399]           # only est changes
    out = orc.estimate(tr, [5000, 2500], lang=[0, 1, 1, 0, 1])
    assert list(out["est"]) == [40, 10, 5, 1, 1]
    out = orc.estimate(tr, [5000], speech_ms=[4000, 4000, 0, 100, 1000])  # VAD: speech-active duration
    assert list(out["est"]) == [20, 20, 1, 1, 5]


def test_estimator_clamp_and_unknown_language():
    """DESIGN.md readings E10/E12: est never leaves the comparator's documented range [1, 2^24]
    (asr_sched.h: wait * est < 2^62), and a language id without a table entry uses entry 0."""
    tr = orc.make_trace([0, 0, 0], [2_000_000_000, 16_777_216, 16_777_217])
    out = orc.estimate(tr, [1_000_000])                  # kappa = 1000 tokens/s: est = d_ms
    assert list(out["est"]) == [1 << 24, 1 << 24, 1 << 24]
    out = orc.estimate(tr, [999_999])
    assert list(out["est"]) == [1 << 24, 16_777_199, 16_777_200]
    tr = orc.make_trace([0, 0, 0], [8000, 8000, 8000])
    out = orc.estimate(tr, [5000, 2500], lang=[1, 2, 255])
    assert list(out["est"]) == [20, 40, 40]


def test_itl_isolated_and_two_overlapping_requests():
    """PAPER.md:214.  Alone, every gap is 8,000 + 50 us: a 6 s request (25 tokens) has 24 of them.
    Unit model (1 ms iterations, no encoder), two slots: A (3 tokens) at t=0, B (2 tokens) arrives at
    500 us and is admitted at 1000: iterations [0,1000) A first token; [1000,2000) A gap, B first
    token; [2000,3000) A gap + B gap.  Three gaps of 1000."""
    cm = orc.cost(*wl.CONFIG_COST)
    p, cnt, sm = orc.itl(orc.make_trace([0], [6000]), orc.FCFS, cm, 4, [1, 50, 100])
    assert (p, cnt, sm) == ([8050, 8050, 8050], 24, 24 * 8050)
    p, cnt, sm = orc.itl(orc.make_trace([0, 500], [3000, 2000]), orc.FCFS, UNIT, 2, [50])
    assert (p, cnt, sm) == ([1000], 3, 3000)
    # an encoder stall is felt by the requests already running: A (3 tokens) alone, then B admitted
    enc = orc.cost(700, 0, 1000, 0, 0, 1)
    p, cnt, sm = orc.itl(orc.make_trace([0, 500], [3000, 2000]), orc.FCFS, enc, 2, [1, 100])
    assert (p, cnt, sm) == ([1000, 1700], 3, 1000 + 1700 + 1000)
    assert orc.itl(orc.make_trace([0], [0]), orc.FCFS, cm, 1, [50]) == ([-1], 0, 0)       # one token: no gap


def test_itl_sum_is_the_decode_time_of_all_requests():
    tr = wl.stress_trace("lognormal", 400, 11, rate_per_s=24.0)
    cm = orc.cost(*wl.CONFIG_COST)
    for pol in POL:
        lat, ttft, _, _ = orc.simulate(tr, pol, cm, 8)
        p, cnt, sm = orc.itl(tr, pol, cm, 8, [25, 50, 90])
        assert sm == int((lat - ttft).sum())
        assert cnt == sum(orc.tokens(cm, int(d)) - 1 for d in tr["dur_ms"])
        assert p[0] <= p[1] <= p[2] and p[0] >= 8000 + 50
