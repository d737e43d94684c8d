"""Pins for the oracle simulator."""
import itertools
import os

import numpy as np
import pytest

import oracle as orc
import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden", "fig1_toy.txt")
CFG = orc.cost(*wl.CONFIG_COST)
TOY = orc.cost(*wl.TOY_COST)
POL = (orc.FCFS, orc.SJF, orc.HRRN)


def _gold():
    g = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        g[tok[0]] = [float(x) if "." in x else int(x) for x in tok[1:]]
    return g


def test_fig1_toy_example():
    """FCFS (5+8+10)/3 = 7.66 s, SJF (2+5+10)/3 = 5.66 s, 1.4x."""
    g = _gold()
    toy = orc.make_trace([0, 0, 0], [8000, 4000, 2000])
    assert [orc.tokens(TOY, d) for d in (8000, 4000, 2000)] == [40, 20, 10]
    lat_f, ttft_f, _, end_f = orc.simulate(toy, orc.FCFS, TOY, 1)
    lat_s, _, _, end_s = orc.simulate(toy, orc.SJF, TOY, 1)
    assert list(lat_f) == g["fcfs"] and list(lat_s) == g["sjf"]
    assert sorted(lat_f) == [5000000, 8000000, 10000000]
    assert sorted(lat_s) == [2000000, 5000000, 10000000]
    # the paper prints the means truncated to two decimals
    assert int(lat_f.sum() / 3 / 1e4) / 100 == g["mean_fcfs_s"][0]
    assert int(lat_s.sum() / 3 / 1e4) / 100 == g["mean_sjf_s"][0]
    assert round(lat_f.sum() / lat_s.sum(), 1) == g["ratio"][0]
    assert end_f == end_s == 10000000
    # derived under the same rules: HRRN picks R1 (all waits 0
    # -> index), then R3 (5e6/2000 > 5e6/4000)
    lat_h, _, _, _ = orc.simulate(toy, orc.HRRN, TOY, 1)
    assert list(lat_h) == [5000000, 10000000, 7000000]
    assert list(ttft_f) == [1100000, 6100000, 9100000]


def service_us(cm_tuple, d, running=1):
    eb, ep, ib, ip, tb, tp = cm_tuple
    tok = max(1, tb + (tp * d) // 1000)
    return eb + ep * d + tok * (ib + ip * running)


@pytest.mark.parametrize("n", [2, 3, 5, 7, 8])
def test_sjf_minimises_mean_completion_bruteforce(n):
    """PAPER.md:63 'minimizes the average waiting time': brute force over all
    n! serving orders of n simultaneous arrivals on one slot.  The completion
    times of an order are cumulative sums of closed-form service times."""
    rng = np.random.default_rng(100 + n)
    dur = rng.choice(np.arange(1000, 35001), size=n, replace=False)
    svc = [service_us(wl.CONFIG_COST, int(d)) for d in dur]
    best = min(sum(itertools.accumulate(svc[i] for i in order))
               for order in itertools.permutations(range(n)))
    tr = orc.make_trace(np.zeros(n), dur)
    lat, _, _, end = orc.simulate(tr, orc.SJF, CFG, 1)
    assert int(lat.sum()) == best
    assert end == sum(svc)
    lat_f, _, _, _ = orc.simulate(tr, orc.FCFS, CFG, 1)
    assert int(lat_f.sum()) == sum(itertools.accumulate(svc))  # index order
    assert int(lat_f.sum()) >= best


def test_one_slot_makespan_and_work_equal_across_policies():
    tr = wl.stress_trace("lognormal", 400, 21, rate_per_s=3.6)  # S1: 97% of 1-slot capacity
    ends, sums = [], []
    for pol in POL:
        lat, ttft, first, end = orc.simulate(tr, pol, CFG, 1)
        ends.append(end)
        # service = completion - start; start = ttft-time minus (enc + 1 iter)
        start = tr["arrival_us"] + ttft - (20000 + 2 * tr["dur_ms"] + 8050)
        sums.append(int((tr["arrival_us"] + lat - start).sum()))
        assert first == tr["arrival_us"][0]
    assert len(set(ends)) == 1 and len(set(sums)) == 1
    assert sums[0] == sum(service_us(wl.CONFIG_COST, int(d)) for d in tr["dur_ms"])
    # and the policies really differ on this trace
    a = orc.simulate(tr, orc.FCFS, CFG, 1)[0]
    b = orc.simulate(tr, orc.SJF, CFG, 1)[0]
    assert not np.array_equal(a, b) and b.mean() < a.mean()


def test_hrrn_equal_est_equals_fcfs_in_simulation():
    tr = wl.stress_trace("equal_est", 600, 22, rate_per_s=25.0)
    for slots in (1, 4, 16):
        a = orc.simulate(tr, orc.FCFS, CFG, slots)
        b = orc.simulate(tr, orc.HRRN, CFG, slots)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[3] == b[3]


@pytest.mark.parametrize("d,e2e,ttft", [(1000, 62250, 30050), (6000, 233250, 40050),
                                        (35000, 1225050, 98050)])
def test_isolated_request_closed_form(d, e2e, ttft):
    # E2E = 20,000 + 2d + tokens * 8,050 ; TTFT = 20,000 + 2d + 8,050
    for pol in POL:
        lat, tt, first, end = orc.simulate(orc.make_trace([12345], [d]), pol, CFG, 16)
        assert (int(lat[0]), int(tt[0])) == (e2e, ttft)
        assert first == 12345 and end == 12345 + e2e


def test_widely_spaced_arrivals_hit_closed_form():
    rng = np.random.default_rng(4)
    dur = rng.integers(1000, 35001, size=50)
    tr = orc.make_trace(np.arange(50) * 5_000_000 + 17, dur)
    want = np.array([service_us(wl.CONFIG_COST, int(d)) for d in dur])
    for pol in POL:
        lat, tt, _, _ = orc.simulate(tr, pol, CFG, 3)
        assert np.array_equal(lat, want)
        assert np.array_equal(tt, 20000 + 2 * dur + 8050)


def test_burst_with_enough_slots_closed_form():
    # slots >= n: everything is admitted in iteration 1 whatever the policy;
    # iteration j costs 8000 + 50 * #{i : tokens_i >= j}
    rng = np.random.default_rng(5)
    n = 40
    dur = rng.integers(1000, 35001, size=n)
    tok = 1 + (4 * dur) // 1000
    tr = orc.make_trace(np.zeros(n), dur)
    t, end_at = 0, {}
    for j in range(1, tok.max() + 1):
        running = int((tok >= j).sum())
        t += 8000 + 50 * running + (int((20000 + 2 * dur).sum()) if j == 1 else 0)
        end_at[j] = t
    for pol in POL:
        lat, tt, _, end = orc.simulate(tr, pol, CFG, 64)
        assert np.array_equal(lat, np.array([end_at[int(k)] for k in tok]))
        assert (tt == end_at[1]).all() and end == end_at[int(tok.max())]


def test_two_slot_hand_worked():
    # A(0,1000ms,5tok) B(0,2000ms,9tok) C(0,1000ms,5tok), 2 slots, FCFS.
    # it1: admit A,B  t = 22000+24000+8100 = 54100  (ttft A,B)
    # it2-5: 4 x 8100 -> 86500  A done
    # it6: admit C    t = 86500+22000+8100 = 116600 (ttft C; B has 6 tokens)
    # it7-9: 3 x 8100 -> 140900 B done (C has 4)
    # it10: 8050 -> 148950 C done
    tr = orc.make_trace([0, 0, 0], [1000, 2000, 1000])
    lat, tt, _, end = orc.simulate(tr, orc.FCFS, CFG, 2)
    assert list(lat) == [86500, 140900, 148950]
    assert list(tt) == [54100, 54100, 116600]
    assert end == 148950


def test_arrival_on_boundary_is_ingested_and_late_one_waits():
    # S13: arrival == t at a boundary joins that step; one microsecond later waits
    one = service_us(wl.CONFIG_COST, 1000)            # 62250
    tr = orc.make_trace([0, 30050], [1000, 1000])     # boundary after iteration 1
    lat, tt, _, _ = orc.simulate(tr, orc.FCFS, CFG, 4)
    assert int(tt[1]) == 22000 + 8100                 # admitted at t = 30050
    tr = orc.make_trace([0, 30051], [1000, 1000])
    lat, tt, _, _ = orc.simulate(tr, orc.FCFS, CFG, 4)
    assert int(tt[1]) == (30050 + 8050 - 30051) + 22000 + 8100
    # A: it1 30050, it2 38100 (B joins), it3 +22000+8100, it4, it5 +8100 each
    assert int(lat[0]) == one + 22000 + 3 * 50        # stalled by B's encoder, 3 shared iterations


@pytest.mark.parametrize("kind,slots,rate", [("lognormal", 16, 25.0), ("uniform", 16, 12.0),
                                             ("burst", 16, 0), ("six", 8, 9.0),
                                             ("misest", 4, 6.0)])
def test_conservation_invariants(kind, slots, rate):
    tr = wl.stress_trace(kind, 700, 31, rate_per_s=rate or 1.0)
    iso = np.array([service_us(wl.CONFIG_COST, int(d)) for d in tr["dur_ms"]])
    outs = {}
    for pol in POL:
        lat, tt, first, end = orc.simulate(tr, pol, CFG, slots)
        assert (lat > 0).all() and (tt > 0).all() and (tt <= lat).all()
        assert (lat >= iso).all()              # nobody beats the isolated closed form
        assert end == int((tr["arrival_us"] + lat).max())
        outs[pol] = lat
    # overload: the policies must actually differ, SJF has the lowest median
    assert not np.array_equal(outs[orc.FCFS], outs[orc.SJF])
    assert np.median(outs[orc.SJF]) <= np.median(outs[orc.FCFS])


def test_empty_trace_and_bad_args():
    lat, tt, first, end = orc.simulate(orc.make_trace([], []), orc.SJF, CFG, 4)
    assert lat.size == 0 and end == 0
    with pytest.raises(ValueError):
        orc.simulate(orc.make_trace([0], [1000]), orc.SJF, CFG, 0)
