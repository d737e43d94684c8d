"""-m gpu parity of the SURVEY.md 8(f) extensions against the oracle, through the C ABI:
preemption under a KV budget, policy switching, TPOT,
the duration-based estimator, P25 and the burst workload."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl
from gpu_util import dev_trace

pytestmark = pytest.mark.gpu
POL = (orc.FCFS, orc.SJF, orc.HRRN)


@pytest.fixture(scope="module")
def asr():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device (there is no CPU fallback)"
    import paper_2603_11273_b200 as m
    return m


def run_ex(asr, traces, replicas, cost, ext_kw, max_slots, summary_only=False):
    """replicas: list of (trace_id, policy, slots) -> (lat list, ttft list, summaries, preempt counts)"""
    import torch
    offs = np.concatenate([[0], np.cumsum([len(t) for t in traces])]).astype(np.int64)
    ns = np.array([len(traces[t]) for t, _, _ in replicas], dtype=np.int64)
    out_off = np.concatenate([[0], np.cumsum(ns)]).astype(np.int64)
    total = int(out_off[-1])
    rep = asr.make_replicas([offs[t] for t, _, _ in replicas], out_off[:-1], ns, [p for _, p, _ in replicas],
                            [s for _, _, s in replicas], 0)
    d_tr, d_rep = dev_trace(np.concatenate(traces)), asr.to_device(rep)
    d_cm, d_ex = asr.to_device(asr.make_cost(*cost)), asr.to_device(asr.make_ext(**ext_kw))
    R = len(replicas)
    d_sum = torch.zeros(R * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    d_pre = torch.full((R,), -5, dtype=torch.int64, device="cuda")
    if summary_only:
        asr.simulate_batched_ex(d_tr, d_rep, R, d_cm, d_ex, 1, total, max_slots, None, None, d_sum, d_pre)
        torch.cuda.synchronize()
        return None, None, d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE), d_pre.cpu().numpy()
    lat = torch.full((max(total, 1),), -7, dtype=torch.int64, device="cuda")
    ttft = torch.full((max(total, 1),), -7, dtype=torch.int64, device="cuda")
    asr.simulate_batched_ex(d_tr, d_rep, R, d_cm, d_ex, 1, total, max_slots, lat, ttft, d_sum, d_pre)
    torch.cuda.synchronize()
    lat, ttft = lat.cpu().numpy(), ttft.cpu().numpy()
    L = [lat[out_off[i]:out_off[i + 1]] for i in range(R)]
    T = [ttft[out_off[i]:out_off[i + 1]] for i in range(R)]
    return L, T, d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE), d_pre.cpu().numpy()


def check_ex(traces, replicas, cost, ext_kw, L, T, S, P, expect_preempt=None):
    cm, ex = orc.cost(*cost), orc.ext(**ext_kw)
    total_pre = 0
    for i, (t, pol, slots) in enumerate(replicas):
        rl, rt, first, end, npre = orc.simulate_ex(traces[t], pol, cm, ex, slots)
        tag = "rep %d pol %d slots %d ext %r" % (i, pol, slots, ext_kw)
        if L is not None:
            assert np.array_equal(L[i], rl), "latency mismatch " + tag
            assert np.array_equal(T[i], rt), "ttft mismatch " + tag
        want = (orc.percentile(rl, 50), orc.percentile(rl, 90), orc.percentile(rt, 50), orc.percentile(rt, 90),
                first, end, len(traces[t]))
        got = tuple(int(S[i][f]) for f in ("p50_e2e_us", "p90_e2e_us", "p50_ttft_us", "p90_ttft_us",
                                           "first_arrival_us", "last_done_us", "n_done"))
        assert got == want, "summary mismatch " + tag
        assert int(P[i]) == npre, "preemption count mismatch " + tag
        total_pre += npre
    if expect_preempt:
        assert total_pre > 0, "the budget never bound: the test does not exercise preemption"


def test_hand_worked_preemption_examples(asr):
    unit = (0, 0, 1000, 0, 0, 1)
    tr1 = orc.make_trace([0, 0], [4000, 4000])
    tr2 = orc.make_trace([0, 0], [4000, 3000])
    tr3 = orc.make_trace([0, 0], [4000, 4000], est=[4000, 2000])
    reps = [(0, orc.FCFS, 2), (1, orc.SJF, 2), (2, orc.HRRN, 2)]
    L, T, S, P = run_ex(asr, [tr1, tr2, tr3], reps, unit, dict(kv_budget=4), 32)
    assert [list(x) for x in L] == [[4000, 8000], [7000, 3000], [8000, 4000]]
    assert [list(x) for x in T] == [[1000, 1000]] * 3 and list(P) == [1, 1, 1]


@pytest.mark.parametrize("slots,max_slots", [(16, 32), (40, 64), (200, 256)])
def test_preemption_on_stress_traces(asr, slots, max_slots):
    traces = [wl.stress_trace("lognormal", 1200, 31, rate_per_s=30.0), wl.stress_trace("burst", 500, 32),
              wl.stress_trace("six", 900, 33, rate_per_s=25.0), wl.stress_trace("misest", 800, 34, rate_per_s=28.0)]
    reps = [(t, p, slots) for t in range(4) for p in POL]
    for ext_kw in (dict(kv_budget=25 * slots, kv_base=20, kv_per_s=2), dict(kv_budget=160 + 12 * slots, kv_base=0, kv_per_s=0)):
        L, T, S, P = run_ex(asr, traces, reps, wl.CONFIG_COST, ext_kw, max_slots)
        check_ex(traces, reps, wl.CONFIG_COST, ext_kw, L, T, S, P, expect_preempt=True)
    _, _, S2, P2 = run_ex(asr, traces, reps, wl.CONFIG_COST, ext_kw, max_slots, summary_only=True)
    assert np.array_equal(S.view(np.uint8), S2.view(np.uint8)) and np.array_equal(P, P2)


def test_extensions_off_match_the_plain_call(asr):
    from gpu_util import run_batched
    traces = [wl.stress_trace("lognormal", 700, 35, rate_per_s=24.0), wl.stress_trace("clumped", 600, 36, rate_per_s=20.0)]
    reps = [(t, p, s) for t in range(2) for p in POL for s in (1, 8, 32)]
    L, T, S, P = run_ex(asr, traces, reps, wl.CONFIG_COST, {}, 32)
    L0, T0, S0 = run_batched(traces, reps, wl.CONFIG_COST, 32)
    for i in range(len(reps)):
        assert np.array_equal(L[i], L0[i]) and np.array_equal(T[i], T0[i])
    assert np.array_equal(S.view(np.uint8), S0.view(np.uint8)) and not P.any()


def test_adaptive_policy(asr):
    traces = [wl.stress_trace("lognormal", 1500, 37, rate_per_s=26.0), wl.stress_trace("uniform", 1000, 38, rate_per_s=13.0)]
    reps = [(t, orc.ADAPTIVE, s) for t in range(2) for s in (4, 16)]
    for ext_kw in (dict(depth1=4, depth2=40, pol=(orc.FCFS, orc.SJF, orc.HRRN)),
                   dict(depth1=2, depth2=2, pol=(orc.FCFS, orc.FCFS, orc.SJF)),
                   dict(depth1=10, depth2=100, pol=(orc.HRRN, orc.SJF, orc.FCFS), kv_budget=700, kv_base=10, kv_per_s=1)):
        L, T, S, P = run_ex(asr, traces, reps, wl.CONFIG_COST, ext_kw, 32)
        check_ex(traces, reps, wl.CONFIG_COST, ext_kw, L, T, S, P)


def test_request_too_large_for_the_budget_flags_the_replica(asr):
    tr = orc.make_trace([0, 10, 20], [3000, 9000, 3000])
    unit = (0, 0, 1000, 0, 0, 1)
    L, T, S, P = run_ex(asr, [tr], [(0, orc.FCFS, 2), (0, orc.SJF, 2)], unit, dict(kv_budget=8), 32)
    assert list(S["n_done"]) == [-1, -1]
    with pytest.raises(ValueError):
        orc.simulate_ex(tr, orc.FCFS, orc.cost(*unit), orc.ext(kv_budget=8), 2)


def test_burst_workload_p25_and_tpot(asr):
    """PAPER.md:202 (A.2): all 500 requests at once; PAPER.md:214 TPOT; PAPER.md:230 P25"""
    import torch
    cfg = wl.burst_config()
    tr = wl.burst_trace(cfg)
    cm = orc.cost(*cfg["cost"])
    d_tr = dev_trace(tr)
    n = len(tr)
    for pol in POL:
        lat, ttft, summ = asr.simulate(d_tr, n, pol, asr.make_cost(*cfg["cost"]), cfg["slots"])
        tp = asr.tpot(d_tr, n, asr.make_cost(*cfg["cost"]), lat, ttft)
        seg = torch.tensor([0, n], dtype=torch.int64, device="cuda")
        pc = asr.percentiles(torch.cat([lat, ttft, tp]), torch.tensor([0, n, 2 * n, 3 * n], dtype=torch.int64,
                                                                        device="cuda"), 3, [25, 50, 90])
        torch.cuda.synchronize()
        rl, rt, _, _ = orc.simulate(tr, pol, cm, cfg["slots"])
        rtp = orc.tpot(tr, cm, rl, rt)
        assert np.array_equal(lat.cpu().numpy(), rl) and np.array_equal(ttft.cpu().numpy(), rt)
        assert np.array_equal(tp.cpu().numpy(), rtp)
        want = [[orc.percentile(v, q) for q in (25, 50, 90)] for v in (rl, rt, rtp)]
        assert pc.cpu().numpy().reshape(3, 3).tolist() == want
        del seg


def test_estimator(asr):
    import torch
    rng = np.random.default_rng(5)
    n = 100003
    tr = orc.make_trace(np.sort(rng.integers(0, 10**9, n)), rng.integers(0, 36000, n), est=rng.integers(-5, 9, n))
    lang = rng.integers(0, 4, n).astype(np.uint8)
    speech = rng.integers(-3, 36000, n).astype(np.int32)
    kap = [5000, 2500, 7321, 1]
    for lg, sp in ((None, None), (lang, None), (lang, speech), (None, speech)):
        d = dev_trace(tr)
        asr.estimate(d, n, kap if lg is not None else kap[:1], None if lg is None else asr.to_device(lg),
                     None if sp is None else asr.to_device(sp))
        torch.cuda.synchronize()
        got = d.cpu().numpy().view(asr.REQ_DTYPE)
        want = orc.estimate(tr, kap if lg is not None else kap[:1], lang=lg, speech_ms=sp)
        assert np.array_equal(got.view(np.uint8), want.view(np.uint8))
    # DESIGN.md E10/E12: est is clamped to the comparator's bound 2^24; an unknown language id reads entry 0
    big = orc.make_trace(np.zeros(6), [2_000_000_000, 1 << 24, (1 << 24) + 1, 8000, 8000, 8000])
    lg6 = np.array([0, 0, 0, 1, 2, 255], dtype=np.uint8)
    for kap2 in ([1_000_000, 2500], [999_999, 5000]):
        d = dev_trace(big)
        asr.estimate(d, 6, kap2, asr.to_device(lg6))
        torch.cuda.synchronize()
        got = d.cpu().numpy().view(asr.REQ_DTYPE)
        want = orc.estimate(big, kap2, lang=lg6)
        assert np.array_equal(got.view(np.uint8), want.view(np.uint8))
        assert got["est"].max() == 1 << 24
    # 8 / 4 / 2 s at kappa = 5 -> 40, 20, 10 tokens
    d = dev_trace(orc.make_trace([0, 0, 0], [8000, 4000, 2000]))
    asr.estimate(d, 3, [5000])
    torch.cuda.synchronize()
    assert list(d.cpu().numpy().view(asr.REQ_DTYPE)["est"]) == [40, 20, 10]


def test_inter_token_latency(asr):
    """weighted nearest-rank percentiles, count and sum of the gap multiset"""
    import torch
    traces = [wl.stress_trace("lognormal", 900, 41, rate_per_s=24.0), wl.burst_trace(),
              wl.stress_trace("uniform", 700, 42, rate_per_s=3.0), orc.make_trace([0], [0]),
              orc.make_trace([0, 500], [3000, 2000])]
    reps = [(t, p, s) for t in range(5) for p in POL for s in (2, 16)] + [(0, orc.SJF, 100), (1, orc.HRRN, 256)]
    offs = np.concatenate([[0], np.cumsum([len(t) for t in traces])]).astype(np.int64)
    ns = np.array([len(traces[t]) for t, _, _ in reps], dtype=np.int64)
    out_off = np.concatenate([[0], np.cumsum(ns)]).astype(np.int64)
    rep = asr.make_replicas([offs[t] for t, _, _ in reps], out_off[:-1], ns, [p for _, p, _ in reps],
                            [s for _, _, s in reps], 0)
    for cost in (wl.CONFIG_COST, (700, 0, 1000, 0, 0, 1), wl.MEDIUM_COST):
        pcts = [1, 25, 50, 90, 99, 100]
        got = asr.itl_batched(dev_trace(np.concatenate(traces)), asr.to_device(rep), len(reps),
                              asr.to_device(asr.make_cost(*cost)), 1, int(out_off[-1]), 256, pcts)
        torch.cuda.synchronize()
        got = got.cpu().numpy()
        for i, (t, pol, slots) in enumerate(reps):
            p, cnt, sm = orc.itl(traces[t], pol, orc.cost(*cost), slots, pcts)
            assert list(got[i]) == p + [cnt, sm], "ITL mismatch rep %d cost %r: %r != %r" % (i, cost, list(got[i]), p + [cnt, sm])
