"""-m gpu: the CUDA simulator (a4+a5+a6) against the oracle, bit-exact, through the C ABI."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl
from gpu_util import check_replica, dev_trace, run_batched

pytestmark = pytest.mark.gpu
POL = (orc.FCFS, orc.SJF, orc.HRRN)


@pytest.fixture(scope="module")
def asr_mod():
    import torch
    assert torch.cuda.is_available()
    import paper_2603_11273_b200 as asr
    return asr


@pytest.fixture(params=["warp", "lane"])
def asr(asr_mod, request):
    """every test runs twice: warp-per-replica only, and thread-per-replica first
    (with hand-over to the warp kernel where SJF/HRRN must choose)"""
    big = 2**31 - 1
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_MIN_REPLICAS, 1 if request.param == "lane" else big)
    yield asr_mod
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_MIN_REPLICAS, 1024)


def test_fig1_toy(asr):
    """PAPER.md:25 on the GPU: FCFS (5, 8, 10) s, SJF (2, 5, 10) s."""
    import torch
    toy = orc.make_trace([0, 0, 0], [8000, 4000, 2000])
    cm = asr.make_cost(*wl.TOY_COST)
    d = dev_trace(toy)
    lat, _, _ = asr.simulate(d, 3, asr.FCFS, cm, 1)
    torch.cuda.synchronize()
    assert lat.cpu().tolist() == [5000000, 8000000, 10000000]
    lat, _, _ = asr.simulate(d, 3, asr.SJF, cm, 1)
    assert lat.cpu().tolist() == [10000000, 5000000, 2000000]
    lat, _, _ = asr.simulate(d, 3, asr.HRRN, cm, 1)
    assert lat.cpu().tolist() == [5000000, 10000000, 7000000]


def test_config1_and_config2(asr, tables):
    c1, c2 = wl.config1(), wl.config2()
    tr1 = orc.gen_trace(c1["seed"], c1["rate_mhz"], c1["dist"], c1["n"], *tables)
    traces = [tr1] + [orc.gen_trace(c2["seed"], r, c2["dist"], c2["n"], *tables) for r in c2["rates_mhz"]]
    reps = [(0, p, c1["slots"]) for p in c1["policies"]]
    reps += [(1 + i, p, c2["slots"]) for i in range(8) for p in c2["policies"]]
    L, T, S = run_batched(traces, reps, wl.CONFIG_COST, 16)
    for i, (t, p, s) in enumerate(reps):
        check_replica(traces[t], p, s, wl.CONFIG_COST, L[i], T[i], S[i], "rep %d" % i)


@pytest.mark.parametrize("kind,rate,n", [("lognormal", 3.6, 2000), ("lognormal", 22.0, 3000),
                                         ("lognormal", 25.0, 3000), ("uniform", 12.0, 3000),
                                         ("burst", 1.0, 500), ("six", 14.0, 2500), ("equal_est", 25.0, 1500),
                                         ("clumped", 1.0, 1500), ("misest", 24.0, 2000)])
def test_stress_traces_all_policies_and_slots(asr, kind, rate, n):
    """S1-S5 of SURVEY.md 8d: overload, bursts and ties, where the policies really differ."""
    tr = wl.stress_trace(kind, n, 7, rate_per_s=rate)
    slot_list = [1, 2, 16, 32] if kind != "burst" else [1, 16, 32]
    reps = [(0, p, s) for s in slot_list for p in POL]
    L, T, S = run_batched([tr], reps, wl.CONFIG_COST, 32)
    differ = False
    for i, (_, p, s) in enumerate(reps):
        check_replica(tr, p, s, wl.CONFIG_COST, L[i], T[i], S[i], "%s slots=%d pol=%d" % (kind, s, p))
    differ = any(not np.array_equal(L[0], L[j]) for j in (1, 2))
    if kind not in ("equal_est",):
        assert differ, "stress trace does not exercise the policy"


@pytest.mark.parametrize("slots", [33, 64, 100, 128, 256])
def test_wide_batches(asr, slots):
    tr = wl.stress_trace("lognormal", 3000, 8, rate_per_s=60.0)
    br = wl.stress_trace("burst", 500, 9)
    reps = [(0, p, slots) for p in POL] + [(1, p, slots) for p in POL]
    L, T, S = run_batched([tr, br], reps, wl.CONFIG_COST, slots)
    for i, (t, p, s) in enumerate(reps):
        check_replica([tr, br][t], p, s, wl.CONFIG_COST, L[i], T[i], S[i], "slots=%d rep=%d" % (slots, i))


def test_mixed_batch_summary_only_and_invalid_descriptors(asr):
    import torch
    rng = np.random.default_rng(1)
    traces = [wl.stress_trace(k, int(n), 100 + i, rate_per_s=r)
              for i, (k, n, r) in enumerate([("lognormal", 1, 5.0), ("lognormal", 33, 30.0), ("uniform", 700, 14.0),
                                             ("burst", 64, 1.0), ("six", 1000, 20.0), ("lognormal", 0, 1.0)])]
    reps = [(t, int(rng.integers(0, 3)), int(rng.choice([1, 3, 8, 32]))) for t in range(6) for _ in range(5)]
    L, T, S = run_batched(traces, reps, wl.CONFIG_COST, 32)
    _, _, S2 = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    for i, (t, p, s) in enumerate(reps):
        if len(traces[t]) == 0:
            assert S[i]["n_done"] == 0 and S[i]["p50_e2e_us"] == -1
            continue
        check_replica(traces[t], p, s, wl.CONFIG_COST, L[i], T[i], S[i], "rep %d" % i)
    assert np.array_equal(S.view(np.uint8), S2.view(np.uint8))
    # invalid descriptors are flagged, the others still run
    tr = traces[2]
    rep = asr.make_replicas([0, 0, 0, 0], [0, 700, 1400, 2100], 700, [0, 9, 1, 2], [8, 8, 0, 64], 0)
    d_sum = torch.zeros(4 * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    asr.simulate_batched(dev_trace(tr), asr.to_device(rep), 4, asr.to_device(asr.make_cost(*wl.CONFIG_COST)), 1,
                         2800, 32, None, None, d_sum)
    torch.cuda.synchronize()
    s = d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)
    assert list(s["n_done"]) == [700, -1, -1, -1]


def test_invalid_descriptor_with_huge_n_does_not_displace_the_others(asr):
    """a descriptor whose n / out_off is out of range sits BEFORE contended SJF/HRRN replicas: it gets
    n_done = -1 and the bitmaps of the replicas behind it stay inside the workspace (they are sized from
    total_requests; the kernels must not trust the n of a descriptor they are going to reject)"""
    import torch
    tr = wl.stress_trace("lognormal", 1500, 31, rate_per_s=26.0)       # overloaded at 8 slots: real choices
    n = len(tr)
    rep = asr.make_replicas([0] * 6, [0, 0, n, 2 * n, 0, 3 * n], [n, 2**31 - 1, n, n, n, n],
                            [orc.FCFS, orc.SJF, orc.SJF, orc.HRRN, orc.HRRN, orc.FCFS], 8, 0)
    rep["out_off"][1] = 2**40                 # out of range as well
    rep["n"][4] = -5                          # negative n
    rep["out_off"][4] = -1
    total = 4 * n
    for summary_only in (False, True):
        d_sum = torch.zeros(6 * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        lat = ttft = None
        if not summary_only:
            lat = torch.full((total,), -7, dtype=torch.int64, device="cuda")
            ttft = torch.full((total,), -7, dtype=torch.int64, device="cuda")
        ws_bytes = asr.workspace_bytes(1, total, 6, 1 if summary_only else 0)
        ws = torch.zeros(ws_bytes + 4096, dtype=torch.uint8, device="cuda")
        ws[ws_bytes:] = 0xA5                  # canary behind the workspace the library was promised
        asr.simulate_batched(dev_trace(tr), asr.to_device(rep), 6, asr.to_device(asr.make_cost(*wl.CONFIG_COST)), 1,
                             total, 8, lat, ttft, d_sum, workspace=ws[:ws_bytes])
        torch.cuda.synchronize()
        assert bool((ws[ws_bytes:] == 0xA5).all()), "wrote past the workspace"
        s = d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)
        assert list(s["n_done"]) == [n, -1, n, n, -1, n]
        for i, pol in ((0, orc.FCFS), (2, orc.SJF), (3, orc.HRRN), (5, orc.FCFS)):
            off = int(rep["out_off"][i])
            check_replica(tr, pol, 8, wl.CONFIG_COST, None if summary_only else lat[off:off + n].cpu().numpy(),
                          None if summary_only else ttft[off:off + n].cpu().numpy(), s[i], "rep %d" % i)


def test_other_cost_models(asr):
    """zero per-running cost, zero encoder, big encoder, token floor"""
    tr = wl.stress_trace("lognormal", 800, 12, rate_per_s=9.0)
    for cost in [(0, 0, 5000, 0, 1, 4), (300000, 0, 20000, 700, 0, 1), (1000, 7, 1, 1, 0, 0),
                 (50000, 1, 12000, 30, 2, 9)]:
        reps = [(0, p, s) for s in (1, 5, 32) for p in POL]
        L, T, S = run_batched([tr], reps, cost, 32)
        for i, (_, p, s) in enumerate(reps):
            check_replica(tr, p, s, cost, L[i], T[i], S[i], "cost=%r" % (cost,))


def test_lane_kernel_hand_overs(asr):
    """cases the thread-per-replica kernel must pass on: a busy period longer than 2^32 us (its
    32-bit proof for order-free outputs fails) and iteration costs beyond 31 bits"""
    toy = (1000000, 0, 100000, 0, 0, 5)           # Fig. 1 cost model: seconds per request
    br = wl.stress_trace("burst", 1500, 21)        # one slot -> ~6000 s of continuous service
    sp = wl.stress_trace("lognormal", 300, 22, rate_per_s=0.5)
    for cost, traces in ((toy, [br]), ((20000, 2, 3_000_000_000, 50, 1, 4), [sp])):
        reps = [(0, p, s) for p in POL for s in (1, 4)]
        L, T, S = run_batched(traces, reps, cost, 32)
        _, _, S2 = run_batched(traces, reps, cost, 32, summary_only=True)
        for i, (t, p, s) in enumerate(reps):
            check_replica(traces[t], p, s, cost, L[i], T[i], S[i], "cost=%r rep %d" % (cost, i))
        assert np.array_equal(S.view(np.uint8), S2.view(np.uint8))


def test_summary_only_long_segments_and_odd_offsets(asr):
    """summary-only calls keep the per-request values in the workspace (uint32, any order, on the
    thread-per-replica path): segments beyond the register-resident percentile path (> 10,240
    values), odd lengths and offsets, light and heavy load, every policy"""
    traces = [wl.stress_trace("lognormal", 12345, 51, rate_per_s=3.0), wl.stress_trace("uniform", 10241, 52, rate_per_s=1.0),
              wl.stress_trace("lognormal", 4099, 53, rate_per_s=21.0), wl.stress_trace("six", 3, 54, rate_per_s=1.0),
              wl.stress_trace("lognormal", 10239, 55, rate_per_s=0.5)]
    reps = [(t, p, s) for t in range(5) for p in POL for s in (7, 32)]
    _, _, S = run_batched(traces, reps, wl.CONFIG_COST, 32, summary_only=True)
    for i, (t, p, s) in enumerate(reps):
        check_replica(traces[t], p, s, wl.CONFIG_COST, None, None, S[i], "rep %d" % i)
