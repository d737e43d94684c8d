"""-m gpu: parity at the arithmetic bounds the boundary documents (include/asr_sched.h: wait < 2^38 us,
est <= 2^24, so wait * est < 2^62).  PAPER.md:282 divides floats; north_star wants the ratio "compared exactly
by 64-bit integer cross-multiplication".  The CUDA path orders candidates by the IEEE double quotient and lets
the exact integer comparator decide only when two quotients are equal, so the cases here are built so that the
doubles TIE while the integer cross-products differ by exactly one -- through the standalone select (pair
alone; pair planted across rank k of a 4,096-record queue) and through the simulator's admit step on every
tier (thread, warp, CTA), plus random inputs that fill the whole documented range.  The oracle compares in
128 bits and would return -4 if an input left the documented range (tests/test_oracle_select.py)."""
import math

import numpy as np
import pytest

import oracle as orc
import workloads as wl
from gpu_util import check_replica, run_batched

pytestmark = pytest.mark.gpu
POL = (orc.FCFS, orc.SJF, orc.HRRN)
E_MAX = 1 << 24
T_MAX = (1 << 38) - 1


@pytest.fixture(scope="module")
def asr_mod():
    import torch
    assert torch.cuda.is_available()
    import paper_2603_11273_b200 as asr
    return asr


@pytest.fixture(params=["lane", "warp", "cta"])
def asr_tier(asr_mod, request):
    """lane: thread per replica first (hands SJF/HRRN to the warp kernel at the first real choice);
    warp: warp per replica, never escalates; cta: warp kernel hands over at the first real choice"""
    big = 2**31 - 1
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_MIN_REPLICAS, 1 if request.param == "lane" else big)
    asr_mod.set_option(asr_mod.OPT_SIM_ESCALATE_WINDOW, 0 if request.param == "cta" else big)
    yield asr_mod
    asr_mod.set_option(asr_mod.OPT_SIM_LANE_MIN_REPLICAS, 1024)
    asr_mod.set_option(asr_mod.OPT_SIM_ESCALATE_WINDOW, 4096)


def near_tie_pair(rng, w_cap=T_MAX):
    """(w_a, e_a, w_b, e_b): w_a*e_b - w_b*e_a == 1 (a is better by one unit), e in (2^23, 2^24],
    w in (2^36, w_cap], and the double quotients w/e AND (w+e)/e are equal."""
    while True:
        e_a, e_b = (int(x) for x in rng.integers((1 << 23) + 1, E_MAX + 1, size=2))
        if math.gcd(e_a, e_b) != 1:
            continue
        w_a0 = pow(e_b, -1, e_a)                       # w_a*e_b = 1 (mod e_a)
        w_b0 = (w_a0 * e_b - 1) // e_a
        t_hi = min((w_cap - w_a0) // e_a, (w_cap - w_b0) // e_b)
        t = t_hi - int(rng.integers(0, 64))
        w_a, w_b = w_a0 + t * e_a, w_b0 + t * e_b
        if not ((1 << 36) < w_a <= w_cap and (1 << 36) < w_b <= w_cap):
            continue
        assert w_a * e_b - w_b * e_a == 1
        if float(w_a) / float(e_a) == float(w_b) / float(e_b) and (w_a + e_a) / e_a == (w_b + e_b) / e_b:
            return w_a, e_a, w_b, e_b


def gpu_select(asr, q2d, policy, now, k):
    import torch
    nq, ql = q2d.shape
    out = asr.select_batched(asr.to_device(q2d), nq, ql, policy, now, k)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_select_pair_alone(asr_mod):
    """the GPU twin of tests/test_oracle_select.py::test_hrrn_needs_exact_arithmetic"""
    rng = np.random.default_rng(38)
    for now in (T_MAX, 1 << 38):
        qs, better_first = [], []
        for i in range(64):
            w_a, e_a, w_b, e_b = near_tie_pair(rng, w_cap=now - 1)
            if i % 2:
                qs.append(orc.make_trace([now - w_a, now - w_b], [e_a, e_b]))
                better_first.append(0)
            else:
                qs.append(orc.make_trace([now - w_b, now - w_a], [e_b, e_a]))
                better_first.append(1)
        q = np.stack(qs)
        for k in (1, 2):
            got = gpu_select(asr_mod, q, orc.HRRN, now, k)
            for i in range(len(qs)):
                want = orc.select(q[i], orc.HRRN, now, k)
                assert want[0] == better_first[i]
                assert np.array_equal(got[i], want), (now, k, i)


@pytest.mark.parametrize("k", [1, 7, 32])
def test_select_pair_straddles_rank_k(asr_mod, k):
    """4,096-record queues: k-1 records clearly better than the pair, the rest clearly worse, the pair at
    ranks k-1 and k, planted at random positions (same chunk, different chunks, either order)"""
    rng = np.random.default_rng(100 + k)
    now, ql, nq = T_MAX, 4096, 48
    q = np.zeros((nq, ql), dtype=wl.REQ)
    pos_a = np.zeros(nq, dtype=np.int64)
    for i in range(nq):
        w_a, e_a, w_b, e_b = near_tie_pair(rng)
        ratio = w_a // e_a                                 # ~2^13 .. 2^15
        e = rng.integers(1 << 20, E_MAX + 1, size=ql)
        w = (rng.random(ql) * np.minimum(float(now), 0.9 * ratio * e)).astype(np.int64)   # ratio < 0.9 * pair's
        best = rng.choice(ql, size=k - 1, replace=False)
        e[best] = rng.integers(1, 1000, size=k - 1)        # ratio > 2^26
        w[best] = rng.integers(1 << 36, now, size=k - 1)
        rest = np.setdiff1d(np.arange(ql), best)
        pa, pb = (int(x) for x in rng.choice(rest, size=2, replace=False))
        if i % 3 == 0:
            pb = pa + 1 if pa + 1 < ql and (pa + 1) not in best else pb      # neighbours
        w[pa], e[pa], w[pb], e[pb] = w_a, e_a, w_b, e_b
        q[i]["arrival_us"], q[i]["dur_ms"], q[i]["est"] = now - w, 1000, e
        pos_a[i] = pa
    got = gpu_select(asr_mod, q, orc.HRRN, now, k)
    for i in range(nq):
        want = orc.select(q[i], orc.HRRN, now, k + 1)
        assert want[k - 1] == pos_a[i]                     # the pair straddles rank k: only a is selected
        assert np.array_equal(got[i], want[:k]), (k, i)
    got = gpu_select(asr_mod, q, orc.HRRN, now, min(32, k + 1))
    for i in range(nq):
        assert np.array_equal(got[i], orc.select(q[i], orc.HRRN, now, min(32, k + 1))), (k, i)


def full_range_queue(rng, n, now, kind):
    arr = rng.integers(0, now + 1, size=n, dtype=np.int64)
    if kind == "uniform":
        est = rng.integers(1, E_MAX + 1, size=n)
    elif kind == "top":                                    # est within a few units of the bound, waits near 2^38
        est = E_MAX - rng.integers(0, 8, size=n)
        arr = rng.integers(0, 1 << 20, size=n, dtype=np.int64)
    elif kind == "family":                                 # w = m*e - 1 for one m: ratios m - 1/e, doubles tie in droves
        est = E_MAX - rng.integers(0, 4096, size=n)
        arr = now - (est.astype(np.int64) * 16000 - 1)
    else:                                                  # log-uniform est, many orders of magnitude
        est = np.exp(rng.uniform(0, math.log(E_MAX), size=n)).astype(np.int64).clip(1, E_MAX)
    return orc.make_trace(arr, np.full(n, 1000), est=est)


@pytest.mark.parametrize("kind", ["uniform", "top", "family", "log"])
@pytest.mark.parametrize("policy", POL)
def test_select_random_queues_over_the_whole_range(asr_mod, kind, policy):
    import torch
    rng = np.random.default_rng(7 + policy)
    now = T_MAX
    for ql, k, nq in [(4096, 32, 24), (300, 5, 40)]:
        q = np.stack([full_range_queue(rng, ql, now, kind) for _ in range(nq)])
        got = gpu_select(asr_mod, q, policy, now, k)
        for i in range(nq):
            assert np.array_equal(got[i], orc.select(q[i], policy, now, k)), (kind, policy, ql, i)
    one = full_range_queue(rng, 50000, now, kind)           # the single-queue call (segment tree + indirect pass)
    out = asr_mod.select(asr_mod.to_device(one), len(one), policy, now, 32)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), orc.select(one, policy, now, 32)), (kind, policy)


# ---- simulator: the clock is carried to ~2^38 by one long first request ---------------------------------------
# cost model: encoder (2^14 - 1) us per ms of audio, nothing else but a 10 us iteration; request 0 has
# dur_ms = 2^24 - 2048 (the documented maximum is 2^24), every other request dur_ms <= 3; one token each.
BIG = (0, (1 << 14) - 1, 10, 0, 1, 0)
DUR0 = E_MAX - 2048
T_STAR = ((1 << 14) - 1) * DUR0 + 10                        # completion of request 0 = the first real admit step


def test_simulate_pair_competes_for_one_slot(asr_tier):
    """one slot: request 0 runs from t = 0 to T_STAR ~ 2^38 - 2^25; a and b arrive meanwhile with waits whose
    double quotients tie at T_STAR and whose cross-products differ by one; exactly one of them is admitted first"""
    rng = np.random.default_rng(5)
    traces, a_first = [], []
    for i in range(24):
        w_a, e_a, w_b, e_b = near_tie_pair(rng, w_cap=T_STAR - 1)
        rows = sorted([(T_STAR - w_a, e_a, "a"), (T_STAR - w_b, e_b, "b")])
        tr = orc.make_trace([0] + [r[0] for r in rows], [DUR0, 1, 2], est=[5] + [r[1] for r in rows])
        traces.append(tr)
        a_first.append(1 + [r[2] for r in rows].index("a"))
    reps = [(i, p, 1) for i in range(len(traces)) for p in (orc.HRRN, orc.SJF, orc.FCFS)]
    L, T, S = run_batched(traces, reps, BIG, 1)
    for j, (i, p, s) in enumerate(reps):
        check_replica(traces[i], p, s, BIG, L[j], T[j], S[j], "pair %d pol %d" % (i, p))
        if p == orc.HRRN:                                   # a got the slot: its TTFT is the smaller one
            other = 3 - a_first[i]
            assert L[j][a_first[i]] + traces[i]["arrival_us"][a_first[i]] < L[j][other] + traces[i]["arrival_us"][other]


@pytest.mark.parametrize("n,slots,durs", [(3000, 1, (0,)), (2500, 4, (0,)), (400, 3, (0, 1, 2, 3)), (6000, 16, (0,))])
def test_simulate_random_traces_at_the_bounds(asr_tier, n, slots, durs):
    """arrivals over the whole range [1, T_STAR), est up to 2^24, everything waits behind request 0 and is then
    drained at now ~ 2^38 - 2^25 .. 2^38: deep windows (the CTA tier runs its pool in threshold mode for
    n > 2,048), near-ties of the 'family' kind mixed in"""
    rng = np.random.default_rng(n + slots)
    arr = np.sort(rng.integers(1, T_STAR, size=n - 1, dtype=np.int64))
    est = rng.integers(1, E_MAX + 1, size=n - 1)
    fam = rng.random(n - 1) < 0.3                           # w(T_STAR) = m*e - 1: ratios m - 1/e
    est[fam] = E_MAX - rng.integers(0, 4096, size=int(fam.sum()))
    arr[fam] = T_STAR - (est[fam].astype(np.int64) * 15000 - 1)
    order = np.argsort(arr, kind="stable")
    arr, est = arr[order], est[order]
    dur = rng.choice(np.asarray(durs), size=n - 1)
    tr = orc.make_trace(np.concatenate([[0], arr]), np.concatenate([[DUR0], dur]), est=np.concatenate([[7], est]))
    reps = [(0, p, slots) for p in POL]
    L, T, S = run_batched([tr], reps, BIG, slots)
    for j, (_, p, s) in enumerate(reps):
        check_replica(tr, p, s, BIG, L[j], T[j], S[j], "n=%d slots=%d pol=%d" % (n, slots, p))
    assert int(S[0]["last_done_us"]) <= T_MAX                # the whole run stayed inside the documented range
    L2, T2, S2 = run_batched([tr], reps, BIG, slots, summary_only=True)
    assert np.array_equal(S.view(np.uint8), S2.view(np.uint8))
