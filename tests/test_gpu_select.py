"""-m gpu: the CUDA select (a2+a3) against the oracle, bit-exact, through the C ABI."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu
POL = (orc.FCFS, orc.SJF, orc.HRRN)


@pytest.fixture(scope="module")
def asr():
    import torch
    assert torch.cuda.is_available()
    import paper_2603_11273_b200 as asr
    return asr


def gpu_select_batched(asr, q2d, policy, now, k, q_count=None, now_pq=None):
    import torch
    nq, ql = q2d.shape
    d = asr.to_device(q2d)
    dc = None if q_count is None else torch.from_numpy(np.asarray(q_count, dtype=np.int32)).cuda()
    dn = None if now_pq is None else torch.from_numpy(np.asarray(now_pq, dtype=np.int64)).cuda()
    out = asr.select_batched(d, nq, ql, policy, now, k, q_count=dc, now_per_queue=dn)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("kind", ["random", "six", "proportional", "identical", "few_arrivals", "future", "est_edge"])
@pytest.mark.parametrize("policy", POL)
def test_batched_stress_kinds(asr, kind, policy):
    now = 10**9
    for ql, k, nq in [(1, 4, 3), (31, 32, 5), (32, 32, 5), (33, 7, 5), (257, 32, 9), (700, 32, 17), (4096, 32, 6),
                      (5000, 1, 3)]:
        q = np.stack([wl.stress_queue(kind, ql, 1000 * ql + i, now) for i in range(nq)])
        got = gpu_select_batched(asr, q, policy, now, k)
        for i in range(nq):
            assert np.array_equal(got[i], orc.select(q[i], policy, now, k)), (kind, policy, ql, k, i)


@pytest.mark.parametrize("kind", ["random", "six", "proportional", "identical", "few_arrivals", "future", "est_edge"])
@pytest.mark.parametrize("policy", POL)
def test_wide_k_stress_kinds(asr, kind, policy):
    """32 < k <= 256 (up to 256 slots to admit into): the shared-memory sort kernel, same tie kinds,
    queues shorter than k, exactly one round, several rounds with the kept k carried along"""
    now = 10**9
    for ql, k, nq in [(20, 33, 3), (64, 64, 4), (300, 100, 5), (3840, 256, 3), (3841, 256, 2), (4096, 33, 3),
                      (9000, 256, 2), (700, 255, 4)]:
        q = np.stack([wl.stress_queue(kind, ql, 2000 * ql + i, now) for i in range(nq)])
        got = gpu_select_batched(asr, q, policy, now, k)
        for i in range(nq):
            assert np.array_equal(got[i], orc.select(q[i], policy, now, k)), (kind, policy, ql, k, i)


@pytest.mark.parametrize("policy", POL)
def test_wide_k_ragged_per_queue_now_and_single_queue(asr, policy):
    import torch
    rng = np.random.default_rng(50 + policy)
    nq, ql, k = 24, 900, 100
    now = 10**8
    q = np.stack([wl.stress_queue("random" if i % 2 else "six", ql, 977 + i, now) for i in range(nq)])
    counts = rng.integers(0, ql + 1, size=nq)
    counts[:4] = [0, 1, ql, 99]
    nows = rng.integers(1, 2 * now, size=nq)
    got = gpu_select_batched(asr, q, policy, now, k, q_count=counts, now_pq=nows)
    for i in range(nq):
        assert np.array_equal(got[i], orc.select(q[i][:counts[i]], policy, int(nows[i]), k)), i
    for n, kk in ((5000, 64), (40000, 256)):     # the single-queue call: segments, then the reported positions
        qq = wl.stress_queue("random", n, n + 3, 10**10)
        out = asr.select(asr.to_device(qq), n, policy, 10**10, kk)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), orc.select(qq, policy, 10**10, kk)), (policy, n, kk)


@pytest.mark.parametrize("policy", POL)
def test_ragged_counts_and_per_queue_now(asr, policy):
    rng = np.random.default_rng(policy)
    nq, ql, k = 40, 600, 32
    now = 10**8
    q = np.stack([wl.stress_queue("random" if i % 2 else "few_arrivals", ql, 77 + i, now) for i in range(nq)])
    counts = rng.integers(0, ql + 1, size=nq)
    counts[:4] = [0, 1, ql, 31]
    nows = rng.integers(1, 2 * now, size=nq)
    got = gpu_select_batched(asr, q, policy, now, k, q_count=counts, now_pq=nows)
    for i in range(nq):
        assert np.array_equal(got[i], orc.select(q[i][:counts[i]], policy, int(nows[i]), k)), i


@pytest.mark.parametrize("policy", POL)
@pytest.mark.parametrize("n", [0, 1, 4096, 4097, 20000, 300000])
def test_single_queue_any_length(asr, policy, n):
    import torch
    now = 10**10
    q = wl.stress_queue("random" if n != 20000 else "six", n, n + 1, now)
    d = asr.to_device(q) if n else torch.zeros(16, dtype=torch.uint8, device="cuda")
    for k in (1, 32):
        out = asr.select(d, n, policy, now, k)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), orc.select(q, policy, now, k)), (policy, n, k)


def test_generated_config5_queues_small(asr, tables):
    """config-5 recipe at oracle-friendly size: 96 queues x 4096, k = 32, seed 5."""
    import torch
    cfg = wl.config5(n_queues=96)
    d_tab = asr.tables_to_device(*tables)
    dq = asr.gen_queues(cfg["seed"], 0, cfg["n_queues"] * cfg["q_len"], cfg["now"], d_tab)
    torch.cuda.synchronize()
    q = dq.cpu().numpy().view(asr.REQ_DTYPE).reshape(cfg["n_queues"], cfg["q_len"])
    ref = orc.gen_queue(cfg["seed"], 0, q.size, cfg["now"], tables[0]).reshape(q.shape)
    assert np.array_equal(q.view(np.uint8), ref.view(np.uint8))
    for pol in cfg["policies"]:
        got = asr.select_batched(dq, cfg["n_queues"], cfg["q_len"], pol, cfg["now"], cfg["k"]).cpu().numpy()
        for i in range(cfg["n_queues"]):
            assert np.array_equal(got[i], orc.select(ref[i], pol, cfg["now"], cfg["k"])), (pol, i)


def test_select_host_entry(asr):
    now = 10**9
    q = np.stack([wl.stress_queue("random", 300, i, now) for i in range(8)])
    got = asr.select_host(q, 8, 300, orc.HRRN, now, 16)
    for i in range(8):
        assert np.array_equal(got[i], orc.select(q[i], orc.HRRN, now, 16))


@pytest.mark.parametrize("policy", POL)
@pytest.mark.parametrize("k", [32, 5])
def test_many_queues_per_warp_with_drifting_distributions(asr, policy, k):
    """Every warp of the persistent grid serves six queues in a row whose key distributions jump
    around, so a threshold carried over from the previous queue is in turn well calibrated, far
    too strict (nothing passes: the queue is read again), far too loose (cuts inside the queue),
    or meets a queue shorter than k / an empty queue / a queue of identical keys."""
    import torch
    now = 10**9
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    gw = sm * 20                       # queues in flight: one per warp of the persistent grid
    nq, ql = 6 * gw, 128
    rng = np.random.default_rng(1000 * policy + k)
    q = np.zeros((nq, ql), dtype=wl.REQ)
    counts = np.full(nq, ql, dtype=np.int32)
    kind = (np.arange(nq) // gw + np.arange(nq) % 3) % 6
    arr = rng.integers(0, now, size=(nq, ql), dtype=np.int64)
    dur = rng.integers(1000, 35001, size=(nq, ql)).astype(np.int32)
    late = kind == 1                   # recent arrivals, long jobs: worst under every policy
    arr[late] = now - rng.integers(0, 1000, size=(int(late.sum()), ql))
    dur[late] = rng.integers(30000, 35001, size=(int(late.sum()), ql))
    early = kind == 2                  # old arrivals, short jobs: best under every policy
    arr[early] = rng.integers(0, 1000, size=(int(early.sum()), ql))
    dur[early] = rng.integers(1, 50, size=(int(early.sum()), ql))
    same = kind == 4                   # identical keys: the index decides
    arr[same] = now // 3
    dur[same] = 7000
    q["arrival_us"], q["dur_ms"], q["est"] = arr, dur, dur
    short = kind == 5                  # shorter than k, or empty
    counts[short] = rng.integers(0, max(2, k), size=int(short.sum()))
    got = gpu_select_batched(asr, q, policy, now, k, q_count=counts)
    pick = np.unique(np.concatenate([np.arange(0, nq, 37), np.arange(gw - 3, nq, gw), np.arange(gw, nq, gw)]))
    for i in pick:
        assert np.array_equal(got[i], orc.select(q[i][:counts[i]], policy, now, k)), (policy, k, int(i), int(kind[i]))
    # every queue: k distinct valid indices, then -1 padding
    valid = np.minimum(counts, k)
    for i in range(0, nq, 11):
        v = got[i][:valid[i]]
        assert len(set(v.tolist())) == len(v) and (v >= 0).all() and (v < counts[i]).all()
        assert (got[i][valid[i]:] == -1).all()
