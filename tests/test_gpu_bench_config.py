"""-m gpu: parity at BASELINE.json's full per-unit sizes, in the launch configuration bench.py times.

config 3: the sweep pipeline (gen_trace_batched -> simulate_batched, summary-only, default kernel
choice) on a block of whole seeds x 8 rates x 3 policies x 10,000 requests; EVERY summary of the
block is compared with the oracle, and per-request arrays for a sample of replicas.
config 5: 4,096-record queues, k = 32, HRRN and SJF; a sample of queues of a large batch.
"""
import concurrent.futures as cf
import os

import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def asr():
    import torch
    assert torch.cuda.is_available()
    import paper_2603_11273_b200 as asr
    return asr


def _oracle_summary(args):
    seed, rate, dist, n, pol, slots, tables = args
    tr = orc.gen_trace(seed, rate, dist, n, *tables)
    lat, ttft, first, end = orc.simulate(tr, pol, orc.cost(*wl.CONFIG_COST), slots)
    return (orc.percentile(lat, 50), orc.percentile(lat, 90), orc.percentile(ttft, 50), orc.percentile(ttft, 90),
            first, end, n), lat, ttft


@pytest.mark.parametrize("seed0,n_seeds", [(0, 24), (2048 - 12, 24), (4096 - 24, 24)])
def test_config3_block_full_length(asr, tables, seed0, n_seeds):
    """whole seeds of the replica sweep at n = 10,000 (lognormal block, the block that
    straddles the lognormal/uniform boundary, uniform block)"""
    import torch
    from paper_2603_11273_b200 import binding as B
    cfg = wl.config3(n_seeds=n_seeds, seed0=seed0)
    n, slots, pols = cfg["n"], cfg["slots"], cfg["policies"]
    seeds = np.repeat(np.arange(n_seeds, dtype=np.uint64) + np.uint64(seed0), 8)
    rates = np.tile(np.asarray(cfg["rates_mhz"], dtype=np.int32), n_seeds)
    dist = (seeds >= 2048).astype(np.int32)          # the full config's split (seeds 0..2047 lognormal)
    T = len(seeds)
    R = T * len(pols)
    assert R >= 512
    specs = np.zeros(T, dtype=asr.SPEC_DTYPE)
    specs["seed"], specs["rate_mhz"], specs["dist"] = seeds, rates, dist
    rep = asr.make_replicas(np.repeat(np.arange(T, dtype=np.int64) * n, 3), np.arange(R, dtype=np.int64) * n, n,
                            np.tile(np.asarray(pols, dtype=np.int32), T), slots, 0)
    d_tab = asr.tables_to_device(*tables)
    d_tr = asr.gen_trace_batched(asr.to_device(specs), T, n, d_tab)
    d_sum = torch.zeros(R * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    d_cost = asr.to_device(asr.make_cost(*cfg["cost"]))
    asr.set_option(asr.OPT_SIM_LANE_MIN_REPLICAS, 512)      # the kernel choice of the full sweep
    try:
        asr.simulate_batched(d_tr, asr.to_device(rep), R, d_cost, 1, R * n, slots, None, None, d_sum)
        lat = torch.full((R * n,), -7, dtype=torch.int64, device="cuda")
        ttft = torch.full((R * n,), -7, dtype=torch.int64, device="cuda")
        d_sum2 = torch.zeros_like(d_sum)
        asr.simulate_batched(d_tr, asr.to_device(rep), R, d_cost, 1, R * n, slots, lat, ttft, d_sum2)
        torch.cuda.synchronize()
    finally:
        asr.set_option(asr.OPT_SIM_LANE_MIN_REPLICAS, 1024)
    S = d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)
    assert np.array_equal(S.view(np.uint8), d_sum2.cpu().numpy())
    jobs = [(int(seeds[r // 3]), int(rates[r // 3]), int(dist[r // 3]), n, pols[r % 3], slots, tables) for r in range(R)]
    with cf.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        want = list(ex.map(_oracle_summary, jobs))
    fields = ("p50_e2e_us", "p90_e2e_us", "p50_ttft_us", "p90_ttft_us", "first_arrival_us", "last_done_us", "n_done")
    for r in range(R):
        got = tuple(int(S[r][f]) for f in fields)
        assert got == want[r][0], "replica %d: %r != %r" % (r, got, want[r][0])
    lat, ttft = lat.cpu().numpy(), ttft.cpu().numpy()
    for r in range(0, R, 7):
        assert np.array_equal(lat[r * n:(r + 1) * n], want[r][1]), r
        assert np.array_equal(ttft[r * n:(r + 1) * n], want[r][2]), r


def test_config5_sampled_queues(asr, tables):
    """8,192 queues x 4,096 in one launch (every SM busy, many queues per warp); 96 sampled queues"""
    import torch
    cfg = wl.config5(n_queues=8192)
    nq, ql, k, now = cfg["n_queues"], cfg["q_len"], cfg["k"], cfg["now"]
    d_tab = asr.tables_to_device(*tables)
    first = 1000 * ql     # queues 1000.. of the config-5 stream
    d_q = asr.gen_queues(cfg["seed"], first, nq * ql, now, d_tab)
    torch.cuda.synchronize()
    pick = np.unique(np.concatenate([np.arange(4), np.arange(nq - 4, nq),
                                     np.random.default_rng(3).integers(0, nq, size=88)]))
    q = d_q.cpu().numpy().view(asr.REQ_DTYPE).reshape(nq, ql)
    for i in pick[:8]:
        ref = orc.gen_queue(cfg["seed"], first + int(i) * ql, ql, now, tables[0])
        assert np.array_equal(q[i].view(np.uint8), ref.view(np.uint8))
    for pol in cfg["policies"] + (wl.FCFS,):
        got = asr.select_batched(d_q, nq, ql, pol, now, k).cpu().numpy()
        assert got.min() >= 0 and got.max() < ql
        for i in pick:
            assert np.array_equal(got[i], orc.select(q[i], pol, now, k)), (pol, i)
        # properties that hold for every queue: k distinct indices
        s = np.sort(got, axis=1)
        assert (s[:, 1:] != s[:, :-1]).all()
