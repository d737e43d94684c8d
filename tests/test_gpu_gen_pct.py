"""-m gpu: trace generator (a1) and segmented percentiles (a6) against the oracle."""
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


def test_gen_trace_matches_oracle(asr, tables):
    import torch
    d_tab = asr.tables_to_device(*tables)
    for seed, rate, dist, n in [(0, 2000, 0, 1000), (1, 500, 1, 3000), (1, 4000, 1, 3000), (4, 35408, 0, 70000),
                                (9, 1, 0, 5), (2**40 + 3, 123457, 1, 257), (7, 1000, 0, 1), (7, 1000, 0, 255),
                                (7, 1000, 0, 256), (7, 1000, 0, 0), (3, 2_000_000_000, 0, 300)]:
        out = asr.gen_trace(seed, rate, dist, n, d_tab)
        torch.cuda.synchronize()
        got = out.cpu().numpy().view(asr.REQ_DTYPE)
        ref = orc.gen_trace(seed, rate, dist, n, *tables)
        assert np.array_equal(got.view(np.uint8), ref.view(np.uint8)), (seed, rate, dist, n)


def test_gen_trace_batched_matches_oracle(asr, tables):
    import torch
    cfg = wl.config3(n_seeds=6, n=700)
    seeds, rates, dist = wl.config3_traces(cfg)
    specs = np.zeros(len(seeds), dtype=asr.SPEC_DTYPE)
    specs["seed"], specs["rate_mhz"], specs["dist"] = seeds, rates, dist
    d_tab = asr.tables_to_device(*tables)
    out = asr.gen_trace_batched(asr.to_device(specs), len(specs), cfg["n"], d_tab)
    torch.cuda.synchronize()
    got = out.cpu().numpy().view(asr.REQ_DTYPE).reshape(len(specs), cfg["n"])
    assert set(dist[:24]) == {0} and set(dist[24:]) == {1}
    for t in range(len(specs)):
        ref = orc.gen_trace(int(seeds[t]), int(rates[t]), int(dist[t]), cfg["n"], *tables)
        assert np.array_equal(got[t].view(np.uint8), ref.view(np.uint8)), t


def test_gen_trace_batched_irregular_runs(asr, tables):
    """specs that do not fall into aligned blocks of eight rates per seed: runs of equal (seed, dist) of
    every length, the same seed under both distributions, repeated rates, a partial last block, and record
    counts around the generator's 1,024-record step"""
    import torch
    d_tab = asr.tables_to_device(*tables)
    rng = np.random.default_rng(11)
    seeds, rates, dist = [], [], []
    for run_len in (1, 3, 2, 8, 5, 9, 1, 1, 7, 4, 2):
        sd, ds = int(rng.integers(0, 2**63)), int(rng.integers(0, 2))
        for _ in range(run_len):
            seeds.append(sd); dist.append(ds); rates.append(int(rng.integers(1, 40000)))
    seeds += [5, 5, 5, 5]; dist += [0, 1, 0, 1]; rates += [777, 777, 2_000_000_000, 1000000]   # mean gap 0 us: a burst
    assert len(seeds) % 8 != 0
    for n in (1, 1023, 1024, 1025, 2500):
        specs = np.zeros(len(seeds), dtype=asr.SPEC_DTYPE)
        specs["seed"], specs["rate_mhz"], specs["dist"] = seeds, rates, dist
        out = asr.gen_trace_batched(asr.to_device(specs), len(specs), n, d_tab)
        torch.cuda.synchronize()
        got = out.cpu().numpy().view(asr.REQ_DTYPE).reshape(len(specs), n)
        for t in range(len(specs)):
            ref = orc.gen_trace(seeds[t], rates[t], dist[t], n, *tables)
            assert np.array_equal(got[t].view(np.uint8), ref.view(np.uint8)), (n, t)


def test_percentiles_match_oracle(asr):
    import torch
    rng = np.random.default_rng(2)
    segs = [rng.integers(0, 10**7, size=n) for n in (0, 1, 2, 99, 100, 101, 1000, 10000, 12288, 12289, 40000)]
    segs += [np.full(500, 42), rng.integers(-2**62, 2**62, size=3000), np.array([2**63 - 1, -2**63, 0, 5]),
             rng.integers(0, 3, size=5000), np.arange(7777)[::-1] * 2**33]
    vals = np.concatenate(segs).astype(np.int64)
    off = np.concatenate([[0], np.cumsum([len(s) for s in segs])]).astype(np.int64)
    pcts = [1, 25, 50, 90, 99, 100]
    d_vals = torch.from_numpy(vals).cuda()
    out = asr.percentiles(d_vals, torch.from_numpy(off).cuda(), len(segs), pcts)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    for s, seg in enumerate(segs):
        for j, p in enumerate(pcts):
            assert got[s, j] == orc.percentile(seg, p), (s, p)
    # `values` is not modified (asr_sched.h): the DEVICE buffer still holds the input
    assert np.array_equal(d_vals.cpu().numpy(), np.concatenate(segs).astype(np.int64))
