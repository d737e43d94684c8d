"""Helpers shared by the -m gpu parity tests."""
import numpy as np

import oracle as orc
import paper_2603_11273_b200 as asr
import workloads as wl


def dev_trace(tr):
    return asr.to_device(np.ascontiguousarray(tr, dtype=asr.REQ_DTYPE))


def run_batched(traces, replicas, cost_tuple, max_slots, summary_only=False):
    """traces: list of REQ arrays; replicas: list of (trace_id, policy, slots).
    -> (lat[list], ttft[list], summaries)"""
    import torch
    offs = np.concatenate([[0], np.cumsum([len(t) for t in traces])]).astype(np.int64)
    all_tr = np.concatenate(traces) if traces else np.zeros(0, dtype=asr.REQ_DTYPE)
    ns = np.array([len(traces[t]) for t, _, _ in replicas], dtype=np.int64)
    out_off = np.concatenate([[0], np.cumsum(ns)]).astype(np.int64)
    total = int(out_off[-1])
    rep = asr.make_replicas([offs[t] for t, _, _ in replicas], out_off[:-1], ns,
                            [p for _, p, _ in replicas], [s for _, _, s in replicas], 0)
    d_tr = dev_trace(all_tr)
    d_rep = asr.to_device(rep)
    d_cm = asr.to_device(asr.make_cost(*cost_tuple))
    d_sum = torch.zeros(len(replicas) * asr.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    if summary_only:
        asr.simulate_batched(d_tr, d_rep, len(replicas), d_cm, 1, total, max_slots, None, None, d_sum)
        torch.cuda.synchronize()
        return None, None, d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)
    lat = torch.full((max(total, 1),), -7, dtype=torch.int64, device="cuda")
    ttft = torch.full((max(total, 1),), -7, dtype=torch.int64, device="cuda")
    asr.simulate_batched(d_tr, d_rep, len(replicas), d_cm, 1, total, max_slots, lat, ttft, d_sum)
    torch.cuda.synchronize()
    lat, ttft = lat.cpu().numpy(), ttft.cpu().numpy()
    L = [lat[out_off[i]:out_off[i + 1]] for i in range(len(replicas))]
    T = [ttft[out_off[i]:out_off[i + 1]] for i in range(len(replicas))]
    return L, T, d_sum.cpu().numpy().view(asr.SUMMARY_DTYPE)


def check_replica(tr, policy, slots, cost_tuple, lat, ttft, summ, tag=""):
    rl, rt, first, end = orc.simulate(tr, policy, orc.cost(*cost_tuple), slots)
    if lat is not None:
        assert np.array_equal(lat, rl), "latency mismatch " + tag
        assert np.array_equal(ttft, rt), "ttft mismatch " + tag
    want = (orc.percentile(rl, 50), orc.percentile(rl, 90), orc.percentile(rt, 50), orc.percentile(rt, 90),
            first, end, len(tr))
    got = tuple(int(summ[f]) for f in ("p50_e2e_us", "p90_e2e_us", "p50_ttft_us", "p90_ttft_us",
                                       "first_arrival_us", "last_done_us", "n_done"))
    assert got == want, "summary mismatch %s: %r != %r" % (tag, got, want)
