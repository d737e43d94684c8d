"""-m gpu: asr_sched_select_static, the entry point that allocates nothing (include/asr_sched.h): its scratch is a
device array built into the library.  Its output must equal asr_sched_select's (and the oracle's) bit for bit,
on calls in a row that share the array, whatever ran before in the process.  Collected last on purpose."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu
POL = (orc.FCFS, orc.SJF, orc.HRRN)
NOW = 10**10


@pytest.fixture(scope="module")
def asr():
    import torch
    assert torch.cuda.is_available()
    import paper_2603_11273_b200 as asr
    return asr


def test_select_static_equals_select_on_calls_in_a_row(asr):
    """a three-level queue, then a two-level one that finds the first call's leftovers in the array, then the first
    again; k = 32 (streaming kernel) and k = 200 (wide kernel); free device memory does not move"""
    import torch
    cases = [("random", 2_000_000, 31), ("six", 300_000, 32), ("random", 2_000_000, 31)]
    queues = {(kind, n): wl.stress_queue(kind, n, n + 7, NOW) for kind, n, _ in cases}
    dq = {key: asr.to_device(q) for key, q in queues.items()}
    want = {}
    for kind, n, k in cases:
        for policy in POL:
            for kk in (k, 200):
                if (kind, n, policy, kk) not in want:
                    want[(kind, n, policy, kk)] = asr.select(dq[(kind, n)], n, policy, NOW, kk).cpu().numpy()
    out = {kk: torch.full((kk,), -7, dtype=torch.int32, device="cuda") for kk in (31, 32, 200)}
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    alloc0 = torch.cuda.memory_allocated()
    got = []
    for kind, n, k in cases:
        for policy in POL:
            for kk in (k, 200):
                asr.select_static(dq[(kind, n)], n, policy, NOW, kk, out[kk])
                torch.cuda.synchronize()
                # (device allocations come in 2 MiB pages: anything allocated behind torch's back would show)
                assert abs(torch.cuda.mem_get_info()[0] - free0) < (1 << 20) and torch.cuda.memory_allocated() == alloc0
                got.append(((kind, n, policy, kk), out[kk].cpu().numpy().copy()))
    for key, g in got:
        assert np.array_equal(g, want[key]), key
    # and against the oracle, on the queue it finishes in a second
    q = queues[("six", 300_000)]
    for policy in POL:
        assert np.array_equal(want[("six", 300_000, policy, 32)], orc.select(q, policy, NOW, 32)), policy


def test_select_static_small_and_rejected_sizes(asr):
    import torch
    q = wl.stress_queue("random", 4096, 11, NOW)
    d = asr.to_device(q)
    out = torch.full((8,), -7, dtype=torch.int32, device="cuda")
    asr.select_static(d, 4096, orc.HRRN, NOW, 8, out)   # one segment: no scratch at all
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), orc.select(q, orc.HRRN, NOW, 8))
    assert asr.workspace_bytes(0, 33_000_000, 32) <= asr.SELECT_STATIC_SCRATCH_BYTES < asr.workspace_bytes(0, 34_000_000, 32)
    for n, k in ((34_000_000, 32), (4_200_000, 256)):   # decided from the sizes alone, before any launch
        with pytest.raises(asr.AsrSchedError) as e:
            asr.select_static(d, n, orc.SJF, NOW, k, out)
        assert "scratch" in str(e.value)
    with pytest.raises(asr.AsrSchedError):
        asr.select_static(d, 4096, orc.SJF, NOW, 257, out)
