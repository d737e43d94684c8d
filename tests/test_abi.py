"""The C-ABI library loads and exports every symbol include/asr_sched.h declares.
No compute call is made here (no GPU on this box)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HDR = os.path.join(ROOT, "include", "asr_sched.h")


@pytest.fixture(scope="module")
def asr():
    import __graft_entry__ as g
    g.build()
    import paper_2603_11273_b200 as asr
    return asr


def declared_symbols():
    text = open(HDR).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(asr_sched_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(asr):
    names = declared_symbols()
    assert len(names) >= 14
    L = ctypes.CDLL(asr.lib_path())
    for n in names:
        assert hasattr(L, n), n
    from paper_2603_11273_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_version_error_and_counters(asr):
    assert asr.version() == 100
    assert isinstance(asr.last_error(), str)
    assert asr.launch_count() >= 0


def test_struct_sizes_match_header(asr):
    assert asr.REQ_DTYPE.itemsize == 16
    assert asr.COST_DTYPE.itemsize == 40
    assert asr.REPLICA_DTYPE.itemsize == 32
    assert asr.SUMMARY_DTYPE.itemsize == 56
    assert asr.SPEC_DTYPE.itemsize == 16


def test_workspace_sizes(asr):
    from paper_2603_11273_b200 import binding as b
    assert asr.workspace_bytes(b.OP_SELECT, 4096, 32) == 0
    small = asr.workspace_bytes(b.OP_SELECT, 10**6, 32)
    assert small >= 4 * 32 * (10**6 // 4096)
    full = asr.workspace_bytes(b.OP_SIMULATE, 10**6, 100, 0)
    summ = asr.workspace_bytes(b.OP_SIMULATE, 10**6, 100, 1)
    assert summ >= full + 16 * 10**6
    assert asr.workspace_bytes(99, 1, 1) == 0


def test_argument_errors_need_no_gpu(asr):
    """-1 / -3 are decided before any CUDA call."""
    L = asr.lib()
    assert L.asr_sched_select_batched(None, 4, 16, None, 7, 0, None, 4, None, None) == -1
    assert "policy" in asr.last_error()
    assert L.asr_sched_select_batched(None, 4, 16, None, 1, 0, None, 257, None, None) == -3
    assert L.asr_sched_select(None, -1, 0, 0, 1, None, None, 0, None) == -1
    assert L.asr_sched_select(None, 10, 0, 0, 300, None, None, 0, None) == -3
    cm = asr.make_cost(1, 1, 1, 1, 1, 1)
    assert L.asr_sched_simulate(None, 10, 0, cm.ctypes.data, 0, None, None, None, None, 0, None) == -1
    assert L.asr_sched_simulate(None, 10, 0, cm.ctypes.data, 257, None, None, None, None, 0, None) == -3
    assert L.asr_sched_simulate(None, 10, 0, cm.ctypes.data, 4, None, None, None, None, 0, None) == -1  # workspace
    pc = np.array([50, 101], dtype=np.int32)
    assert L.asr_sched_percentiles(None, None, 1, pc.ctypes.data, 2, None, None, 0, None) == -1
    pc9 = np.arange(1, 10, dtype=np.int32)
    assert L.asr_sched_percentiles(None, None, 1, pc9.ctypes.data, 9, None, None, 0, None) == -3
    assert L.asr_sched_gen_trace(0, 0, 0, 10, None, None, None) == -1
    assert L.asr_sched_select_host(None, 1, 1, 0, 0, 257, None) == -3
    # tuning options: known ids and value ranges only
    from paper_2603_11273_b200 import binding as b
    assert L.asr_sched_set_option(b.OPT_SIM_LANE_SPLIT, 2) == -1
    assert L.asr_sched_set_option(b.OPT_SIM_LANE_SPLIT, 0) == 0 and L.asr_sched_set_option(b.OPT_SIM_LANE_SPLIT, 1) == 0
    assert L.asr_sched_set_option(77, 1) == -1
    # zero-size work is a no-op that needs no device
    assert L.asr_sched_select_batched(None, 0, 16, None, 1, 0, None, 4, None, None) == 0
    assert L.asr_sched_percentiles(None, None, 0, pc.ctypes.data, 0, None, None, 0, None) == 0


def test_missing_library_fails_loudly(asr, monkeypatch):
    from paper_2603_11273_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", "/nonexistent/libasr_sched.so")
    with pytest.raises(binding.AsrSchedError):
        binding.lib()


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2603_11273_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2603_11273_b200" not in src and "asr_sched.h" not in src
