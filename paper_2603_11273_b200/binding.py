"""ctypes binding of include/asr_sched.h -- argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "libasr_sched.so")

FCFS, SJF, HRRN, ADAPTIVE = 0, 1, 2, 3
DIST_LOGNORMAL, DIST_UNIFORM = 0, 1
OP_SELECT, OP_SIMULATE, OP_PERCENTILES, OP_SIMULATE_EX, OP_ITL = 0, 1, 2, 3, 4

# numpy views of the ABI structs (include/asr_sched.h)
REQ_DTYPE = np.dtype([("arrival_us", "<i8"), ("dur_ms", "<i4"), ("est", "<i4")])
COST_DTYPE = np.dtype([("enc_base_us", "<i8"), ("enc_per_ms_us", "<i8"), ("iter_base_us", "<i8"),
                       ("iter_per_running_us", "<i8"), ("tok_base", "<i4"), ("tok_per_s", "<i4")])
REPLICA_DTYPE = np.dtype([("trace_off", "<i8"), ("out_off", "<i8"), ("n", "<i4"), ("policy", "<i4"),
                          ("slots", "<i4"), ("cm_id", "<i4")])
SUMMARY_DTYPE = np.dtype([("p50_e2e_us", "<i8"), ("p90_e2e_us", "<i8"), ("p50_ttft_us", "<i8"),
                          ("p90_ttft_us", "<i8"), ("first_arrival_us", "<i8"), ("last_done_us", "<i8"),
                          ("n_done", "<i8")])
SPEC_DTYPE = np.dtype([("seed", "<u8"), ("rate_mhz", "<i4"), ("dist", "<i4")])
TABLES_DTYPE = np.dtype([("ln_dur", "<u4", (4097,)), ("exp_t", "<u4", (4097,))])
EXT_DTYPE = np.dtype([("kv_budget", "<i8"), ("kv_base", "<i8"), ("kv_per_s", "<i8"), ("depth1", "<i4"),
                      ("depth2", "<i4"), ("pol", "<i4", (3,)), ("pad", "<i4")])
assert EXT_DTYPE.itemsize == 48
assert REQ_DTYPE.itemsize == 16 and COST_DTYPE.itemsize == 40 and REPLICA_DTYPE.itemsize == 32
assert SUMMARY_DTYPE.itemsize == 56 and SPEC_DTYPE.itemsize == 16 and TABLES_DTYPE.itemsize == 2 * 4097 * 4

EXPORTS = (
    "asr_sched_select", "asr_sched_select_batched", "asr_sched_simulate", "asr_sched_simulate_batched",
    "asr_sched_percentiles", "asr_sched_gen_trace", "asr_sched_gen_trace_batched", "asr_sched_gen_queues",
    "asr_sched_sweep_host", "asr_sched_select_host", "asr_sched_select_static", "asr_sched_simulate_batched_ex", "asr_sched_tpot",
    "asr_sched_estimate", "asr_sched_itl_batched", "asr_sched_trim_scratch", "asr_sched_workspace_bytes", "asr_sched_last_error",
    "asr_sched_version", "asr_sched_launch_count", "asr_sched_timing_enable", "asr_sched_timing_reset",
    "asr_sched_timing_read", "asr_sched_kernel_name", "asr_sched_set_option",
)


class AsrSchedError(RuntimeError):
    pass


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Load libasr_sched.so.  Fails loudly when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise AsrSchedError(
                "libasr_sched.so is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        vp, i64, i32, u64, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_uint64, C.c_size_t
        L.asr_sched_select.argtypes = [vp, i64, i32, i64, i32, vp, vp, sz, vp]
        L.asr_sched_select_static.argtypes = [vp, i64, i32, i64, i32, vp, vp]
        L.asr_sched_select_batched.argtypes = [vp, i32, i32, vp, i32, i64, vp, i32, vp, vp]
        L.asr_sched_simulate.argtypes = [vp, i64, i32, vp, i32, vp, vp, vp, vp, sz, vp]
        L.asr_sched_simulate_batched.argtypes = [vp, vp, i32, vp, i32, i64, i32, vp, vp, vp, vp, sz, vp]
        L.asr_sched_percentiles.argtypes = [vp, vp, i32, vp, i32, vp, vp, sz, vp]
        L.asr_sched_gen_trace.argtypes = [u64, i32, i32, i64, vp, vp, vp]
        L.asr_sched_gen_trace_batched.argtypes = [vp, i32, i64, vp, vp, vp]
        L.asr_sched_gen_queues.argtypes = [u64, i64, i64, i64, vp, vp, vp]
        L.asr_sched_sweep_host.argtypes = [vp, i32, i64, vp, vp, i32, i32, vp, vp]
        L.asr_sched_select_host.argtypes = [vp, i32, i32, i32, i64, i32, vp]
        L.asr_sched_simulate_batched_ex.argtypes = [vp, vp, i32, vp, vp, i32, i64, i32, vp, vp, vp, vp, vp, sz, vp]
        L.asr_sched_tpot.argtypes = [vp, i64, vp, vp, vp, vp, vp]
        L.asr_sched_estimate.argtypes = [vp, i64, vp, i32, vp, vp, vp]
        L.asr_sched_itl_batched.argtypes = [vp, vp, i32, vp, i32, i64, i32, vp, i32, vp, vp, sz, vp]
        for name in EXPORTS[:16]:
            getattr(L, name).restype = C.c_int
        L.asr_sched_workspace_bytes.argtypes = [i32, i64, i64, i64]
        L.asr_sched_workspace_bytes.restype = sz
        L.asr_sched_last_error.restype = C.c_char_p
        L.asr_sched_version.restype = C.c_int
        L.asr_sched_launch_count.restype = i64
        L.asr_sched_timing_enable.argtypes = [C.c_int]
        L.asr_sched_timing_read.argtypes = [i32, C.POINTER(C.c_double), C.POINTER(i64)]
        L.asr_sched_kernel_name.argtypes = [i32]
        L.asr_sched_kernel_name.restype = C.c_char_p
        L.asr_sched_set_option.argtypes = [i32, i64]
        L.asr_sched_set_option.restype = C.c_int
        _lib = L
    return _lib


def version() -> int:
    return lib().asr_sched_version()


def last_error() -> str:
    return lib().asr_sched_last_error().decode()


def launch_count() -> int:
    return int(lib().asr_sched_launch_count())


OPT_SIM_LANE_MIN_REPLICAS = 0
OPT_SIM_ESCALATE_WINDOW = 1
OPT_SIM_LANE_SPLIT = 2


def set_option(option: int, value: int):
    _check(lib().asr_sched_set_option(option, value), "asr_sched_set_option")


def timing_enable(on: bool):
    lib().asr_sched_timing_enable(1 if on else 0)


def timing_reset():
    lib().asr_sched_timing_reset()


def timing_read() -> dict:
    """-> {kernel name: (total device ms, launches)} since the last reset (synchronises)."""
    out, kid = {}, 0
    while True:
        name = lib().asr_sched_kernel_name(kid)
        if name is None:
            return out
        ms, n = C.c_double(0.0), C.c_int64(0)
        _check(lib().asr_sched_timing_read(kid, C.byref(ms), C.byref(n)), "asr_sched_timing_read")
        out[name.decode()] = (ms.value, int(n.value))
        kid += 1


def workspace_bytes(op: int, a: int, b: int, c: int = 0) -> int:
    return int(lib().asr_sched_workspace_bytes(op, a, b, c))


def _check(rc: int, what: str):
    if rc != 0:
        raise AsrSchedError("%s failed (rc=%d): %s" % (what, rc, last_error()))


def _torch():
    import torch
    return torch


def _ptr(t):
    return 0 if t is None else t.data_ptr()


def _stream():
    return _torch().cuda.current_stream().cuda_stream


def to_device(a: np.ndarray, device="cuda"):
    """numpy (possibly structured) -> flat uint8 device tensor with the same bytes."""
    torch = _torch()
    a = np.ascontiguousarray(a)
    return torch.from_numpy(a.view(np.uint8).reshape(-1)).to(device)


def from_device(t, dtype) -> np.ndarray:
    return t.detach().cpu().numpy().view(dtype)


def make_tables(ln_dur, exp_t) -> np.ndarray:
    t = np.zeros(1, dtype=TABLES_DTYPE)
    t["ln_dur"][0] = np.asarray(ln_dur, dtype=np.uint32)
    t["exp_t"][0] = np.asarray(exp_t, dtype=np.uint32)
    return t


def tables_to_device(ln_dur, exp_t, device="cuda"):
    return to_device(make_tables(ln_dur, exp_t), device)


def make_cost(enc_base_us, enc_per_ms_us, iter_base_us, iter_per_running_us, tok_base, tok_per_s) -> np.ndarray:
    c = np.zeros(1, dtype=COST_DTYPE)
    c[0] = (enc_base_us, enc_per_ms_us, iter_base_us, iter_per_running_us, tok_base, tok_per_s)
    return c


def make_replicas(trace_off, out_off, n, policy, slots, cm_id=0) -> np.ndarray:
    trace_off = np.asarray(trace_off, dtype=np.int64)
    r = np.zeros(trace_off.shape[0], dtype=REPLICA_DTYPE)
    r["trace_off"], r["out_off"], r["n"] = trace_off, out_off, n
    r["policy"], r["slots"], r["cm_id"] = policy, slots, cm_id
    return r


def _workspace(nbytes: int, device):
    torch = _torch()
    return torch.empty(max(int(nbytes), 16), dtype=torch.uint8, device=device)


# ---------------------------------------------------------------------------
# device-pointer calls (same names as the ABI, minus the prefix)
# ---------------------------------------------------------------------------

def select(keys, n: int, policy: int, now: int, k: int, out_idx=None, workspace=None):
    """asr_sched_select: keys = uint8 device tensor of n asr_req_t.  -> int32[k] device tensor."""
    torch = _torch()
    if out_idx is None:
        out_idx = torch.empty(max(k, 1), dtype=torch.int32, device=keys.device)[:k]
    if workspace is None:
        workspace = _workspace(workspace_bytes(OP_SELECT, n, k), keys.device)
    _check(lib().asr_sched_select(_ptr(keys), n, policy, now, k, _ptr(out_idx), _ptr(workspace),
                                  workspace.numel(), _stream()), "asr_sched_select")
    return out_idx


SELECT_STATIC_SCRATCH_BYTES = 1 << 20


def select_static(keys, n: int, policy: int, now: int, k: int, out_idx):
    """asr_sched_select_static: asr_sched_select with the library's built-in scratch; allocates nothing (the caller
    passes out_idx, an int32[k] device tensor)."""
    _check(lib().asr_sched_select_static(_ptr(keys), n, policy, now, k, _ptr(out_idx), _stream()),
           "asr_sched_select_static")
    return out_idx


def select_batched(keys, n_queues: int, q_len: int, policy: int, now: int, k: int, q_count=None,
                   now_per_queue=None, out_idx=None):
    torch = _torch()
    if out_idx is None:
        out_idx = torch.empty((n_queues, k), dtype=torch.int32, device=keys.device)
    _check(lib().asr_sched_select_batched(_ptr(keys), n_queues, q_len, _ptr(q_count), policy, now,
                                          _ptr(now_per_queue), k, _ptr(out_idx), _stream()),
           "asr_sched_select_batched")
    return out_idx


def simulate(trace, n: int, policy: int, cm: np.ndarray, slots: int, want_outputs=True, want_summary=True,
             workspace=None):
    """asr_sched_simulate -> (lat, ttft, summary) device tensors (None where not requested)."""
    torch = _torch()
    dev = trace.device
    lat = torch.empty(max(n, 1), dtype=torch.int64, device=dev)[:n] if want_outputs else None
    ttft = torch.empty(max(n, 1), dtype=torch.int64, device=dev)[:n] if want_outputs else None
    summ = torch.zeros(SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device=dev) if want_summary else None
    if workspace is None:
        workspace = _workspace(workspace_bytes(OP_SIMULATE, n, 1, 0 if want_outputs else 1), dev)
    cm = np.ascontiguousarray(cm, dtype=COST_DTYPE)
    _check(lib().asr_sched_simulate(_ptr(trace), n, policy, cm.ctypes.data, slots, _ptr(lat), _ptr(ttft),
                                    _ptr(summ), _ptr(workspace), workspace.numel(), _stream()),
           "asr_sched_simulate")
    return lat, ttft, summ


def simulate_batched(traces, replicas, n_replicas: int, cms, n_cms: int, total_requests: int, max_slots: int,
                     out_lat=None, out_ttft=None, out_summary=None, workspace=None):
    summary_only = out_lat is None
    if workspace is None:
        workspace = _workspace(workspace_bytes(OP_SIMULATE, total_requests, n_replicas, 1 if summary_only else 0),
                               traces.device)
    _check(lib().asr_sched_simulate_batched(_ptr(traces), _ptr(replicas), n_replicas, _ptr(cms), n_cms,
                                            total_requests, max_slots, _ptr(out_lat), _ptr(out_ttft),
                                            _ptr(out_summary), _ptr(workspace), workspace.numel(), _stream()),
           "asr_sched_simulate_batched")
    return out_lat, out_ttft, out_summary


def make_ext(kv_budget=0, kv_base=0, kv_per_s=0, depth1=0, depth2=0, pol=(0, 0, 0)) -> np.ndarray:
    e = np.zeros(1, dtype=EXT_DTYPE)
    e["kv_budget"], e["kv_base"], e["kv_per_s"] = kv_budget, kv_base, kv_per_s
    e["depth1"], e["depth2"] = depth1, depth2
    e["pol"][0] = pol
    return e


def simulate_batched_ex(traces, replicas, n_replicas: int, cms, exts, n_cms: int, total_requests: int,
                        max_slots: int, out_lat=None, out_ttft=None, out_summary=None, out_preempt=None,
                        workspace=None):
    """asr_sched_simulate_batched_ex: KV-budget preemption and policy switching (exts[cm_id])."""
    summary_only = out_lat is None
    if workspace is None:
        workspace = _workspace(workspace_bytes(OP_SIMULATE_EX, total_requests, n_replicas, 1 if summary_only else 0),
                               traces.device)
    _check(lib().asr_sched_simulate_batched_ex(_ptr(traces), _ptr(replicas), n_replicas, _ptr(cms), _ptr(exts), n_cms,
                                               total_requests, max_slots, _ptr(out_lat), _ptr(out_ttft),
                                               _ptr(out_summary), _ptr(out_preempt), _ptr(workspace),
                                               workspace.numel(), _stream()),
           "asr_sched_simulate_batched_ex")
    return out_lat, out_ttft, out_summary, out_preempt


def itl_batched(traces, replicas, n_replicas: int, cms, n_cms: int, total_requests: int, max_slots: int, pcts,
                out=None, workspace=None):
    """asr_sched_itl_batched -> int64 [n_replicas, n_pct + 2] device tensor: percentiles, gap count, gap sum"""
    torch = _torch()
    pcts = np.ascontiguousarray(pcts, dtype=np.int32)
    if out is None:
        out = torch.empty((max(n_replicas, 1), len(pcts) + 2), dtype=torch.int64, device=traces.device)[:n_replicas]
    if workspace is None:
        workspace = _workspace(workspace_bytes(OP_ITL, total_requests, n_replicas, 0), traces.device)
    _check(lib().asr_sched_itl_batched(_ptr(traces), _ptr(replicas), n_replicas, _ptr(cms), n_cms, total_requests,
                                       max_slots, pcts.ctypes.data, len(pcts), _ptr(out), _ptr(workspace),
                                       workspace.numel(), _stream()), "asr_sched_itl_batched")
    return out


def tpot(trace, n: int, cm: np.ndarray, lat, ttft, out=None):
    """asr_sched_tpot -> int64[n] device tensor, (lat - ttft) / (tokens - 1), -1 for one-token requests"""
    torch = _torch()
    if out is None:
        out = torch.empty(max(n, 1), dtype=torch.int64, device=trace.device)[:n]
    cm = np.ascontiguousarray(cm, dtype=COST_DTYPE)
    _check(lib().asr_sched_tpot(_ptr(trace), n, cm.ctypes.data, _ptr(lat), _ptr(ttft), _ptr(out), _stream()),
           "asr_sched_tpot")
    return out


def estimate(recs, n: int, kappa_milli_by_lang, lang=None, speech_ms=None):
    """asr_sched_estimate: rewrites est of the device records in place"""
    kap = np.ascontiguousarray(kappa_milli_by_lang, dtype=np.int32)
    _check(lib().asr_sched_estimate(_ptr(recs), n, kap.ctypes.data, kap.shape[0], _ptr(lang), _ptr(speech_ms),
                                    _stream()), "asr_sched_estimate")
    return recs


def percentiles(values, seg_off, n_seg: int, pcts, out=None):
    torch = _torch()
    pcts = np.ascontiguousarray(pcts, dtype=np.int32)
    if out is None:
        out = torch.empty((max(n_seg, 1), max(len(pcts), 1)), dtype=torch.int64,
                          device=seg_off.device)[:n_seg, :len(pcts)].contiguous()
    _check(lib().asr_sched_percentiles(_ptr(values), _ptr(seg_off), n_seg, pcts.ctypes.data, len(pcts),
                                       _ptr(out), 0, 0, _stream()), "asr_sched_percentiles")
    return out


def gen_trace(seed: int, rate_mhz: int, dist: int, n: int, tables, out=None):
    torch = _torch()
    if out is None:
        out = torch.empty(max(n, 1) * 16, dtype=torch.uint8, device=tables.device)[:n * 16]
    _check(lib().asr_sched_gen_trace(seed, rate_mhz, dist, n, _ptr(tables), _ptr(out), _stream()),
           "asr_sched_gen_trace")
    return out


def gen_trace_batched(specs, n_traces: int, n_per_trace: int, tables, out=None):
    torch = _torch()
    if out is None:
        out = torch.empty(max(n_traces * n_per_trace, 1) * 16, dtype=torch.uint8,
                          device=tables.device)[:n_traces * n_per_trace * 16]
    _check(lib().asr_sched_gen_trace_batched(_ptr(specs), n_traces, n_per_trace, _ptr(tables), _ptr(out),
                                             _stream()), "asr_sched_gen_trace_batched")
    return out


def gen_queues(seed: int, first: int, n: int, now: int, tables, out=None):
    torch = _torch()
    if out is None:
        out = torch.empty(max(n, 1) * 16, dtype=torch.uint8, device=tables.device)[:n * 16]
    _check(lib().asr_sched_gen_queues(seed, first, n, now, _ptr(tables), _ptr(out), _stream()),
           "asr_sched_gen_queues")
    return out


# ---------------------------------------------------------------------------
# synchronous host-buffer calls
# ---------------------------------------------------------------------------

def _host_ptr(a):
    """numpy array or (pinned) CPU torch tensor -> address"""
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()


def sweep_host(specs, n_per_trace: int, tables, policies, slots: int, cm, out_summary=None):
    """asr_sched_sweep_host: all arguments HOST.  -> SUMMARY_DTYPE[n_traces*n_policies]."""
    specs = np.ascontiguousarray(specs, dtype=SPEC_DTYPE)
    policies = np.ascontiguousarray(policies, dtype=np.int32)
    cm = np.ascontiguousarray(cm, dtype=COST_DTYPE)
    tables = np.ascontiguousarray(tables, dtype=TABLES_DTYPE)
    n_rep = specs.shape[0] * policies.shape[0]
    if out_summary is None:
        out_summary = np.zeros(n_rep, dtype=SUMMARY_DTYPE)
    _check(lib().asr_sched_sweep_host(specs.ctypes.data, specs.shape[0], n_per_trace, tables.ctypes.data,
                                      policies.ctypes.data, policies.shape[0], slots, cm.ctypes.data,
                                      _host_ptr(out_summary)), "asr_sched_sweep_host")
    return out_summary


def trim_scratch():
    _check(lib().asr_sched_trim_scratch(), "asr_sched_trim_scratch")


def select_host(keys, n_queues: int, q_len: int, policy: int, now: int, k: int, out_idx=None):
    """asr_sched_select_host: keys / out_idx HOST (numpy or pinned torch CPU tensors)."""
    if out_idx is None:
        out_idx = np.empty((n_queues, k), dtype=np.int32)
    _check(lib().asr_sched_select_host(_host_ptr(keys), n_queues, q_len, policy, now, k, _host_ptr(out_idx)),
           "asr_sched_select_host")
    return out_idx
