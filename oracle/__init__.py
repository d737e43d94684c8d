"""CPU ORACLE -- test infrastructure, NOT the product.

Thin ctypes view of ``asr_oracle.c`` (plain C, gcc).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2603_11273_b200`` and shares no code with the CUDA path.

Record layout (numpy structured dtype ``REQ``): int64 arrival_us, int32 dur_ms,
int32 est -- PAPER.md:57-59, 254-262.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "asr_oracle.c")
_HDR = os.path.join(_HERE, "asr_oracle.h")
# ASR_ORACLE_SANITIZE=1 (set by tests/test_oracle_sanitized.py for a child pytest run): the same source built
# with -fsanitize=address,undefined into a library of its own
_SANITIZE = os.environ.get("ASR_ORACLE_SANITIZE", "") == "1"
_LIB = os.path.join(_HERE, "libasr_oracle_san.so" if _SANITIZE else "libasr_oracle.so")

FCFS, SJF, HRRN, ADAPTIVE = 0, 1, 2, 3
DIST_LOGNORMAL, DIST_UNIFORM = 0, 1

REQ = np.dtype([("arrival_us", "<i8"), ("dur_ms", "<i4"), ("est", "<i4")])


class Cost(C.Structure):
    _fields_ = [
        ("enc_base_us", C.c_int64),
        ("enc_per_ms_us", C.c_int64),
        ("iter_base_us", C.c_int64),
        ("iter_per_running_us", C.c_int64),
        ("tok_base", C.c_int32),
        ("tok_per_s", C.c_int32),
    ]


class Ext(C.Structure):
    """orc_ext_t: KV-memory model (f1) and policy switching (f3)"""
    _fields_ = [
        ("kv_budget", C.c_int64),
        ("kv_base", C.c_int64),
        ("kv_per_s", C.c_int64),
        ("depth1", C.c_int32),
        ("depth2", C.c_int32),
        ("pol", C.c_int32 * 3),
        ("pad", C.c_int32),
    ]


def ext(kv_budget=0, kv_base=0, kv_per_s=0, depth1=0, depth2=0, pol=(0, 0, 0)) -> Ext:
    return Ext(kv_budget, kv_base, kv_per_s, depth1, depth2, (C.c_int32 * 3)(*pol), 0)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no SIMD tricks asked for)."""
    stale = (
        force
        or not os.path.exists(_LIB)
        or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    )
    if stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-g", "-O1"] if _SANITIZE else ["-O2"]
        subprocess.check_call(
            ["gcc"] + san + ["-std=gnu11", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i64, i32, u64, u32 = C.c_void_p, C.c_int64, C.c_int32, C.c_uint64, C.c_uint32
        L.orc_better.restype = C.c_int
        L.orc_better.argtypes = [vp, i64, vp, i64, C.c_int, i64]
        L.orc_bound_violations.restype = i64
        L.orc_bound_violations.argtypes = []
        L.orc_bound_violations_reset.restype = None
        L.orc_bound_violations_reset.argtypes = []
        L.orc_select.restype = C.c_int
        L.orc_select.argtypes = [vp, i64, C.c_int, i64, i32, vp]
        L.orc_simulate.restype = C.c_int
        L.orc_simulate.argtypes = [vp, i64, C.c_int, C.POINTER(Cost), i32, vp, vp,
                                   C.POINTER(i64), C.POINTER(i64)]
        L.orc_percentile.restype = i64
        L.orc_percentile.argtypes = [vp, i64, i32]
        L.orc_simulate_ex.restype = C.c_int
        L.orc_simulate_ex.argtypes = [vp, i64, C.c_int, C.POINTER(Cost), C.POINTER(Ext), i32, vp, vp,
                                      C.POINTER(i64), C.POINTER(i64), C.POINTER(i64)]
        L.orc_itl.restype = C.c_int
        L.orc_itl.argtypes = [vp, i64, C.c_int, C.POINTER(Cost), i32, vp, i32, vp, C.POINTER(i64), C.POINTER(i64)]
        L.orc_tpot.restype = C.c_int
        L.orc_tpot.argtypes = [vp, i64, C.POINTER(Cost), vp, vp, vp]
        L.orc_estimate.restype = C.c_int
        L.orc_estimate.argtypes = [vp, i64, vp, i32, vp, vp]
        L.orc_tokens.restype = i64
        L.orc_tokens.argtypes = [C.POINTER(Cost), i32]
        L.orc_enc_cost.restype = i64
        L.orc_enc_cost.argtypes = [C.POINTER(Cost), i32]
        L.orc_fmix64.restype = u64
        L.orc_fmix64.argtypes = [u64]
        L.orc_mix64.restype = u64
        L.orc_mix64.argtypes = [u64, u32, u64]
        L.orc_gen_trace.restype = C.c_int
        L.orc_gen_trace.argtypes = [u64, i32, i32, i64, vp, vp, vp]
        L.orc_gen_queue.restype = C.c_int
        L.orc_gen_queue.argtypes = [u64, i64, i64, i64, vp, vp]
        _lib = L
    return _lib


def _req(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=REQ)
    return a


def make_trace(arrival_us, dur_ms, est=None) -> np.ndarray:
    arrival_us = np.asarray(arrival_us, dtype=np.int64)
    out = np.zeros(arrival_us.shape[0], dtype=REQ)
    out["arrival_us"] = arrival_us
    out["dur_ms"] = np.asarray(dur_ms, dtype=np.int32)
    out["est"] = out["dur_ms"] if est is None else np.asarray(est, dtype=np.int32)
    return out


def cost(enc_base_us, enc_per_ms_us, iter_base_us, iter_per_running_us, tok_base, tok_per_s) -> Cost:
    return Cost(enc_base_us, enc_per_ms_us, iter_base_us, iter_per_running_us, tok_base, tok_per_s)


def better(q, ia: int, ib: int, policy: int, now: int) -> bool:
    q = _req(q)
    base = q.ctypes.data
    return bool(lib().orc_better(base + 16 * ia, ia, base + 16 * ib, ib, policy, now))


def bound_violations() -> int:
    """HRRN cross-products >= 2^62 seen by this thread's orc_better calls (outside the boundary's bounds)"""
    return int(lib().orc_bound_violations())


def select(q, policy: int, now: int, k: int) -> np.ndarray:
    q = _req(q)
    out = np.empty(k, dtype=np.int32)
    rc = lib().orc_select(q.ctypes.data, q.shape[0], policy, now, k, out.ctypes.data)
    if rc != 0:
        raise ValueError("orc_select rc=%d" % rc)
    return out


def simulate(trace, policy: int, cm: Cost, slots: int):
    """-> (lat[n], ttft[n], first_arrival_us, last_done_us)"""
    trace = _req(trace)
    n = trace.shape[0]
    lat = np.full(n, -1, dtype=np.int64)
    ttft = np.full(n, -1, dtype=np.int64)
    fa, ld = C.c_int64(0), C.c_int64(0)
    rc = lib().orc_simulate(trace.ctypes.data, n, policy, C.byref(cm), slots,
                            lat.ctypes.data, ttft.ctypes.data, C.byref(fa), C.byref(ld))
    if rc != 0:
        raise ValueError("orc_simulate rc=%d" % rc)
    return lat, ttft, fa.value, ld.value


def simulate_ex(trace, policy: int, cm: Cost, ex, slots: int):
    """orc_simulate_ex -> (lat[n], ttft[n], first_arrival_us, last_done_us, n_preempt)"""
    trace = _req(trace)
    n = trace.shape[0]
    lat = np.full(n, -1, dtype=np.int64)
    ttft = np.full(n, -1, dtype=np.int64)
    fa, ld, npre = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    rc = lib().orc_simulate_ex(trace.ctypes.data, n, policy, C.byref(cm), C.byref(ex) if ex is not None else None,
                               slots, lat.ctypes.data, ttft.ctypes.data, C.byref(fa), C.byref(ld), C.byref(npre))
    if rc != 0:
        raise ValueError("orc_simulate_ex rc=%d" % rc)
    return lat, ttft, fa.value, ld.value, npre.value


def itl(trace, policy: int, cm: Cost, slots: int, pcts):
    """orc_itl -> (percentiles list, count, sum) of the inter-token gaps"""
    trace = _req(trace)
    pc = np.ascontiguousarray(pcts, dtype=np.int32)
    out = np.empty(len(pc), dtype=np.int64)
    cnt, sm = C.c_int64(0), C.c_int64(0)
    rc = lib().orc_itl(trace.ctypes.data, trace.shape[0], policy, C.byref(cm), slots, pc.ctypes.data, len(pc),
                       out.ctypes.data, C.byref(cnt), C.byref(sm))
    if rc != 0:
        raise ValueError("orc_itl rc=%d" % rc)
    return [int(x) for x in out], cnt.value, sm.value


def tpot(trace, cm: Cost, lat, ttft) -> np.ndarray:
    trace = _req(trace)
    lat = np.ascontiguousarray(lat, dtype=np.int64)
    ttft = np.ascontiguousarray(ttft, dtype=np.int64)
    out = np.empty(trace.shape[0], dtype=np.int64)
    rc = lib().orc_tpot(trace.ctypes.data, trace.shape[0], C.byref(cm), lat.ctypes.data, ttft.ctypes.data,
                        out.ctypes.data)
    if rc != 0:
        raise ValueError("orc_tpot rc=%d" % rc)
    return out


def estimate(recs, kappa_milli_by_lang, lang=None, speech_ms=None) -> np.ndarray:
    """returns a copy of recs with est = max(1, floor(d_ms * kappa_milli / 1e6))"""
    out = _req(recs).copy()
    kap = np.ascontiguousarray(kappa_milli_by_lang, dtype=np.int32)
    lg = None if lang is None else np.ascontiguousarray(lang, dtype=np.uint8)
    sp = None if speech_ms is None else np.ascontiguousarray(speech_ms, dtype=np.int32)
    rc = lib().orc_estimate(out.ctypes.data, out.shape[0], kap.ctypes.data, kap.shape[0],
                            None if lg is None else lg.ctypes.data, None if sp is None else sp.ctypes.data)
    if rc != 0:
        raise ValueError("orc_estimate rc=%d" % rc)
    return out


def percentile(v, p: int) -> int:
    v = np.ascontiguousarray(v, dtype=np.int64)
    return int(lib().orc_percentile(v.ctypes.data, v.shape[0], p))


def tokens(cm: Cost, dur_ms: int) -> int:
    return int(lib().orc_tokens(C.byref(cm), dur_ms))


def enc_cost(cm: Cost, dur_ms: int) -> int:
    return int(lib().orc_enc_cost(C.byref(cm), dur_ms))


def fmix64(z: int) -> int:
    return int(lib().orc_fmix64(z & 0xFFFFFFFFFFFFFFFF))


def mix64(seed: int, stream: int, i: int) -> int:
    return int(lib().orc_mix64(seed, stream, i))


def _tab(t) -> np.ndarray:
    t = np.ascontiguousarray(t, dtype=np.uint32)
    assert t.shape == (4097,)
    return t


def gen_trace(seed: int, rate_mhz: int, dist: int, n: int, ln_dur, exp_t) -> np.ndarray:
    ln_dur, exp_t = _tab(ln_dur), _tab(exp_t)
    out = np.zeros(n, dtype=REQ)
    rc = lib().orc_gen_trace(seed, rate_mhz, dist, n, ln_dur.ctypes.data,
                             exp_t.ctypes.data, out.ctypes.data)
    if rc != 0:
        raise ValueError("orc_gen_trace rc=%d" % rc)
    return out


def gen_queue(seed: int, first: int, n: int, now: int, ln_dur) -> np.ndarray:
    ln_dur = _tab(ln_dur)
    out = np.zeros(n, dtype=REQ)
    rc = lib().orc_gen_queue(seed, first, n, now, ln_dur.ctypes.data, out.ctypes.data)
    if rc != 0:
        raise ValueError("orc_gen_queue rc=%d" % rc)
    return out
