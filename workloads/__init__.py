"""Seeded synthetic INPUTS shared by the oracle tests and the CUDA tests/bench.

This module holds none of the method's arithmetic: no comparator, no
simulator, no percentile, no counter-RNG mixing, no table interpolation.
It only produces *data* that both sides receive as inputs:

* the two quantile tables the trace generator interpolates (built once, in
  float64, with the Python stdlib only -- ``statistics.NormalDist``,
  ``math``), standing in for the duration distribution of LibriSpeech
  test-clean (1-35 s, right-skewed) and for the unit
  exponential that a Poisson arrival process draws;
* the parameter sets of BASELINE.json's five configs (seeds, rates, slots);
* hand-built stress traces S1-S5 made with numpy's
  seeded PCG64, because configs 1-3 never queue deeply enough to exercise
  the policy.

Neither ``oracle`` nor ``paper_2603_11273_b200`` is imported here.
"""
from __future__ import annotations

import functools
import math
import statistics
import zlib

import numpy as np

REQ = np.dtype([("arrival_us", "<i8"), ("dur_ms", "<i4"), ("est", "<i4")])

FCFS, SJF, HRRN = 0, 1, 2
POLICY_NAMES = {FCFS: "fcfs", SJF: "sjf", HRRN: "hrrn"}
DIST_LOGNORMAL, DIST_UNIFORM = 0, 1

# BASELINE.json configs[0]: admission encoder cost 20,000 + 2*dur_ms us; an
# iteration costs 8,000 + 50*running us; tokens = 1 + 4*dur_ms/1000.
# (enc_base_us, enc_per_ms_us, iter_base_us, iter_per_running_us, tok_base, tok_per_s)
CONFIG_COST = (20000, 2, 8000, 50, 1, 4)
# PAPER.md:25 Fig. 1 toy: 1 s encoder, 0.1 s per token, 5 tokens per second of audio
TOY_COST = (1000000, 0, 100000, 0, 0, 5)

TABLE_CELLS = 4096


@functools.lru_cache(maxsize=None)
def ln_dur_table() -> np.ndarray:
    """uint32[4097]: quantiles (ms) of lognormal(mu=ln 6 s, sigma=0.6) clipped
    to [1000, 35000] ms at probabilities j/4096 (BASELINE.json configs[0])."""
    nd = statistics.NormalDist()
    t = np.empty(TABLE_CELLS + 1, dtype=np.uint32)
    t[0], t[TABLE_CELLS] = 1000, 35000
    for j in range(1, TABLE_CELLS):
        v = round(6000.0 * math.exp(0.6 * nd.inv_cdf(j / TABLE_CELLS)))
        t[j] = min(35000, max(1000, v))
    return t


@functools.lru_cache(maxsize=None)
def exp_table() -> np.ndarray:
    """uint32[4097]: Q32 quantiles of the unit exponential truncated to
    [0, ln 2): round(-ln(1 - j/8192) * 2^32); entry 4096 is ln 2 in Q32."""
    t = np.empty(TABLE_CELLS + 1, dtype=np.uint32)
    for j in range(TABLE_CELLS + 1):
        t[j] = round(-math.log1p(-j / (2.0 * TABLE_CELLS)) * 4294967296.0)
    return t


def table_checksum() -> int:
    return zlib.crc32(ln_dur_table().tobytes() + exp_table().tobytes())


RATES_MHZ = (500, 1000, 1500, 2000, 2500, 3000, 3500, 4000)  # 0.5 .. 4 req/s


def config1():
    """Single replica x 3 policies, 1,000 requests, seed 0, 2 req/s, 16 slots."""
    return dict(name="config1", seed=0, n=1000, rate_mhz=2000, dist=DIST_LOGNORMAL,
                slots=16, policies=(FCFS, SJF, HRRN), cost=CONFIG_COST)


def config2():
    """Drift workload: 3,000 requests, uniform durations, 8 rates x 3 policies, seed 1."""
    return dict(name="config2", seed=1, n=3000, rates_mhz=RATES_MHZ, dist=DIST_UNIFORM,
                slots=16, policies=(FCFS, SJF, HRRN), cost=CONFIG_COST)


def config3(n_seeds: int = 4096, n: int = 10000, seed0: int = 0):
    """Replica sweep: seeds x 8 rates x 3 policies, 32 slots.  The first half of
    the seeds is lognormal, the second half uniform.  ``seed0`` shifts the seed
    block (used to give every rank of a multi-GPU run its own replicas)."""
    return dict(name="config3", n_seeds=n_seeds, seed0=seed0, n=n, rates_mhz=RATES_MHZ,
                slots=32, policies=(FCFS, SJF, HRRN), cost=CONFIG_COST)


def config3_traces(cfg):
    """-> (seed[T], rate_mhz[T], dist[T]) for the T = n_seeds*8 distinct traces,
    seed-major; trace (s, r) has index s*8 + r."""
    S, R = cfg["n_seeds"], len(cfg["rates_mhz"])
    seeds = np.repeat(np.arange(S, dtype=np.uint64) + np.uint64(cfg["seed0"]), R)
    rates = np.tile(np.asarray(cfg["rates_mhz"], dtype=np.int32), S)
    dist = np.repeat((np.arange(S) >= S // 2).astype(np.int32), R)
    return seeds, rates, dist


def config4(n: int = 1000000):
    """Deep backlog: one trace, Poisson at 1.3x the 256-slot capacity
    (27.237 req/s analytic) -> 35,408 mHz; HRRN and SJF."""
    return dict(name="config4", seed=4, n=n, rate_mhz=35408, dist=DIST_LOGNORMAL,
                slots=256, policies=(HRRN, SJF), cost=CONFIG_COST)


def config5(n_queues: int = 65536, q_len: int = 4096):
    """Standalone batched select: queues x waiting requests, now = 1e10 us, k = 32."""
    return dict(name="config5", seed=5, n_queues=n_queues, q_len=q_len,
                now=10_000_000_000, k=32, policies=(HRRN, SJF))


# ---------------------------------------------------------------------------
# Stress traces (not part of the timed metric): numpy PCG64, fixed seeds.
# ---------------------------------------------------------------------------

def _trace(arrival_us, dur_ms, est=None) -> np.ndarray:
    out = np.zeros(len(arrival_us), dtype=REQ)
    out["arrival_us"] = np.asarray(arrival_us, dtype=np.int64)
    out["dur_ms"] = np.asarray(dur_ms, dtype=np.int32)
    out["est"] = out["dur_ms"] if est is None else np.asarray(est, dtype=np.int32)
    return out


def _poisson_arrivals(rng, n, rate_per_s):
    gaps = np.floor(rng.exponential(1e6 / rate_per_s, size=n)).astype(np.int64)
    return np.cumsum(gaps)


def _lognormal_ms(rng, n):
    d = np.exp(rng.normal(math.log(6000.0), 0.6, size=n))
    return np.clip(np.rint(d), 1000, 35000).astype(np.int32)


def stress_trace(kind: str, n: int, seed: int, rate_per_s: float = 22.0) -> np.ndarray:
    """S1-S5 of SURVEY.md section 8d plus a few tie-heavy shapes."""
    rng = np.random.Generator(np.random.PCG64(seed))
    if kind == "lognormal":          # S1/S2: overload near / above capacity
        return _trace(_poisson_arrivals(rng, n, rate_per_s), _lognormal_ms(rng, n))
    if kind == "uniform":            # S4
        return _trace(_poisson_arrivals(rng, n, rate_per_s),
                      rng.integers(1000, 35001, size=n))
    if kind == "burst":              # S3: everything arrives at once
        return _trace(np.zeros(n, dtype=np.int64), _lognormal_ms(rng, n))
    if kind == "six":                # S5: durations {5,...,30} s
        return _trace(_poisson_arrivals(rng, n, rate_per_s),
                      rng.integers(1, 7, size=n) * 5000)
    if kind == "equal_est":          # S5: HRRN must equal FCFS
        d = _lognormal_ms(rng, n)
        return _trace(_poisson_arrivals(rng, n, rate_per_s), d, est=np.full(n, 7000))
    if kind == "clumped":            # many identical arrival stamps + few durations
        arr = np.sort(rng.integers(0, max(2, n // 8), size=n)) * 250000
        return _trace(arr, rng.integers(1, 4, size=n) * 4000)
    if kind == "misest":             # est decoupled from dur (PAPER.md:144 silence)
        d = _lognormal_ms(rng, n)
        est = np.maximum(0, (d * rng.uniform(0.2, 1.8, size=n)).astype(np.int32) // 40)
        return _trace(_poisson_arrivals(rng, n, rate_per_s), d, est=est)
    raise ValueError(kind)


# A.3: a smaller model that saturates later (~21 vs ~18 req/s).  Same shape of cost,
# the fixed terms scaled by 0.85: analytic capacity at 16 slots 22.2 req/s (lognormal) against 19.8 for CONFIG_COST.
MEDIUM_COST = (17000, 2, 6800, 42, 1, 4)


def burst_config(n: int = 500):
    """A.2: all n requests arrive at once (request rate = inf), LibriSpeech-like
    durations, the setup of config 1 otherwise."""
    return dict(name="burst", seed=12, n=n, slots=16, policies=(FCFS, SJF, HRRN), cost=CONFIG_COST)


def burst_trace(cfg=None) -> np.ndarray:
    cfg = cfg or burst_config()
    return stress_trace("burst", cfg["n"], cfg["seed"])


def stress_queue(kind: str, n: int, seed: int, now: int) -> np.ndarray:
    """Unsorted waiting queues for the standalone select, with injected ties."""
    rng = np.random.Generator(np.random.PCG64(seed))
    arr = rng.integers(0, max(1, now), size=n, dtype=np.int64)
    if kind == "random":
        return _trace(arr, _lognormal_ms(rng, n))
    if kind == "six":                # massive SJF ties on est
        return _trace(arr, rng.integers(1, 7, size=n) * 5000)
    if kind == "proportional":       # massive exact HRRN ratio ties: w = c * e
        e = rng.integers(1, 9, size=n).astype(np.int64) * 1000
        c = rng.integers(1, 4, size=n).astype(np.int64)
        return _trace(now - c * e, e.astype(np.int32))
    if kind == "identical":          # every key equal -> index order decides
        return _trace(np.full(n, now // 2, dtype=np.int64), np.full(n, 5000))
    if kind == "few_arrivals":       # few distinct stamps, few distinct est
        return _trace(rng.integers(0, 5, size=n, dtype=np.int64) * (now // 8),
                      rng.integers(1, 4, size=n) * 3000)
    if kind == "future":             # some arrivals after `now` (w reads as 0)
        arr2 = rng.integers(0, 2 * max(1, now), size=n, dtype=np.int64)
        return _trace(arr2, _lognormal_ms(rng, n))
    if kind == "est_edge":           # est 0 / negative read as 1; large est
        est = rng.integers(-2, 3, size=n).astype(np.int32)
        est[rng.random(n) < 0.3] = 1 << 24
        return _trace(arr, _lognormal_ms(rng, n), est=est)
    raise ValueError(kind)


def shard(n_units: int, rank: int, world: int):
    """Contiguous block partition of independent units (replicas, queues)."""
    base, extra = divmod(n_units, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)
