"""Pins for the oracle's counter-based generator (
PAPER.md:80,96,98).  Closed forms are evaluated here with the stdlib only."""
import math
import os
from statistics import NormalDist

import numpy as np

import oracle as orc
import workloads as wl

KAT = os.path.join(os.path.dirname(__file__), "golden", "splitmix64_kat.txt")
G = 0x9E3779B97F4A7C15
M = (1 << 64) - 1


def test_fmix64_is_splitmix64_output_function():
    want = [int(l) for l in open(KAT) if l.strip() and not l.startswith("#")]
    assert [orc.fmix64(((i + 1) * G) & M) for i in range(3)] == want


def test_mix64_streams_are_distinct_and_stable():
    seen = {orc.mix64(s, st, i) for s in range(8) for st in range(4) for i in range(64)}
    assert len(seen) == 8 * 4 * 64
    # adjacent seeds are not shifted copies of one another
    a = [orc.mix64(3, 0, i) for i in range(1, 65)]
    b = [orc.mix64(4, 0, i) for i in range(0, 64)]
    assert a != b
    # bit balance over many draws
    bits = np.array([[(orc.mix64(9, 2, i) >> b) & 1 for b in range(64)] for i in range(4000)])
    assert np.all(np.abs(bits.mean(axis=0) - 0.5) < 0.04)


def test_tables_shape_and_monotone(tables):
    ln_dur, exp_t = tables
    assert ln_dur.shape == exp_t.shape == (4097,)
    assert ln_dur[0] == 1000 and ln_dur[-1] == 35000 and np.all(np.diff(ln_dur.astype(np.int64)) >= 0)
    assert exp_t[0] == 0 and exp_t[-1] == round(math.log(2) * 2**32)
    assert np.all(np.diff(exp_t.astype(np.int64)) > 0)
    assert ln_dur[2048] == 6000  # the median of lognormal(ln 6 s, .) is 6 s


def clipped_lognormal_moments(mu, sig, a, b):
    """E[clip(X,a,b)] and sd for X ~ lognormal(mu, sig): partial expectations
    E[X^k; a<=X<=b] = exp(k mu + k^2 sig^2/2) [Phi((ln b - mu - k sig^2)/sig) - Phi((ln a - ...)/sig)]."""
    Phi = NormalDist().cdf
    za, zb = (math.log(a) - mu) / sig, (math.log(b) - mu) / sig
    pa, pb = Phi(za), 1 - Phi(zb)
    def part(k):
        return math.exp(k * mu + k * k * sig * sig / 2) * (Phi(zb - k * sig) - Phi(za - k * sig))
    m1 = a * pa + b * pb + part(1)
    m2 = a * a * pa + b * b * pb + part(2)
    return m1, math.sqrt(m2 - m1 * m1), pa, pb


def test_lognormal_durations_match_closed_form(tables):
    ln_dur, exp_t = tables
    n = 400_000
    tr = orc.gen_trace(123, 2000, orc.DIST_LOGNORMAL, n, ln_dur, exp_t)
    d = tr["dur_ms"].astype(np.float64)
    m1, sd, pa, pb = clipped_lognormal_moments(math.log(6000.0), 0.6, 1000.0, 35000.0)
    assert abs(m1 - 7172) < 2 and abs(sd - 4638) < 3          # SURVEY.md 8c-P figures
    assert abs(d.mean() - m1) < 35                              # se ~ 7.3
    assert abs(d.std() - sd) < 60
    assert d.min() >= 1000 and d.max() <= 35000
    assert abs(np.median(d) - 6000) < 40
    # quantile check against the lognormal CDF at a few points
    for x in (2000, 4000, 9000, 15000, 25000):
        want = NormalDist().cdf((math.log(x) - math.log(6000.0)) / 0.6)
        assert abs((d <= x).mean() - want) < 0.004
    assert np.array_equal(tr["est"], tr["dur_ms"])


def test_uniform_durations(tables):
    ln_dur, exp_t = tables
    tr = orc.gen_trace(7, 1000, orc.DIST_UNIFORM, 400_000, ln_dur, exp_t)
    d = tr["dur_ms"].astype(np.float64)
    assert d.min() == 1000 and d.max() == 35000
    assert abs(d.mean() - 18000) < 60            # sd 9815.2 / sqrt(n) = 15.5
    assert abs(d.std() - 9815.2) < 50


def test_poisson_gaps(tables):
    ln_dur, exp_t = tables
    n = 400_000
    for rate_mhz in (500, 4000, 35408):
        tr = orc.gen_trace(rate_mhz, rate_mhz, orc.DIST_UNIFORM, n, ln_dur, exp_t)
        arr = tr["arrival_us"]
        gaps = np.diff(np.concatenate([[0], arr])).astype(np.float64)
        mean_gap = 10**9 // rate_mhz
        assert (gaps >= 0).all()                                   # non-decreasing
        assert abs(gaps.mean() / mean_gap - 1) < 0.01              # se 0.16%
        assert abs(gaps.std() / mean_gap - 1) < 0.02               # exponential: cv = 1
        assert abs((gaps > mean_gap).mean() - math.exp(-1)) < 0.004
        assert abs((gaps > 3 * mean_gap).mean() - math.exp(-3)) < 0.002
        # memoryless: no serial correlation
        assert abs(np.corrcoef(gaps[:-1], gaps[1:])[0, 1]) < 0.01


def test_common_random_numbers_across_rates_and_determinism(tables):
    ln_dur, exp_t = tables
    a = orc.gen_trace(42, 1000, orc.DIST_LOGNORMAL, 5000, ln_dur, exp_t)
    b = orc.gen_trace(42, 1000, orc.DIST_LOGNORMAL, 5000, ln_dur, exp_t)
    c = orc.gen_trace(42, 2000, orc.DIST_LOGNORMAL, 5000, ln_dur, exp_t)
    assert np.array_equal(a, b)
    assert np.array_equal(a["dur_ms"], c["dur_ms"])      # PAPER.md:98 identical sequences
    # halving the mean gap halves every gap up to the floor
    ga = np.diff(np.concatenate([[0], a["arrival_us"]]))
    gc = np.diff(np.concatenate([[0], c["arrival_us"]]))
    assert np.all(np.abs(ga - 2 * gc) <= 1)
    # a prefix of a longer trace is the shorter trace
    assert np.array_equal(a[:100], orc.gen_trace(42, 1000, orc.DIST_LOGNORMAL, 100, ln_dur, exp_t))


def test_queue_generator(tables):
    ln_dur, _ = tables
    now = 10**10
    q = orc.gen_queue(5, 0, 200_000, now, ln_dur)
    a = q["arrival_us"].astype(np.float64)
    assert a.min() >= 0 and a.max() < now
    assert abs(a.mean() / now - 0.5) < 0.003 and abs(a.std() / now - 12 ** -0.5) < 0.003
    assert np.array_equal(q[1000:1100], orc.gen_queue(5, 1000, 100, now, ln_dur))
    m1, _, _, _ = clipped_lognormal_moments(math.log(6000.0), 0.6, 1000.0, 35000.0)
    assert abs(q["dur_ms"].mean() - m1) < 45
