"""Pins for the oracle's comparator and selector.

The independent reference here evaluates the paper's HRRN formula
(wait + est) / est as an exact Fraction and sorts plain Python tuples -- it
never cross-multiplies and never calls the oracle's comparator."""
import itertools
from fractions import Fraction

import numpy as np
import pytest

import oracle as orc
import workloads as wl


def ref_order(q, policy, now):
    """Paper's keys, written out: FCFS arrival order; SJF tuple
    (est, arrival, id); HRRN ratio, highest first."""
    keys = []
    for i, r in enumerate(q):
        a, e = int(r["arrival_us"]), max(1, int(r["est"]))
        if policy == orc.FCFS:
            keys.append((a, i))
        elif policy == orc.SJF:
            keys.append((e, a, i))
        else:
            w = max(0, now - a)
            keys.append((-Fraction(w + e, e), a, i))
    return [k[-1] for k in sorted(keys)]


def rand_queue(rng, n, now, ties):
    if ties:
        arr = rng.integers(0, 4, size=n) * (now // 4)
        est = rng.integers(1, 4, size=n) * 1000
    else:
        arr = rng.integers(0, now + 1, size=n)
        est = rng.integers(1, 40000, size=n)
    return orc.make_trace(arr, est)


@pytest.mark.parametrize("policy", [orc.FCFS, orc.SJF, orc.HRRN])
@pytest.mark.parametrize("ties", [False, True])
def test_select_matches_fraction_sort(policy, ties):
    rng = np.random.default_rng(11 + policy)
    for n in [0, 1, 2, 3, 5, 8, 17, 64, 200]:
        now = int(rng.integers(1, 10**7))
        q = rand_queue(rng, n, now, ties)
        want = ref_order(q, policy, now)
        for k in {0, 1, min(n, 3), n, n + 2}:
            got = orc.select(q, policy, now, k)
            exp = (want + [-1] * k)[:k] if k > n else want[:k]
            assert list(got) == exp


def test_better_is_strict_total_order():
    rng = np.random.default_rng(5)
    now = 10**6
    q = rand_queue(rng, 12, now, ties=True)
    for policy in (orc.FCFS, orc.SJF, orc.HRRN):
        for i, j in itertools.permutations(range(12), 2):
            assert orc.better(q, i, j, policy, now) != orc.better(q, j, i, policy, now)
        for i in range(12):
            assert not orc.better(q, i, i, policy, now)


def test_prefix_property_and_k_padding():
    rng = np.random.default_rng(6)
    q = rand_queue(rng, 50, 10**6, ties=True)
    for policy in (orc.FCFS, orc.SJF, orc.HRRN):
        full = orc.select(q, policy, 10**6, 50)
        for k in range(0, 51, 7):
            assert list(orc.select(q, policy, 10**6, k)) == list(full[:k])
        assert list(orc.select(q, policy, 10**6, 53)[50:]) == [-1, -1, -1]


def test_hrrn_equal_est_is_fcfs():
    # north_star invariant: HRRN with equal lengths equals FCFS
    rng = np.random.default_rng(7)
    arr = rng.integers(0, 10**6, size=300)
    q = orc.make_trace(arr, np.full(300, 7000))
    a = orc.select(q, orc.HRRN, 10**6, 300)
    b = orc.select(q, orc.FCFS, 10**6, 300)
    assert list(a) == list(b)


def test_sjf_independent_of_now_and_hrrn_scale_invariant():
    rng = np.random.default_rng(8)
    q = rand_queue(rng, 200, 10**6, ties=False)
    assert list(orc.select(q, orc.SJF, 5, 200)) == list(orc.select(q, orc.SJF, 10**9, 200))
    # DESIGN.md S4: (w + c*e)/(c*e) is monotone in w/e for every c > 0
    q3 = q.copy()
    q3["est"] = q["est"] * 3
    assert list(orc.select(q, orc.HRRN, 10**6, 200)) == list(orc.select(q3, orc.HRRN, 10**6, 200))


def test_permutation_equivariance():
    rng = np.random.default_rng(9)
    n, now = 100, 10**7
    q = orc.make_trace(rng.permutation(10**6)[:n] * 7, rng.integers(1, 30000, size=n))
    perm = rng.permutation(n)
    qp = q[perm]
    for policy in (orc.FCFS, orc.SJF, orc.HRRN):
        a = orc.select(q, policy, now, n)
        b = orc.select(qp, policy, now, n)
        assert [int(perm[j]) for j in b] == list(a)


def test_hand_built_ties():
    now = 10000
    # proportional pairs (w, e) = (2000, 2000) and (1000, 1000): ratios equal
    # (both 2) -> earlier arrival wins: arrival 8000 (w=2000) before 9000.
    q = orc.make_trace([9000, 8000, 9000, 0], [1000, 2000, 1000, 10000])
    #   idx0: w=1000 e=1000 ratio 2 ; idx1: w=2000 e=2000 ratio 2
    #   idx2: same as idx0          ; idx3: w=10000 e=10000 ratio 2
    assert list(orc.select(q, orc.HRRN, now, 4)) == [3, 1, 0, 2]
    # SJF: equal est -> earlier arrival -> lower index
    q = orc.make_trace([50, 10, 10, 70], [3000, 3000, 3000, 2000])
    assert list(orc.select(q, orc.SJF, now, 4)) == [3, 1, 2, 0]
    # est < 1 reads as 1 (PAPER.md:260 max(1, .)): est 0 and est 1 tie -> arrival
    q = orc.make_trace([5, 4, 3], [1000, 1000, 1000], est=[0, 1, -7])
    assert list(orc.select(q, orc.SJF, now, 3)) == [2, 1, 0]
    # arrival after now: w = 0 -> lowest ratio, ordered by arrival among them
    q = orc.make_trace([now + 5, now + 1, now - 1], [1000, 1000, 1000])
    assert list(orc.select(q, orc.HRRN, now, 3)) == [2, 1, 0]


def test_hrrn_needs_exact_arithmetic():
    # Two response ratios inside the documented bounds (wait < 2^38 us,
    # est <= 2^24) whose cross-products differ by exactly 1: float64 division
    # (Listing 3) cannot separate them, integers can (S5).
    m = 1 << 14
    e_a, e_b = (1 << 23) + 1, 1 << 23
    w_a, w_b = e_a * m - 1, e_b * m - 1
    assert w_a * e_b - w_b * e_a == 1                 # a is better by one unit
    assert (w_a + e_a) / e_a == (w_b + e_b) / e_b     # ...and doubles tie
    now = 1 << 38
    q = orc.make_trace([now - w_b, now - w_a], [e_b, e_a])   # b first in the array
    assert list(orc.select(q, orc.HRRN, now, 2)) == [1, 0]


def test_products_beyond_the_documented_bounds_are_reported():
    """the oracle multiplies in 128 bits and reports a cross-product that would not fit the
    boundary's int64 contract (wait < 2^38, est <= 2^24 => wait * est < 2^62) instead of silently ordering it."""
    e_max, now = 1 << 24, (1 << 38) - 1
    inside = orc.make_trace([0, 1, now - 5], [e_max, e_max - 1, 7])        # largest legal products
    assert orc.bound_violations() == orc.bound_violations()
    before = orc.bound_violations()
    assert list(orc.select(inside, orc.HRRN, now, 3)) == ref_order(inside, orc.HRRN, now)
    assert orc.bound_violations() == before
    outside = orc.make_trace([0, 1], [e_max, e_max])                        # wait 2^38: product 2^62
    with pytest.raises(ValueError, match="rc=-4"):
        orc.select(outside, orc.HRRN, 1 << 38, 2)
    assert orc.bound_violations() > before
    # the other policies never multiply: no report
    assert list(orc.select(outside, orc.SJF, 1 << 38, 2)) == [0, 1]
    assert list(orc.select(outside, orc.FCFS, 1 << 38, 2)) == [0, 1]
    # and the simulator passes the report on: one slot, two requests wait 2^38 us behind a long first one
    cm = orc.cost(1 << 38, 0, 10, 0, 1, 0)
    tr = orc.make_trace([0, 0, 0], [1, 1, 1], est=[1, e_max, e_max])
    with pytest.raises(ValueError, match="rc=-4"):
        orc.simulate(tr, orc.HRRN, cm, 1)
    orc.simulate(tr, orc.FCFS, cm, 1)


def test_six_duration_ties_stress():
    # PAPER.md:96 synthetic split {5,...,30} s -> massive SJF ties
    q = wl.stress_queue("six", 500, 3, 10**8)
    for policy in (orc.SJF, orc.HRRN):
        assert list(orc.select(q, policy, 10**8, 500)) == ref_order(q, policy, 10**8)
