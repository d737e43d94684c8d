"""Pins for the oracle's nearest-rank percentile (S8)."""
import os

import numpy as np

import oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden", "nearest_rank.txt")


def test_textbook_example():
    vals, cases = None, []
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        if tok[0] == "values":
            vals = [int(x) for x in tok[1:]]
        else:
            cases.append((int(tok[0]), int(tok[1])))
    assert len(cases) == 6
    for shuffled in (vals, vals[::-1], [vals[i] for i in (2, 0, 4, 1, 3)]):
        for p, want in cases:
            assert orc.percentile(shuffled, p) == want


def test_special_cases():
    assert orc.percentile([], 50) == -1
    assert orc.percentile([42], 1) == 42 and orc.percentile([42], 100) == 42
    assert orc.percentile([7] * 13, 90) == 7
    v = np.arange(1000, dtype=np.int64)[::-1] * 3
    assert orc.percentile(v, 50) == 499 * 3      # rank 500 -> index 499
    assert orc.percentile(v, 90) == 899 * 3
    assert orc.percentile(v, 100) == 999 * 3 and orc.percentile(v, 1) == 9 * 3


def test_against_sort_and_count_definition():
    # definition: smallest value v such that at least p% of the data are <= v
    rng = np.random.default_rng(3)
    for n in (1, 2, 3, 10, 99, 100, 101, 1234):
        v = rng.integers(-10**12, 10**12, size=n)
        for p in (1, 25, 50, 90, 99, 100):
            got = orc.percentile(v, p)
            assert got in v
            assert np.count_nonzero(v <= got) * 100 >= p * n
            smaller = v[v < got]
            if smaller.size:
                assert np.count_nonzero(v <= smaller.max()) * 100 < p * n
