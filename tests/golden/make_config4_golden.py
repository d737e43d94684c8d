#!/usr/bin/env python
"""Writes tests/golden/config4_oracle.txt: the CPU oracle's results on
BASELINE.json configs[3] (deep backlog: 1,000,000 requests, 256 slots, Poisson
arrivals at 1.3x capacity, HRRN and SJF) at FULL size.

The oracle steps one engine iteration at a time and re-sorts the whole waiting
queue at every admission, so the full config takes tens of minutes per policy
on one core -- too slow for a test, which is why its results are stored.  This
script calls only `oracle/` and `workloads/` (the seeded input recipe); nothing
in the file it writes comes from the CUDA path.

    python tests/golden/make_config4_golden.py [--n 1000000]

Stored per policy: the summary (nearest-rank p50/p90 of E2E latency and TTFT,
first arrival, last completion), three 64-bit digests of each per-request
array (sum, position-weighted sum, xor-rotate chain, all mod 2^64) and every
STRIDE-th element, so that a full-size GPU run can be compared without storing
16 MB of values.
"""
from __future__ import annotations

import argparse
import concurrent.futures as cf
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

STRIDE = 49999   # 1e6 / 49999 -> 21 samples per array


def digests(v: np.ndarray):
    """(sum, sum of (i+1)*v[i], xor of rotl(v[i], i mod 64)) mod 2^64 -- plain definitions"""
    u = v.astype(np.uint64)
    i = np.arange(len(u), dtype=np.uint64)
    with np.errstate(over="ignore"):
        s = int(u.sum(dtype=np.uint64))
        w = int(((i + np.uint64(1)) * u).sum(dtype=np.uint64))
        r = i % np.uint64(64)
        rot = (u << r) | (u >> ((np.uint64(64) - r) % np.uint64(64)))
        x = int(np.bitwise_xor.reduce(rot))
    return s, w, x


def run_policy(args):
    n, pol = args
    import oracle as orc
    import workloads as wl
    cfg = wl.config4(n=n)
    tr = orc.gen_trace(cfg["seed"], cfg["rate_mhz"], cfg["dist"], n, wl.ln_dur_table(), wl.exp_table())
    t0 = time.time()
    lat, ttft, first, end = orc.simulate(tr, pol, orc.cost(*cfg["cost"]), cfg["slots"])
    dt = time.time() - t0
    out = {"policy": pol, "seconds": dt, "first": first, "end": end}
    for name, v in (("lat", lat), ("ttft", ttft)):
        out[name + "_p50"] = orc.percentile(v, 50)
        out[name + "_p90"] = orc.percentile(v, 90)
        out[name + "_dig"] = digests(v)
        out[name + "_samples"] = [int(x) for x in v[::STRIDE]]
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=1000000)
    ap.add_argument("--out", default=os.path.join(HERE, "config4_oracle.txt"))
    a = ap.parse_args()
    import workloads as wl
    cfg = wl.config4(n=a.n)
    with cf.ProcessPoolExecutor(max_workers=len(cfg["policies"])) as ex:
        res = list(ex.map(run_policy, [(a.n, p) for p in cfg["policies"]]))
    with open(a.out, "w") as f:
        f.write("# CPU oracle on BASELINE.json configs[3] (deep backlog), written by tests/golden/make_config4_golden.py\n")
        f.write("# seed %d rate_mhz %d n %d slots %d cost %s tables_crc32 %d stride %d\n"
                % (cfg["seed"], cfg["rate_mhz"], a.n, cfg["slots"], " ".join(map(str, cfg["cost"])),
                   wl.table_checksum(), STRIDE))
        for r in res:
            f.write("policy %d oracle_seconds %.0f\n" % (r["policy"], r["seconds"]))
            f.write("summary %d %d %d %d %d %d\n" % (r["lat_p50"], r["lat_p90"], r["ttft_p50"], r["ttft_p90"],
                                                    r["first"], r["end"]))
            for name in ("lat", "ttft"):
                f.write("%s_digest %d %d %d\n" % ((name,) + tuple(r[name + "_dig"])))
                f.write("%s_samples %s\n" % (name, " ".join(map(str, r[name + "_samples"]))))
    print("wrote", a.out)


if __name__ == "__main__":
    main()
