"""world_size-2 `gloo` test (CPU) of the multi-process plumbing bench.py uses at N > 1: rendezvous,
barrier, max / sum over ranks, and the disjoint unit blocks (replicas and queues are
independent units, no data-path collective).  The reference arm's rank rule is covered too."""
import json
import os
import socket
import subprocess
import sys
import textwrap

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    from paper_2603_11273_b200 import dist as D
    import workloads as wl
    rank, world, local = D.init(backend="gloo")
    D.barrier()
    mx = D.max_over_ranks(10.0 + rank)            # device time of the slowest rank
    sm = D.sum_over_ranks(1.0 + rank)
    seeds = wl.config3(n_seeds=8, n=10, seed0=D.seed_block(rank, 8))
    s, r, d = wl.config3_traces(seeds)
    lo, hi = wl.shard(65536 + 1, rank, world)
    D.barrier()
    print(json.dumps({"rank": rank, "world": world, "max": mx, "sum": sm, "seed_lo": int(min(s)),
                      "seed_hi": int(max(s)), "shard": [lo, hi]}), flush=True)
    D.finalize()
""") % ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_ranks_over_gloo():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda o: o["rank"])
    assert [o["world"] for o in outs] == [2, 2]
    assert [o["max"] for o in outs] == [11.0, 11.0] and [o["sum"] for o in outs] == [3.0, 3.0]
    # weak scaling: rank r simulates its own block of seeds, the blocks do not overlap
    assert (outs[0]["seed_lo"], outs[0]["seed_hi"]) == (0, 7) and (outs[1]["seed_lo"], outs[1]["seed_hi"]) == (8, 15)
    # the generic block partition covers every unit exactly once
    assert outs[0]["shard"][0] == 0 and outs[0]["shard"][1] == outs[1]["shard"][0] and outs[1]["shard"][1] == 65537


def test_shard_partitions_exactly():
    for n in (0, 1, 7, 98304, 65537):
        for world in (1, 2, 3, 8):
            blocks = [wl.shard(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1


def test_reference_arm_only_rank0_prints():
    """bench.py --impl reference under torchrun: rank 0 alone runs and prints, the others exit 0 silently"""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", CUDA_VISIBLE_DEVICES="")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=240)
    assert p.returncode == 0 and p.stdout.strip() == ""
    env["RANK"] = "0"
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--ref-replicas", "16", "--n", "500"], env=env,
                       capture_output=True, text=True, timeout=240)
    assert p.returncode == 0, p.stderr[-2000:]
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "requests/s"
