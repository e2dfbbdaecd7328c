"""N > 1 host logic on CPU (gloo, world size 2): shard ranges tile the slot range, the per-rank benchmark rows are the rows a
single process would draw for those global indices, and the timing reductions are max / sum over ranks."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_2509_04336_b200 import dist as D, workloads as W
rank, world, local = D.init("gloo")
assert world == 2 and dist.get_backend() == "gloo"
n = 701
lo, hi = D.shard_range(n, rank, world)
rows = W.uniform_rows(lo, hi, 11, seed=5)
full = W.uniform_rows(0, n, 11, seed=5)
assert np.array_equal(rows, full[lo:hi])
gathered = [None] * world
dist.all_gather_object(gathered, (lo, hi))
D.barrier()
mx = D.max_over_ranks(10.0 + rank)
sm = D.sum_over_ranks(hi - lo)
if rank == 0:
    print(json.dumps(dict(ranges=gathered, mx=mx, sm=sm)))
D.finalize()
"""


def test_gloo_world2_sharding(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(script)]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=240, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r["ranges"] == [[0, 351], [351, 701]] and r["mx"] == 11.0 and r["sm"] == 701.0


def test_shard_ranges_tile_any_partition():
    from paper_2509_04336_b200 import dist as D
    for n in (1, 2, 500, 700, 65536, 131071):
        for world in (1, 2, 3, 4, 8):
            edges = [D.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[i][1] == edges[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1


def test_uniform_rows_are_index_keyed():
    from paper_2509_04336_b200 import workloads as W
    a = W.uniform_rows(0, 100, 11, seed=3)
    b = W.uniform_rows(40, 60, 11, seed=3)
    assert np.array_equal(a[40:60], b) and a.min() > 0.0 and a.max() < 1.0
    assert not np.array_equal(W.uniform_rows(0, 10, 11, seed=4), a[:10])


def test_bench_gpus_flag_dispatch():
    """`bench.py --gpus N`: without a launcher and N > 1 it starts N ranks itself (torch.distributed.run, one per GPU); under a
    launcher the flag must agree with WORLD_SIZE; both arms read the flag the same way; the traffic figure comes from profiles/."""
    import argparse
    import sys
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    ns = argparse.Namespace
    assert bench.resolve_world(ns(gpus=1), {}) == "run"
    assert bench.resolve_world(ns(gpus=4), {}) == "spawn"
    assert bench.resolve_world(ns(gpus=4), {"WORLD_SIZE": "4"}) == "run"
    with pytest.raises(SystemExit):
        bench.resolve_world(ns(gpus=8), {"WORLD_SIZE": "2"})
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "7", "--impl", "reference"], port=29999)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29999"
    assert cmd[-6:] == ["--gpus", "4", "--steps", "7", "--impl", "reference"] and cmd[-7].endswith("bench.py")
    tr, f = bench.traffic_from_profile("k_bins_lp")
    assert f and f.startswith("profiles/") and 1e6 < tr < 1e9
    assert bench._profile_key("r02b_x") > bench._profile_key("r01ai_x") > bench._profile_key("r01z_x")
