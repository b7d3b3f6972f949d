"""N > 1 path on CPU: world-size-2 `gloo` processes shard one global batch (no data-path collective),
and the max-over-ranks reduction bench.py uses for its timing works across ranks."""
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np
import torch
import torch.distributed as dist
from paper_2507_12349_b200.sharding import shard_bounds, shard_vertices, max_over_ranks
from cos_workloads import get_config, draw_vertices
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
w = get_config(1).scaled(batch=101)
v = draw_vertices(w)
b0, b1, mine = shard_vertices(v, w.batch, rank, world)      # the slicing `bench.py --scaling strong` does
assert (b0, b1) == shard_bounds(w.batch, rank, world)
assert mine["sites"].shape == (w.n, 2, b1 - b0) and mine["sites"].flags["C_CONTIGUOUS"]
assert np.array_equal(mine["sites"], v["sites"][..., b0:b1])
local = mine["tau"]
# every rank reports (bounds, checksum of its slice); gathered only for the TEST, not on the data path
objs = [None] * world
dist.all_gather_object(objs, (b0, b1, float(local.sum())))
ms = max_over_ranks([10.0 + rank, 5.0 - rank])
if rank == 0:
    print(json.dumps({"shards": objs, "ms": ms, "total": float(v["tau"].sum())}))
dist.barrier()
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_bounds_cover_exactly_once():
    from paper_2507_12349_b200.sharding import shard_bounds
    for batch in (0, 1, 7, 64, 8192, 65537):
        for world in (1, 2, 3, 8):
            seen = np.zeros(batch, dtype=np.int64)
            sizes = []
            for r in range(world):
                b0, b1 = shard_bounds(batch, r, world)
                assert 0 <= b0 <= b1 <= batch
                seen[b0:b1] += 1
                sizes.append(b1 - b0)
            assert np.all(seen == 1)
            assert max(sizes) - min(sizes) <= 1


def test_two_rank_gloo_sharding(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)]
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="1")
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=240, env=env)
    assert res.returncode == 0, res.stderr[-2000:]
    line = [ln for ln in res.stdout.splitlines() if ln.startswith("{")][-1]
    d = json.loads(line)
    (a0, a1, s0), (b0, b1, s1) = d["shards"]
    assert (a0, a1, b0, b1) == (0, 51, 51, 101)
    assert abs((s0 + s1) - d["total"]) <= 1e-9 * abs(d["total"])
    assert d["ms"] == [11.0, 5.0]
