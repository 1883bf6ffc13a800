"""N > 1 host logic on CPU: contiguous balanced column shards, and a world_size-2 gloo run in which
every rank builds its shard of the same seeded batch and the max-over-ranks timing reduction works."""
import os
import socket
import subprocess
import sys

import numpy as np

from paper_1606_05474_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, numpy as np, torch, torch.distributed as dist
sys.path.insert(0, os.environ["REPO"])
from paper_1606_05474_b200 import inputs
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
inp, nc = bench.workload(3, 5, world, rank)
assert nc == 5 and inp.params["n_cols"] == 5 and inp.T0.shape == (5, 100)
full = inputs.make_config(3, n_cols=10)
sl = list(inputs.shard_columns(10, rank, world))
assert np.array_equal(inp.T0, full.T0[sl]) and np.array_equal(inp.kscale, full.kscale[sl])
# gather the shards' first temperatures: together they are the full batch, in order, no overlap
t = torch.from_numpy(np.ascontiguousarray(inp.T0[:, 0]))
out = [torch.empty_like(t) for _ in range(world)]
dist.all_gather(out, t)
assert np.array_equal(torch.cat(out).numpy(), full.T0[:, 0])
ms = torch.tensor([10.0 + rank], dtype=torch.float64)
dist.all_reduce(ms, op=dist.ReduceOp.MAX)
assert ms.item() == 10.0 + world - 1
dist.destroy_process_group()
print("ok", rank)
'''


def test_shard_columns_partition():
    for n, w in ((8192, 8), (10, 3), (5, 8), (1, 2)):
        parts = [list(inputs.shard_columns(n, r, w)) for r in range(w)]
        assert sum(parts, []) == list(range(n))
        assert max(map(len, parts)) - min(map(len, parts)) <= 1


def test_take_columns_keeps_shared_arrays():
    full = inputs.make_config(3, n_cols=6)
    part = full.take_columns([4, 1])
    assert part.params["n_cols"] == 2 and part.ktab is full.ktab
    assert np.array_equal(part.T0, full.T0[[4, 1]]) and np.array_equal(part.f_star_scale, full.f_star_scale[[4, 1]])


def test_world_size_2_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), REPO=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for p in procs:
        out, _ = p.communicate(timeout=240)
        assert p.returncode == 0 and "ok" in out, out
