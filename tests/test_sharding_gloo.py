"""N>1 host path on CPU: world size 2, gloo.  No GPU, no oracle."""
import os
import socket
import subprocess
import sys

import numpy as np

from paper_2303_08123_b200 import sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
import numpy as np
import torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2303_08123_b200 import sharding, workloads as w
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
total = 7
rng = np.random.default_rng(5)
table = w.protocols_alphabet(rng, total) if rank == 0 else (None, None, None)
dose, delay, nfrac = sharding.broadcast_protocols(*table, dist=dist)
d, t, nf, first = sharding.shard_protocols(dose, delay, nfrac, world, rank)
# stand-in "fitness": a function of the GLOBAL id and the protocol only, so the gathered vector must not depend on the split
local = np.array([1000.0 * (first + i) + d[i].sum() for i in range(len(nf))], np.float32)
full = sharding.gather_fitness(local, total, dist)
expect = np.array([1000.0 * g + dose[g].sum() for g in range(total)], np.float32)
assert np.array_equal(full, expect), (rank, full, expect)
print("rank", rank, "ok", first, len(nf))
dist.destroy_process_group()
"""


def test_shard_range_is_a_partition():
    for total in (1, 7, 64, 16384):
        for world in (1, 2, 3, 8):
            parts = [sharding.shard_range(total, world, r) for r in range(world)]
            assert parts[0][0] == 0 and sum(c for _, c in parts) == total
            for (f0, c0), (f1, _) in zip(parts, parts[1:]):
                assert f1 == f0 + c0
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1


def test_world_size_2_gloo_gather_is_split_independent(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(script), ROOT]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rank 0 ok 0 4" in r.stdout and "rank 1 ok 4 3" in r.stdout
