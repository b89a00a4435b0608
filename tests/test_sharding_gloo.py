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
sys.stdout.write("rank %d ok %d %d\n" % (rank, first, len(nf))); sys.stdout.flush()
dist.destroy_process_group()
"""


WORKER_GA = r"""
import os, sys
import numpy as np
import torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2303_08123_b200 import ga, workloads as w


class StubBatch:
    # stands in for binding.CaBatch on the CPU: "fitness" of a simulation = a function of its GLOBAL id and its protocol
    def __init__(self, batch):
        self.batch = batch
    def set_state(self, *a, **k):
        pass
    def set_rng(self, rng_seed, sim_id_base):
        self.base = sim_id_base
    def set_protocols(self, dose, delay, nfrac, t0_h=0.0):
        self.dose, self.delay = np.asarray(dose), np.asarray(delay)
    def run(self, t_end):
        self.t_end = t_end
    def fitness(self):
        ids = self.base + np.arange(self.batch)
        return (1000.0 - self.dose.sum(1) - 0.01 * self.delay.sum(1) + 0.001 * (ids % 7)).astype(np.float32)


dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
rng = np.random.default_rng(11)
dose, delay, nfrac = w.protocols_alphabet(rng, 13)
snap = dict(state=None, clock=None, damage=None, o2=None, glc=None, h=None, step=0)
spp = 3
mean, per_sim = ga.evaluate_population(StubBatch(5), snap, dose, delay, nfrac, spp, 1, 0.0, 1.0, dist=dist)
ids = np.arange(13 * spp)
expect = (1000.0 - dose[ids // spp].sum(1) - 0.01 * delay[ids // spp].sum(1) + 0.001 * (ids % 7)).astype(np.float32)
assert np.array_equal(per_sim, expect), (rank, per_sim[:6], expect[:6])
assert np.allclose(mean, expect.reshape(13, spp).mean(1))
# three generations of the loop: every rank ends with the same population (rank 0's, broadcast)
hist, pop, fit = ga.run_ga(StubBatch(5), snap, dose, delay, nfrac, 3, spp, 1, 0.0, 1.0, ga_seed=5 + rank, dist=dist)
import hashlib
digest = hashlib.sha1(np.ascontiguousarray(pop[0]).tobytes() + np.ascontiguousarray(pop[1]).tobytes()).hexdigest()
all_d = [None] * world
dist.all_gather_object(all_d, digest)
assert len(set(all_d)) == 1, all_d
assert hist[-1][0] >= hist[0][0] - 1e-6
sys.stdout.write("rank %d ga ok\\n" % rank); sys.stdout.flush()
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


def test_world_size_2_gloo_population_evaluation_is_sharded_and_split_independent(tmp_path):
    """ga.evaluate_population(dist=...) -- the product's N > 1 entry point -- with a stub context: every rank gets the same
    per-simulation fitness vector as a single process would, and the GA loop keeps the ranks' populations identical."""
    script = tmp_path / "worker_ga.py"
    script.write_text(WORKER_GA)
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(script), ROOT]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rank 0 ga ok" in r.stdout and "rank 1 ga ok" in r.stdout
