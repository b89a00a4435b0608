#!/usr/bin/env python
"""Writes tests/golden/reduced_c2_ensemble.txt: the fp64 ORACLE's final counts for a reduced BASELINE configs[1] job.

    python tests/golden/make_reduced_c2_ensemble.py [--workers N]

This script calls only oracle/ (and the data-only input generators of workloads.py); no value in the output comes from
the CUDA path.  It is the reference side of SURVEY 8(c) comparison protocol (3) / north_star's third tolerance: "final
per-protocol tumour counts within 1 % (or within the oracle's own seed-to-seed 95 % interval on long horizons)", which is
the paper's own way of validating a GPU port against CPU code (Fig. 3 l.357).

Scenario (`workloads.reduced_c2()`): 32^3 lattice, one shared pre-grown spheroid (BALL r = 4, 6 h untreated warm-up),
8 random protocols of 4 fractions from the configs[1] dose alphabet with delays from {6, 12, 18, 24} h, 30 seeds each
(global simulation id = 30 * protocol + seed), horizon = 5 simulated days after the start of treatment (75 600 CA steps
in all).  About 95 s per simulation on one core; 240 simulations.
"""
import argparse
import os
import sys
import time
from concurrent.futures import ProcessPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import ca_oracle as o                      # noqa: E402
from paper_2303_08123_b200 import workloads as w       # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "reduced_c2_ensemble.txt")


def one(job):
    pro, seed_idx = job
    cfg = w.reduced_c2()
    p = w.default_params()
    nx, ny, nz = cfg["dims"]
    sim = o.OracleSim(nx, ny, nz, p)
    sid = cfg["seeds_per_protocol"] * pro + seed_idx
    # the warm-up is part of every simulation: shared initial draws (sim id 0), own id for the dynamics [D G17]
    sim.seed(cfg["init"]["kind"], center=cfg["init"]["center"], radius=cfg["init"]["radius"], shared_init=True,
             rng_seed=cfg["rng_seed"], sim_id=sid)
    sim.set_protocol(cfg["dose"][pro], cfg["delay"][pro], t0_h=cfg["t0_h"])
    sim.run(cfg["t0_h"] + cfg["horizon_h"])
    c = sim.counts()
    return pro, seed_idx, int(c[0]), int(c[1]), int(c[3]), int(c[12])


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workers", type=int, default=max(1, (os.cpu_count() or 2) - 1))
    args = ap.parse_args()
    o.build()
    cfg = w.reduced_c2()
    jobs = [(pr, s) for pr in range(cfg["population"]) for s in range(cfg["seeds_per_protocol"])]
    t0 = time.time()
    with ProcessPoolExecutor(args.workers) as ex:
        rows = list(ex.map(one, jobs, chunksize=1))
    rows.sort()
    with open(OUT, "w") as f:
        f.write("# fp64 oracle (oracle/ca_oracle.c), reduced BASELINE configs[1] job: written by tests/golden/make_reduced_c2_ensemble.py\n")
        f.write("# which calls only oracle/.  Lattice %dx%dx%d, %d protocols x %d seeds, t0 = %g h, horizon %g h, rng_seed %d.\n"
                % (*cfg["dims"], cfg["population"], cfg["seeds_per_protocol"], cfg["t0_h"], cfg["horizon_h"], cfg["rng_seed"]))
        f.write("# Reference side of north_star's long-horizon tolerance and of PAPER.md l.69 / Fig. 3 (l.357).\n")
        for pr in range(cfg["population"]):
            f.write("# protocol %d: dose %s Gy, delay %s h\n" % (pr, cfg["dose"][pr].tolist(), cfg["delay"][pr].tolist()))
        f.write("# columns: protocol seed live doomed dead occupied\n")
        for r in rows:
            f.write("%d %d %d %d %d %d\n" % r)
    print("wrote", OUT, "in %.0f s" % (time.time() - t0))


if __name__ == "__main__":
    main()
