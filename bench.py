#!/usr/bin/env python
"""bench.py -- headline measurement of the batched fitness-evaluation hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--ca-steps S] [--impl ours|reference]

Workload (N=1): BASELINE.json configs[1] -- 64 simulations on a 64^3 lattice, one pre-grown ~3k-cell
spheroid shared by the batch, a random 10-fraction protocol per simulation (synthetic, seeded).
One bench "step" = S CA steps (default 600 = one simulated hour) of the WHOLE hot path over the
whole batch (irradiate where scheduled, diffusion-reaction, cell state, division) followed by the
per-simulation reduction and fitness readout.  value = lattice site-updates/s = batch * sites * S / t.
For N>1 every rank runs its own 64 simulations (weak scaling, no data-path collective).
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2303_08123_b200 import workloads as w   # noqa: E402

B_ALG = 25.0            # algorithmic bytes per site-update (DESIGN.md section 8 / SURVEY 8(d))
HORIZON_STEPS = 432000  # configs[1], [2]: 30 days at 600 steps/h; configs[3]: 40 days


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic_bytes():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of k_diffuse_fused, from the committed ncu summary."""
    import glob
    import re
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_ncu_fused_*.txt")))
    if not files:
        return None
    txt = open(files[-1]).read()
    tot = 0.0
    for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        m = re.search(key + r"\s+([0-9.]+)\s+(\w+)", txt)
        if not m:
            return None
        tot += float(m.group(1)) * {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(m.group(2), 0.0)
    return tot


def full_horizon_record():
    """measured whole-job figure of `bench.py --full-horizon`, as committed under profiles/ (context for the extrapolated one)"""
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_full_horizon_c2.txt")))
    if not files:
        return None
    try:
        d = json.loads(open(files[-1]).read().strip().splitlines()[-1])
        return {"protocols_per_hour": d["value"], "us_per_ca_step": d["us_per_ca_step"], "source": os.path.basename(files[-1])}
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            c = [x.strip() for x in r.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for n, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(cfg, params, snapshot, steps, sim_id):
    """The oracle as it stands, one thread, advancing ONE simulation of the workload `steps` CA steps."""
    from oracle import ca_oracle as o
    nx, ny, nz = cfg["dims"]
    r = o.OracleSim(nx, ny, nz, params)
    if snapshot is None:
        r.seed(cfg["init"]["kind"], center=cfg["init"]["center"], radius=cfg["init"]["radius"],
               shared_init=cfg["init"]["shared_init"], rng_seed=cfg["rng_seed"], sim_id=sim_id)
    else:
        r.set_state(state=snapshot["state"], clock=snapshot["clock"], damage=snapshot["damage"],
                    o2=snapshot["o2"].astype(np.float64), glc=snapshot["glc"].astype(np.float64),
                    h=snapshot["h"].astype(np.float64), step=snapshot["step"])
        r.set_rng(cfg["rng_seed"], sim_id)
    t0 = time.perf_counter()
    r.step(steps)
    r.fitness()
    dt = time.perf_counter() - t0
    return nx * ny * nz * steps / dt, dt


def bench_config(args):
    """configs[1] (c2) is the headline.  --workload c3s / c4s are REDUCED-BATCH probes of the configs[2] / configs[3]
    lattices (96^3, 80^3: the tiled diffusion kernel), not headline numbers; config.workload says which one ran."""
    if args.workload == "c2":
        cfg = dict(w.config(2))
        if args.tumour_radius is not None:      # probe of the late phase of the job: the same workload started from a larger spheroid
            cfg["init"] = dict(cfg["init"], radius=float(args.tumour_radius))
            cfg["name"] += "-r%g" % args.tumour_radius
        return cfg
    k = 3 if args.workload == "c3s" else 4
    cfg = dict(w.config(k))
    batch = args.batch if args.batch else (64 if k == 3 else 96)
    cfg["batch"] = batch
    for key in ("dose", "delay", "nfrac"):
        cfg[key] = cfg[key][:batch]
    if k == 3:      # stand-in for the pre-grown 64-site spheroid (G19): a ball seeded directly, 3 h of warm-up
        cfg["init"] = dict(kind="ball", center=(48, 48, 48), radius=32.0, shared_init=True)
        cfg["warmup_h"], cfg["t0_h"] = 3.0, 3.0
    cfg["name"] += "-reduced"
    return cfg


def run_full_horizon(args):
    """--full-horizon: evaluate the whole workload to its horizon once (c2: 432 000 CA steps) and report the MEASURED
    protocols/hour, protocol upload and fitness download included, plus the counts the run ended with."""
    import torch
    from paper_2303_08123_b200 import binding
    cfg = bench_config(args)
    params = w.default_params()
    B = cfg["batch"]
    nx, ny, nz = cfg["dims"]
    torch.cuda.set_device(0)
    g = binding.CaBatch(B, nx, ny, nz, params, max_frac=10, device=0)
    if args.fused is not None:
        g.set_option("fused", args.fused)
    if args.cell_path is not None:
        g.set_option("cell_path", args.cell_path)
    g.seed(rng_seed=cfg["rng_seed"], sim_id_base=0, **cfg["init"])
    g.run(cfg["warmup_h"])
    g.sync()
    t_end = cfg["t0_h"] + cfg["horizon_h"]
    steps = int(round((t_end - cfg["warmup_h"]) * params["steps_per_hour"]))
    t0 = time.perf_counter()
    g.set_protocols(cfg["dose"], cfg["delay"], cfg["nfrac"], t0_h=cfg["t0_h"])
    g.run(t_end)
    fit = g.fitness()
    dt = time.perf_counter() - t0
    cnt = g.counts()
    line = {"metric": "protocols_per_hour_measured", "value": B * 3600.0 / dt, "unit": "protocols/h", "n_gpus": 1,
            "seconds": dt, "ca_steps": steps, "site_updates_per_s": B * nx * ny * nz * steps / dt, "us_per_ca_step": dt / steps * 1e6,
            "config": {"workload": cfg["name"], "batch": B, "dims": [nx, ny, nz], "horizon_h": cfg["horizon_h"]},
            "fitness_min_mean_max": [float(fit.min()), float(fit.mean()), float(fit.max())],
            "live_min_mean_max": [int(cnt[:, 0].min()), float(cnt[:, 0].mean()), int(cnt[:, 0].max())],
            "occupied_min_mean_max": [int(cnt[:, 12].min()), float(cnt[:, 12].mean()), int(cnt[:, 12].max())],
            "gpu_launches": g.launch_count, "data": "synthetic", "options": {"fused": args.fused, "cell_path": args.cell_path},
            "fitness": [float(x) for x in fit], "counts_live": [int(x) for x in cnt[:, 0]], "counts_dead": [int(x) for x in cnt[:, 3]]}
    print(json.dumps(line))
    g.close()


def run_ga_probe(args):
    """--ga: the configs[4] loop at reduced size -- a population of protocols x 4 seeds streamed through one batch context,
    host tournament selection + mutation between generations (paper_2303_08123_b200/ga.py).  Reduced horizon and
    population (stated in the line): a probe of the streaming driver, not the headline."""
    import torch
    from paper_2303_08123_b200 import binding, ga
    cfg = w.config(5)
    params = w.default_params()
    nx, ny, nz = cfg["dims"]
    torch.cuda.set_device(0)
    B = args.ga_batch
    g = binding.CaBatch(B, nx, ny, nz, params, max_frac=10, device=0)
    if args.chains is not None:
        g.set_option("chains", args.chains)
    if args.reserve_sms is not None:
        g.set_option("reserve_sms", args.reserve_sms)
    g.seed(rng_seed=cfg["rng_seed"], sim_id_base=0, **cfg["init"])
    g.run(cfg["warmup_h"])
    snap = g.get_state(0)
    npro, spp = args.ga_population, cfg["seeds_per_protocol"]
    dose, delay, nfrac = cfg["dose"][:npro], cfg["delay"][:npro], cfg["nfrac"][:npro]
    t_end = cfg["t0_h"] + args.ga_horizon_h
    t0 = time.perf_counter()
    hist, _, fit = ga.run_ga(g, snap, dose, delay, nfrac, args.ga_generations, spp, cfg["rng_seed"], cfg["t0_h"], t_end, ga_seed=cfg["rng_seed"])
    dt = time.perf_counter() - t0
    steps = int(round(args.ga_horizon_h * params["steps_per_hour"]))
    sims = npro * spp * args.ga_generations
    line = {"metric": "ga_protocol_evaluations_per_hour_reduced_horizon", "value": npro * args.ga_generations * 3600.0 / dt, "unit": "protocols/h",
            "seconds": dt, "site_updates_per_s": sims * nx * ny * nz * steps / dt,
            "config": {"workload": "BASELINE configs[4] REDUCED (probe): population %d x %d seeds, %d generations, horizon %.0f h of 720 h, batches of %d on %dx%dx%d"
                       % (npro, spp, args.ga_generations, args.ga_horizon_h, B, nx, ny, nz)},
            "best_mean_fitness_per_generation": hist, "data": "synthetic", "gpu_launches": g.launch_count}
    print(json.dumps(line))
    g.close()


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric / unit / config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = w.config(2)
    params = w.default_params()
    sample_steps = max(1, min(args.ca_steps, 150))
    vals = []
    for i in range(args.warmup + args.steps):
        v, dt = oracle_sample(cfg, params, None, sample_steps, 0)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals])) * 1e3
    sample = "1 of %d simulations x %d CA steps per step (64^3 lattice, from ca_seed BALL r=9)" % (cfg["batch"], sample_steps)
    line = {"impl": "reference", "metric": "site_updates_per_s", "value": value, "unit": "site-updates/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE configs[1]: 64 sims x 64^3, 10-fraction protocols (bounded sample)", "sample": sample},
            "cpu_baseline": {"value": value, "unit": "site-updates/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "site-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2303_08123_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit("--gpus %d but WORLD_SIZE=%d: launch N>1 with torch.distributed.run" % (args.gpus, world))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = bench_config(args)
    params = w.default_params()
    B = cfg["batch"]
    nx, ny, nz = cfg["dims"]
    sites = nx * ny * nz
    S = args.ca_steps
    # weak scaling: rank r evaluates protocols / global sim ids [r*B, (r+1)*B)
    rng = np.random.default_rng(cfg["rng_seed"] + 1000 * rank)
    dose, delay, nfrac = (cfg["dose"], cfg["delay"], cfg["nfrac"]) if rank == 0 else w.protocols_alphabet(rng, B)
    g = binding.CaBatch(B, nx, ny, nz, params, max_frac=10, device=local)
    if args.fused is not None:
        g.set_option("fused", args.fused)
    if args.graph_steps is not None:
        g.set_option("graph_steps", args.graph_steps)
    if args.cluster is not None:
        g.set_option("cluster", args.cluster)
    if args.chains is not None:
        g.set_option("chains", args.chains)
    if args.reserve_sms is not None:
        g.set_option("reserve_sms", args.reserve_sms)
    stream = g.stream

    # ---- untimed setup: shared pre-grown spheroid + quasi-steady fields (c2 recipe)
    g.seed(rng_seed=cfg["rng_seed"], sim_id_base=rank * B, **cfg["init"])
    g.run(cfg["warmup_h"])
    g.set_protocols(dose, delay, nfrac, t0_h=cfg["t0_h"])
    snapshot = g.get_state(0)                              # host copy: e2e upload source and oracle sample input
    t_now = cfg["warmup_h"]
    dt_h = S / params["steps_per_hour"]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    fit_dev = torch.zeros(B, dtype=torch.float32, device="cuda")

    def one_step():
        nonlocal t_now
        t_now += dt_h
        g.run(t_now)
        g.fitness(out=fit_dev)

    for _ in range(args.warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = g.launch_count
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(args.steps):
            one_step()
        ev1.record(stream)
    barrier()
    g.sync()
    launches = g.launch_count - launches0
    clocks = sampler.stop() if rank == 0 else None
    ms = ev0.elapsed_time(ev1)
    t = torch.tensor([ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    ms_per_step = ms_total / args.steps
    value = world * B * sites * S / (ms_per_step * 1e-3)

    # ---- dominant kernel alone: the diffusion-reaction stage, CUDA events on its stream
    reps = 30
    with torch.cuda.stream(stream):
        for _ in range(3):
            g.stage(1)
        l0 = g.launch_count
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0.record(stream)
        for _ in range(reps):
            g.stage(1)
        k1.record(stream)
    torch.cuda.synchronize()
    per_stage_launches = (g.launch_count - l0) / reps
    stage_ms = k0.elapsed_time(k1) / reps
    launch_ms = stage_ms / per_stage_launches
    peak, peak_src = measured_peaks()
    # algorithmic bytes per launch = 25 B x sites x (CA steps one launch completes)
    achieved = B_ALG * B * sites * (1.0 / per_stage_launches) / (launch_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": ("k_diffuse_fused" if args.workload == "c2" else "k_diffuse_tiled") + ": diffusion-reaction stage S1, all n_sub sub-steps (%d launch(es) per CA step)" % round(per_stage_launches),
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "launch_ms": launch_ms, "traffic": ncu_traffic_bytes() if (args.workload == "c2" and args.tumour_radius is None) else None, "traffic_unit": "bytes/launch (ncu --set full, profiles/)",
                "algorithmic_bytes_per_launch": B_ALG * B * sites / per_stage_launches, "stage_share_of_step": stage_ms * S / ms_per_step}

    # ---- end to end through the C ABI with HOST buffers: snapshot + protocols up, fitness down, every step
    fit_host = None
    e2e_steps = max(1, min(args.steps, 3))
    h2d = sum(snapshot[k].nbytes for k in ("state", "clock", "damage", "o2", "glc", "h")) + dose.astype(np.float32).nbytes * 2 + nfrac.nbytes
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        g.set_state(0, B, state=snapshot["state"], clock=snapshot["clock"], damage=snapshot["damage"],
                    o2=snapshot["o2"], glc=snapshot["glc"], h=snapshot["h"], step=snapshot["step"])
        g.set_protocols(dose, delay, nfrac, t0_h=cfg["t0_h"])
        g.run(cfg["warmup_h"] + dt_h)
        fit_host = g.fitness()
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    te = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e = {"value": world * B * sites * S / float(te.item()), "unit": "site-updates/s",
           "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(fit_host.nbytes), "ms_per_step": float(te.item()) * 1e3}

    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            osteps = args.oracle_steps
            v, dt = oracle_sample(cfg, params, snapshot, osteps, 0)
            cpu = {"value": v, "unit": "site-updates/s", "cores": 1, "kind": "oracle", "seconds": dt,
                   "sample": "1 of %d simulations x %d CA steps from the GPU's post-warm-up snapshot (64^3)" % (B, osteps)}
        line = {"metric": "site_updates_per_s", "value": value, "unit": "site-updates/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "BASELINE configs[%d]%s: %d sims/GPU x %dx%dx%d lattice, shared spheroid, random protocols" % ({"c2": 1, "c3s": 2, "c4s": 3}[args.workload], ("" if args.workload == "c2" else (" FULL BATCH (probe: first steps only, stand-in spheroid)" if B >= (512 if args.workload == "c3s" else 1024) else " REDUCED BATCH (probe, not the headline)")) + ("" if args.tumour_radius is None else " STARTED FROM A BALL OF RADIUS %g (late-phase probe, not the headline)" % args.tumour_radius), B, nx, ny, nz),
                           "ca_steps_per_step": S, "n_sub": params["n_sub"], "l2": "working set %.2f GB/GPU > 126 MB L2 (no flush needed)" % (29.0 * B * sites / 1e9),
                           "sharding": "batch over ranks, no collective"},
                "protocols_per_hour": world * B * 3600.0 / (ms_per_step * 1e-3 / S * (576000 if args.workload == "c4s" else HORIZON_STEPS)),
                "protocols_per_hour_note": "extrapolated from the timed CA steps at the start of treatment (~3k-cell tumours); the tumours regrow to ~1.6e5 cells by day 30 and the late steps cost more: see full_horizon_measured",
                "full_horizon_measured": full_horizon_record() if (args.workload == "c2" and args.tumour_radius is None) else None,
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
                "fitness_sample": [float(x) for x in fit_host[:4]]}
        print(json.dumps(line))
    g.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--ca-steps", type=int, default=600, help="CA steps per bench step (600 = one simulated hour)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=["c2", "c3s", "c4s"], help="c2 = headline; c3s / c4s = reduced-batch probes of the 96^3 / 80^3 lattices")
    ap.add_argument("--fused", type=int, default=None)
    ap.add_argument("--graph-steps", type=int, default=None)
    ap.add_argument("--cell-path", type=int, default=None, help="0: generic S2/S3 scan kernels")
    ap.add_argument("--chains", type=int, default=None)
    ap.add_argument("--reserve-sms", type=int, default=None)
    ap.add_argument("--cluster", type=int, default=None, help="CTAs per simulation of the S2+S3 kernel (1, 2, 4, 8)")
    ap.add_argument("--oracle-steps", type=int, default=1500, help="CA steps of the oracle sample (about 15 s on one core)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--batch", type=int, default=0, help="c3s / c4s only: batch size of the probe (default 64 / 96; 512 / 1024 = the full configs)")
    ap.add_argument("--tumour-radius", type=float, default=None, help="c2 only: start from a BALL of this radius instead of 9 (probe of the late, dense phase)")
    ap.add_argument("--ga", action="store_true", help="configs[4] streaming + host GA loop at reduced size (probe)")
    ap.add_argument("--ga-population", type=int, default=128)
    ap.add_argument("--ga-generations", type=int, default=2)
    ap.add_argument("--ga-horizon-h", type=float, default=12.0)
    ap.add_argument("--ga-batch", type=int, default=128)
    ap.add_argument("--full-horizon", action="store_true", help="run the whole workload to its horizon once; measured protocols/h")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.ga:
        run_ga_probe(args)
    elif args.full_horizon:
        run_full_horizon(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
