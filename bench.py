#!/usr/bin/env python
"""bench.py -- measurement of the batched fitness-evaluation hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Headline workload (N = 1): BASELINE.json configs[4] -- the GA population of 4096 protocols x 4 seeds = 16 384 simulations
on a 64^3 lattice -- at the largest batch that is resident in HBM at once (16 384 simulations = 125 GB on a 180 GB B200;
config.workload names the batch that ran).  Every simulation starts from one saved, pre-grown ~3k-cell spheroid
 and has its own 10-fraction protocol; synthetic, seeded.  One bench "step" = S CA steps (default 20) of
the WHOLE hot path over the whole batch (irradiate where scheduled, diffusion-reaction, cell state, division) followed by
the per-simulation reduction and fitness readout.  value = lattice site-updates/s = batch * sites * S / t.

In the same run (N = 1) the line also carries
  per_config            configs[1] (64 x 64^3), configs[2] (512 x 96^3 from the pre-grown 64-site spheroid) and configs[3]
                        (1024 x 80^3), each measured live: whole CA step, its diffusion kernel alone, roofline fraction;
  protocols_per_hour    MEASURED: the whole configs[1] job (432 000 CA steps) evaluated once, upload and readout included;
  e2e                   the headline workload over the SAME simulated window through the C ABI with host buffers;
  cpu_baseline          the oracle on one core and on all host cores (core count and CPU model stated).
For N > 1 every rank runs its own batch (weak scaling, no data-path collective); `--ga` runs the sharded population
evaluation of paper_2303_08123_b200/ga.py instead (a fixed population split over the ranks).
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2303_08123_b200 import workloads as w   # noqa: E402

B_ALG = 25.0            # algorithmic bytes per site-update (DESIGN.md section 8 / SURVEY 8(d))


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(pattern):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the newest committed ncu summary matching `pattern`.
    This is a number from an EARLIER ncu capture, not measured in this run: the caller labels it with its source."""
    import glob
    import re
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", pattern)))
    if not files:
        return None, None, None
    txt = open(files[-1]).read()
    tot = 0.0
    for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        m = re.search(key + r"\s+([0-9.]+)\s+(\w+)", txt)
        if not m:
            return None, None, None
        tot += float(m.group(1)) * {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(m.group(2), 0.0)
    m = re.search(r"--batch (\d+)", txt)
    return tot, "profiles/" + os.path.basename(files[-1]), (int(m.group(1)) if m else None)


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


# ------------------------------------------------------------------------------------------ oracle legs --
def oracle_sample(dims, params, snapshot, steps, rng_seed, sim_id, init=None):
    """The oracle as it stands, one thread, advancing ONE simulation `steps` CA steps; returns (site-updates/s, seconds)."""
    from oracle import ca_oracle as o
    nx, ny, nz = dims
    r = o.OracleSim(nx, ny, nz, params)
    if snapshot is None:
        r.seed(init["kind"], center=init["center"], radius=init["radius"], shared_init=init["shared_init"], rng_seed=rng_seed, sim_id=sim_id)
    else:
        r.set_state(state=snapshot["state"], clock=snapshot["clock"], damage=snapshot["damage"],
                    o2=snapshot["o2"].astype(np.float64), glc=snapshot["glc"].astype(np.float64),
                    h=snapshot["h"].astype(np.float64), step=snapshot["step"])
        r.set_rng(rng_seed, sim_id)
    t0 = time.perf_counter()
    r.step(steps)
    r.fitness()
    dt = time.perf_counter() - t0
    return nx * ny * nz * steps / dt, dt


_WORKER = r"""
import sys, json, time
import numpy as np
sys.path.insert(0, sys.argv[1])
import bench
from paper_2303_08123_b200 import workloads as w
d = np.load(sys.argv[2])
snap = {k: d[k] for k in ("state", "clock", "damage", "o2", "glc", "h")}
snap["step"] = int(d["step"])
dims = tuple(int(x) for x in d["dims"])
v, dt = bench.oracle_sample(dims, w.default_params(), snap, int(sys.argv[3]), int(d["rng_seed"]), int(sys.argv[4]))
print(json.dumps({"v": v, "dt": dt}))
"""


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_all_cores(dims, snapshot, steps, rng_seed):
    """`nproc` independent oracle processes, one simulation each, started together: whole-host site-updates/s."""
    n = min(os.cpu_count() or 1, 256)
    with tempfile.TemporaryDirectory() as td:
        path = os.path.join(td, "snap.npz")
        np.savez(path, dims=np.array(dims), rng_seed=np.array(rng_seed), step=np.array(snapshot["step"]),
                 **{k: snapshot[k] for k in ("state", "clock", "damage", "o2", "glc", "h")})
        script = os.path.join(td, "worker.py")
        open(script, "w").write(_WORKER)
        t0 = time.perf_counter()
        procs = [subprocess.Popen([sys.executable, script, ROOT, path, str(steps), str(i)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
                 for i in range(n)]
        outs = [p.communicate()[0] for p in procs]
        wall = time.perf_counter() - t0
    ok = [json.loads(o.strip().splitlines()[-1]) for o in outs if o.strip()]
    if not ok:
        return None
    sites = dims[0] * dims[1] * dims[2]
    # every process advanced `steps` steps; the slowest one bounds the throughput of the host as a whole
    return {"value": len(ok) * sites * steps / max(x["dt"] for x in ok), "processes": len(ok), "seconds": wall}


# ------------------------------------------------------------------------------------------ GPU helpers --
def make_batch(binding, torch, batch, dims, params, max_frac, device):
    """CaBatch of `batch` simulations, halving the batch while the workspace does not fit (returns ctx, batch)."""
    while True:
        try:
            return binding.CaBatch(batch, dims[0], dims[1], dims[2], params, max_frac=max_frac, device=device), batch
        except (RuntimeError, binding.CaError) as e:
            if "out of memory" not in str(e).lower() or batch <= 64:
                raise
            torch.cuda.empty_cache()
            batch //= 2


def warm_snapshot(binding, cfg, params, device):
    """The saved tumour every simulation starts from: ONE simulation seeded and warmed up, exported."""
    nx, ny, nz = cfg["dims"]
    g = binding.CaBatch(1, nx, ny, nz, params, max_frac=1, device=device)
    g.seed(rng_seed=cfg["rng_seed"], sim_id_base=0, **cfg["init"])
    g.run(cfg["warmup_h"])
    snap = g.get_state(0)
    g.close()
    return snap


def load_snapshot(g, snap):
    g.set_state(0, g.batch, state=snap["state"], clock=snap["clock"], damage=snap["damage"], o2=snap["o2"], glc=snap["glc"], h=snap["h"], step=snap["step"])


def remaining_table(dose, delay, nfrac, t0_h, t_now):
    """The protocol table as it stands at time t_now: fractions already delivered become (0 Gy, 0 h) no-ops so that the
    later ones keep their list index (the irradiation draws are keyed by it) and their absolute time."""
    dose, delay = np.array(dose, np.float64), np.array(delay, np.float64)
    T = t0_h + np.cumsum(delay, axis=1)
    nd, nt = np.zeros_like(dose), np.zeros_like(delay)
    for b in range(len(nfrac)):
        t_prev = t_now
        for j in range(int(nfrac[b])):
            if T[b, j] < t_now - 1e-9:
                continue                                   # delivered: (0, 0) at t_now
            nd[b, j] = dose[b, j]
            nt[b, j] = T[b, j] - t_prev
            t_prev = T[b, j]
    return nd, nt


def time_stage(torch, g, stream, reps):
    """average duration of one diffusion-reaction stage S1 (CUDA events on the context's stream), launches per stage"""
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
    return k0.elapsed_time(k1) / reps, (g.launch_count - l0) / reps


def roofline_block(kernel, B, sites, stage_ms, per_stage_launches, step_ms_per_ca_step, traffic_pattern):
    peak, peak_src = measured_peaks()
    launch_ms = stage_ms / per_stage_launches
    alg = B_ALG * B * sites / per_stage_launches          # 25 B x sites x (CA steps one launch completes)
    achieved = alg / (launch_ms * 1e-3) / 1e9
    traffic, src, tb = ncu_traffic(traffic_pattern) if traffic_pattern else (None, None, None)
    return {"bound": "hbm", "kernel": kernel + ": diffusion-reaction stage S1, all n_sub sub-steps (%d launch(es) per CA step)" % round(per_stage_launches),
            "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
            "launch_ms": launch_ms, "algorithmic_bytes_per_launch": alg,
            "traffic": traffic, "traffic_batch": tb,
            "traffic_over_algorithmic": (traffic / (B_ALG * tb * sites)) if (traffic and tb) else None,
            "traffic_source": (src + " (an earlier ncu --set full capture, at the batch that file names; not measured in this run)") if src else None,
            "stage_share_of_step": stage_ms / step_ms_per_ca_step if step_ms_per_ca_step else None,
            "whole_step_frac": (B_ALG * B * sites / (step_ms_per_ca_step * 1e-3) / 1e9) / peak if step_ms_per_ca_step else None}


def timed_window(torch, g, stream, t_start, dt_h, warmup, steps, fit_dev):
    """`warmup` untimed + `steps` timed bench steps of dt_h simulated hours each; returns (ms total, t_end)"""
    t = t_start
    for _ in range(warmup):
        t += dt_h
        g.run(t)
        g.fitness(out=fit_dev)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(steps):
            t += dt_h
            g.run(t)
            g.fitness(out=fit_dev)
        e1.record(stream)
    torch.cuda.synchronize()
    g.sync()
    return e0.elapsed_time(e1), t


def config_probe(torch, binding, name, cfg, params, snap, device, ca_steps, kernel, traffic_pattern, options=None):
    """one per_config entry: the whole CA step and its diffusion kernel on this configuration, measured now"""
    B = cfg["batch"]
    nx, ny, nz = cfg["dims"]
    sites = nx * ny * nz
    g = binding.CaBatch(B, nx, ny, nz, params, max_frac=cfg["dose"].shape[1], device=device)
    for k, v in (options or {}).items():
        g.set_option(k, v)
    load_snapshot(g, snap)
    g.set_rng(cfg["rng_seed"], 0)
    g.set_protocols(cfg["dose"], cfg["delay"], cfg["nfrac"], t0_h=cfg["t0_h"])
    fit_dev = torch.zeros(B, dtype=torch.float32, device="cuda")
    dt_h = ca_steps / params["steps_per_hour"]
    ms, _ = timed_window(torch, g, g.stream, cfg["t0_h"], dt_h, 3, 3, fit_dev)
    step_ms = ms / 3 / ca_steps
    stage_ms, nl = time_stage(torch, g, g.stream, 10)
    cnt = g.counts()
    kern = {0: "k_diffuse_sub", 1: "k_diffuse_fused", 2: "k_diffuse_slab", 3: "k_diffuse_rows"}[g.get_option("diffusion_kernel")]
    if g.get_option("rows_cluster"):
        kern += " (clusters of %d CTAs, %d resident)" % (g.get_option("rows_cluster"), g.get_option("rows_nclusters"))
    kernel = kern
    out = {"workload": "BASELINE configs[%s]: %d sims x %dx%dx%d" % (name, B, nx, ny, nz), "batch": B, "dims": [nx, ny, nz],
           "resident_gb": 29.0 * B * sites / 1e9, "ca_steps_timed": 3 * ca_steps, "us_per_ca_step": step_ms * 1e3,
           "site_updates_per_s": B * sites / (step_ms * 1e-3), "live_cells_per_sim_mean": float(cnt[:, 0].mean()),
           "dead_cells_per_sim_mean": float(cnt[:, 3].mean()),
           "roofline": roofline_block(kernel, B, sites, stage_ms, nl, step_ms, traffic_pattern)}
    g.close()
    del g
    torch.cuda.empty_cache()
    return out


def full_horizon(torch, binding, cfg, params, snap, device, label="configs[1]"):
    """evaluate the whole workload to its horizon once: MEASURED protocols/hour, upload and readout included"""
    B = cfg["batch"]
    nx, ny, nz = cfg["dims"]
    g = binding.CaBatch(B, nx, ny, nz, params, max_frac=cfg["dose"].shape[1], device=device)
    t_end = cfg["t0_h"] + cfg["horizon_h"]
    steps = int(round(cfg["horizon_h"] * params["steps_per_hour"]))
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    load_snapshot(g, snap)
    g.set_rng(cfg["rng_seed"], 0)
    g.set_protocols(cfg["dose"], cfg["delay"], cfg["nfrac"], t0_h=cfg["t0_h"])
    g.run(t_end)
    fit = g.fitness()
    dt = time.perf_counter() - t0
    cnt = g.counts()
    out = {"workload": "BASELINE %s whole job: %d protocols x %dx%dx%d to %g h" % (label, B, nx, ny, nz, cfg["horizon_h"]),
           "protocols_per_hour": B * 3600.0 / dt, "seconds": dt, "ca_steps": steps, "us_per_ca_step": dt / steps * 1e6,
           "site_updates_per_s": B * nx * ny * nz * steps / dt, "whole_job_frac_of_hbm_roofline": B_ALG * B * nx * ny * nz * steps / dt / 1e9 / measured_peaks()[0],
           "fitness_min_mean_max": [float(fit.min()), float(fit.mean()), float(fit.max())],
           "live_min_mean_max": [int(cnt[:, 0].min()), float(cnt[:, 0].mean()), int(cnt[:, 0].max())],
           "dead_min_mean_max": [int(cnt[:, 3].min()), float(cnt[:, 3].mean()), int(cnt[:, 3].max())], "gpu_launches": g.launch_count}
    g.close()
    torch.cuda.empty_cache()
    return out


# ------------------------------------------------------------------------------------------ arms --
def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric / unit / config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = w.config(5)
    params = w.default_params()
    sample_steps = max(1, min(args.ca_steps or 20, 150)) * 5
    vals = []
    for i in range(args.warmup + args.steps):
        v, dt = oracle_sample(cfg["dims"], params, None, sample_steps, cfg["rng_seed"], 0, init=cfg["init"])
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals])) * 1e3
    sample = "1 of %d simulations x %d CA steps per step (64^3 lattice, from ca_seed BALL r=9), one core of %d (%s)" % (cfg["batch"], sample_steps, os.cpu_count() or 1, cpu_model())
    line = {"impl": "reference", "metric": "site_updates_per_s", "value": value, "unit": "site-updates/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE configs[4]: 16384 sims x 64^3, 10-fraction protocols (bounded sample: one simulation)", "sample": sample},
            "cpu_baseline": {"value": value, "unit": "site-updates/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "site-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_ga(args):
    """--ga: configs[4] as the search loop runs it -- a population of protocols x 4 seeds evaluated through
    ga.evaluate_population (sharded over the ranks when N > 1: a FIXED population, i.e. strong scaling), host selection
    + mutation between generations.  Reduced population / horizon (stated in the line)."""
    import torch
    import torch.distributed as dist
    from paper_2303_08123_b200 import binding, ga
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = w.config(5)
    params = w.default_params()
    nx, ny, nz = cfg["dims"]
    snap = warm_snapshot(binding, cfg, params, local)
    g = binding.CaBatch(args.ga_batch, nx, ny, nz, params, max_frac=10, device=local)
    npro, spp = args.ga_population, cfg["seeds_per_protocol"]
    dose, delay, nfrac = cfg["dose"][:npro], cfg["delay"][:npro], cfg["nfrac"][:npro]
    t_end = cfg["t0_h"] + args.ga_horizon_h
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    hist, _, fit = ga.run_ga(g, snap, dose, delay, nfrac, args.ga_generations, spp, cfg["rng_seed"], cfg["t0_h"], t_end,
                             ga_seed=cfg["rng_seed"], dist=dist if world > 1 else None)
    torch.cuda.synchronize()
    dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(dt, op=dist.ReduceOp.MAX)
    dt = float(dt.item())
    steps = int(round(args.ga_horizon_h * params["steps_per_hour"]))
    sims = npro * spp * args.ga_generations
    if rank == 0:
        line = {"metric": "ga_protocol_evaluations_per_hour_reduced_horizon", "value": npro * args.ga_generations * 3600.0 / dt, "unit": "protocols/h",
                "n_gpus": world, "scaling": "strong", "seconds": dt, "site_updates_per_s": sims * nx * ny * nz * steps / dt,
                "config": {"workload": "BASELINE configs[4] REDUCED: population %d x %d seeds, %d generations, horizon %.0f h of 720 h, batches of %d per rank on %dx%dx%d"
                           % (npro, spp, args.ga_generations, args.ga_horizon_h, args.ga_batch, nx, ny, nz), "sharding": "global simulation ids split contiguously over ranks; one all_gather of fitness per generation"},
                "best_mean_fitness_per_generation": hist, "data": "synthetic", "gpu_launches": g.launch_count}
        print(json.dumps(line))
    g.close()
    if world > 1:
        dist.destroy_process_group()


def run_probe(args):
    """--probe c2|c3|c4 [--batch N] [--tumour-radius R]: ONE per_config entry alone (reduced batch allowed; what the ncu
    captures under profiles/ were taken from).  Not the headline."""
    import torch
    from paper_2303_08123_b200 import binding, pregrow
    torch.cuda.set_device(0)
    params = w.default_params()
    k = {"c2": 2, "c3": 3, "c4": 4}[args.probe]
    cfg = dict(w.config(k))
    if args.batch:
        cfg["batch"] = args.batch
        reps = -(-args.batch // len(cfg["nfrac"]))
        for key in ("dose", "delay", "nfrac"):
            cfg[key] = np.concatenate([cfg[key]] * reps)[:args.batch]
    if k == 3 and args.tumour_radius is None:
        snap, grown_h = pregrow.grow(cfg["dims"], params, cfg["init"], cfg["rng_seed"], target_extent=cfg["pregrow_diameter"], check_h=24.0)
        cfg["t0_h"] = grown_h
    else:
        if k == 3:
            cfg["warmup_h"], cfg["t0_h"] = 3.0, 3.0
        if args.tumour_radius is not None:          # late-phase probe: the same lattice started from a larger seeded ball
            cfg["init"] = dict(cfg["init"], kind="ball", radius=float(args.tumour_radius))
        snap = warm_snapshot(binding, cfg, params, 0)
    kern = "k_diffuse_fused" if k == 2 else "k_diffuse_rows"
    opts = {} if args.rows_cluster is None else {"rows_cluster": args.rows_cluster}
    if args.rows_rp is not None:
        opts["rows_rp"] = args.rows_rp
    out = config_probe(torch, binding, str(k - 1), cfg, params, snap, 0, args.ca_steps or (200 if k == 2 else 20), kern, None, options=opts)
    out["probe"] = {"config": args.probe, "batch": cfg["batch"], "tumour_radius": args.tumour_radius}
    print(json.dumps(out))


def run_whole_job(args):
    """--whole-job c2|c3|c4: evaluate that configuration's WHOLE job once (all its protocols to the horizon) and print the
    measured protocols/hour.  configs[2] / [3] take about an hour of GPU time each; not part of the default run."""
    import torch
    from paper_2303_08123_b200 import binding, pregrow
    torch.cuda.set_device(0)
    params = w.default_params()
    k = {"c2": 2, "c3": 3, "c4": 4}[args.whole_job]
    cfg = dict(w.config(k))
    if args.batch and args.batch < cfg["batch"]:            # the first `batch` protocols of the configuration only (a call on the GPU box is limited to one hour)
        cfg["batch"] = args.batch
        for key in ("dose", "delay", "nfrac"):
            cfg[key] = cfg[key][:args.batch]
    if k == 3:
        snap, grown_h = pregrow.grow(cfg["dims"], params, cfg["init"], cfg["rng_seed"], target_extent=cfg["pregrow_diameter"], check_h=24.0)
        cfg["t0_h"] = grown_h
    else:
        snap = warm_snapshot(binding, cfg, params, 0)
    out = full_horizon(torch, binding, cfg, params, snap, 0, label="configs[%d]%s" % (k - 1, "" if cfg["batch"] == w.config(k)["batch"] else " (first %d protocols)" % cfg["batch"]))
    out["metric"] = "protocols_per_hour_measured"
    print(json.dumps(out))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2303_08123_b200 import binding, pregrow

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit("--gpus %d but WORLD_SIZE=%d: launch N>1 with torch.distributed.run" % (args.gpus, world))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    params = w.default_params()
    cfg = dict(w.config(5))
    nx, ny, nz = cfg["dims"]
    sites = nx * ny * nz
    S = args.ca_steps or 20
    dt_h = S / params["steps_per_hour"]
    snap = warm_snapshot(binding, cfg, params, local)                      # untimed: the saved tumour
    g, B = make_batch(binding, torch, args.batch or cfg["batch"], cfg["dims"], params, 10, local)
    if world > 1:                                                           # every rank must run the same batch size
        bt = torch.tensor([B], device="cuda")
        dist.all_reduce(bt, op=dist.ReduceOp.MIN)
        if int(bt.item()) != B:
            g.close(); del g; torch.cuda.empty_cache()
            g, B = make_batch(binding, torch, int(bt.item()), cfg["dims"], params, 10, local)
    for name, val in (("fused", args.fused), ("graph_steps", args.graph_steps), ("cluster", args.cluster), ("cell_path", args.cell_path)):
        if val is not None:
            g.set_option(name, val)
    stream = g.stream
    # weak scaling: rank r evaluates global simulation ids [r*B, (r+1)*B); simulation i runs protocol i // 4 of its rank's table
    rng = np.random.default_rng(cfg["rng_seed"] + 1000 * rank)
    pd, pt, pn = (cfg["dose"], cfg["delay"], cfg["nfrac"]) if rank == 0 else w.protocols_alphabet(rng, cfg["population"])
    spp = cfg["seeds_per_protocol"]
    pro = (np.arange(B) // spp) % len(pn)
    dose, delay, nfrac = pd[pro], pt[pro], pn[pro]
    fit_dev = torch.zeros(B, dtype=torch.float32, device="cuda")

    # ---- device-resident arm: inputs in HBM before the timed region
    load_snapshot(g, snap)
    g.set_rng(cfg["rng_seed"], rank * B)
    g.set_protocols(dose, delay, nfrac, t0_h=cfg["t0_h"])
    t = cfg["t0_h"]
    for _ in range(args.warmup):
        t += dt_h
        g.run(t)
        g.fitness(out=fit_dev)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = g.launch_count
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(args.steps):
            t += dt_h
            g.run(t)
            g.fitness(out=fit_dev)
        ev1.record(stream)
    barrier()
    g.sync()
    launches = g.launch_count - launches0
    clocks = sampler.stop() if rank == 0 else None
    tm = torch.tensor([ev0.elapsed_time(ev1)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tm, op=dist.ReduceOp.MAX)
    ms_per_step = float(tm.item()) / args.steps
    value = world * B * sites * S / (ms_per_step * 1e-3)
    fit_device_arm = fit_dev.cpu().numpy().copy()
    cnt = g.counts()

    # ---- dominant kernel alone
    stage_ms, nl = time_stage(torch, g, stream, 10 if B >= 4096 else 30)
    roofline = roofline_block("k_diffuse_fused", B, sites, stage_ms, nl, ms_per_step / S, "r02_ncu_fused_c5*.txt")

    # ---- end to end through the C ABI with HOST buffers over the SAME simulated window: every step uploads the protocol
    #      table as it stands (pinned host memory -> device) and reads the fitness back to the host
    load_snapshot(g, snap)
    g.set_rng(cfg["rng_seed"], rank * B)
    pin_d = torch.empty(dose.shape, dtype=torch.float32).pin_memory().numpy()
    pin_t = torch.empty(delay.shape, dtype=torch.float32).pin_memory().numpy()
    t = cfg["t0_h"]
    fit_host = None
    e2e_t = 0.0
    h2d = d2h = 0
    for k in range(args.warmup + args.steps):
        nd, nt = remaining_table(dose, delay, nfrac, cfg["t0_h"], t)        # host bookkeeping, outside the timed part
        pin_d[:], pin_t[:] = nd, nt
        barrier()
        t0 = time.perf_counter()
        g.set_protocols(pin_d, pin_t, nfrac, t0_h=t)
        t += dt_h
        g.run(t)
        fit_host = g.fitness()
        dtk = time.perf_counter() - t0
        if k >= args.warmup:
            e2e_t += dtk
            h2d, d2h = pin_d.nbytes + pin_t.nbytes + nfrac.nbytes, fit_host.nbytes
    te = torch.tensor([e2e_t / args.steps], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e = {"value": world * B * sites * S / float(te.item()), "unit": "site-updates/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
           "ms_per_step": float(te.item()) * 1e3, "window": "the same simulated hours as the device-timed region, from the same saved tumour",
           "fitness_identical_to_device_arm": bool(np.array_equal(fit_host, fit_device_arm))}
    g.close()
    del g
    torch.cuda.empty_cache()

    if rank == 0:
        per_config, fullh, cpu = None, None, None
        if world == 1 and not args.headline_only:
            per_config = {}
            c2 = w.config(2)
            per_config["1"] = config_probe(torch, binding, "1", c2, params, snap, local, 200, "k_diffuse_fused", None)
            c3 = w.config(3)
            snap3, grown_h = pregrow.grow(c3["dims"], params, c3["init"], c3["rng_seed"], target_extent=c3["pregrow_diameter"], check_h=24.0, device=local)
            c3["t0_h"] = grown_h
            per_config["2"] = config_probe(torch, binding, "2", c3, params, snap3, local, 20, "k_diffuse_rows", "r*_ncu_rows_c3*.txt")
            per_config["2"]["pregrown_hours"] = grown_h
            per_config["2"]["pregrown_profile"] = pregrow.radial_profile(snap3)
            c4 = w.config(4)
            snap4 = warm_snapshot(binding, c4, params, local)
            per_config["3"] = config_probe(torch, binding, "3", c4, params, snap4, local, 20, "k_diffuse_rows", "r*_ncu_rows_c4*.txt")
            if not args.skip_full_horizon:
                fullh = full_horizon(torch, binding, c2, params, snap, local)
        if world == 1 and not args.no_cpu_baseline:
            osteps = args.oracle_steps
            v, dt = oracle_sample(cfg["dims"], params, snap, osteps, cfg["rng_seed"], 0)
            allc = oracle_all_cores(cfg["dims"], snap, max(50, osteps // 3), cfg["rng_seed"])
            cpu = {"value": v, "unit": "site-updates/s", "cores": 1, "kind": "oracle", "seconds": dt,
                   "sample": "1 of %d simulations x %d CA steps from the saved post-warm-up tumour (64^3)" % (B, osteps),
                   "nproc": os.cpu_count(), "cpu_model": cpu_model(),
                   "all_cores": None if allc is None else {"value": allc["value"], "unit": "site-updates/s", "cores": allc["processes"], "seconds": allc["seconds"],
                                                           "sample": "%d independent oracle processes, one simulation x %d CA steps each" % (allc["processes"], max(50, osteps // 3))}}
        horizon_steps = int(round(cfg["horizon_h"] * params["steps_per_hour"]))
        line = {"metric": "site_updates_per_s", "value": value, "unit": "site-updates/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "BASELINE configs[4]: %d sims/GPU (of the 16384 = 4096 protocols x 4 seeds) x %dx%dx%d lattice resident at once, one saved ~3k-cell spheroid, 10-fraction protocols"
                                       % (B, nx, ny, nz),
                           "batch_per_gpu": B, "resident_gb_per_gpu": 29.0 * B * sites / 1e9, "ca_steps_per_step": S, "n_sub": params["n_sub"],
                           "simulated_window_h": [cfg["t0_h"] + args.warmup * dt_h, cfg["t0_h"] + (args.warmup + args.steps) * dt_h],
                           "l2": "working set %.1f GB/GPU > 126 MB L2 (no flush needed)" % (29.0 * B * sites / 1e9),
                           "sharding": "batch over ranks, no collective"},
                "live_cells_per_sim_mean": float(cnt[:, 0].mean()),
                "protocols_per_hour": None if fullh is None else fullh["protocols_per_hour"],
                "protocols_per_hour_source": None if fullh is None else "MEASURED in this run: the whole configs[1] job, see full_horizon",
                "protocols_per_hour_headline_window": world * (B / spp) * 3600.0 / (ms_per_step * 1e-3 / S * horizon_steps),
                "protocols_per_hour_headline_window_note": "configs[4] protocols (4 seeds each) per hour IF every CA step of the 432 000 cost what the timed window costs (early treatment, ~3k-cell tumours); tumours regrow and late steps cost more, see full_horizon for a measured whole job",
                "full_horizon": fullh, "per_config": per_config,
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
                "fitness_sample": [float(x) for x in fit_host[:4]]}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--ca-steps", type=int, default=None, help="CA steps per bench step (default 20)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=0, help="simulations per GPU of the headline workload (default 16384, halved until it fits)")
    ap.add_argument("--headline-only", action="store_true", help="skip per_config and the full-horizon job")
    ap.add_argument("--skip-full-horizon", action="store_true", help="skip the measured whole configs[1] job (about 90 s)")
    ap.add_argument("--fused", type=int, default=None)
    ap.add_argument("--graph-steps", type=int, default=None)
    ap.add_argument("--cell-path", type=int, default=None, help="0: generic S2/S3 scan kernels")
    ap.add_argument("--cluster", type=int, default=None, help="CTAs per simulation of the S2+S3 kernel (1, 2, 4, 8)")
    ap.add_argument("--oracle-steps", type=int, default=1500, help="CA steps of the one-core oracle sample (about 15 s)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--probe", default=None, choices=["c2", "c3", "c4"], help="measure ONE configuration alone (with --batch: reduced batch) and print its per_config entry")
    ap.add_argument("--tumour-radius", type=float, default=None, help="--probe only: start from a seeded BALL of this radius (late, dense phase)")
    ap.add_argument("--whole-job", default=None, choices=["c2", "c3", "c4"], help="run that configuration's whole job once and print the measured protocols/hour (c3, c4: about an hour each)")
    ap.add_argument("--rows-rp", type=int, default=None, help="--probe c3 only: row pairs per lane of k_diffuse_rows (1 or 2)")
    ap.add_argument("--rows-cluster", type=int, default=None, help="--probe c3 only: 0 = slabs with a halo, 3 = clusters of 3 CTAs per plane")
    ap.add_argument("--ga", action="store_true", help="configs[4] sharded population evaluation + host GA loop at reduced size")
    ap.add_argument("--ga-population", type=int, default=128)
    ap.add_argument("--ga-generations", type=int, default=2)
    ap.add_argument("--ga-horizon-h", type=float, default=12.0)
    ap.add_argument("--ga-batch", type=int, default=128)
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.whole_job:
        run_whole_job(args)
    elif args.probe:
        run_probe(args)
    elif args.ga:
        run_ga(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
