"""GPU tests of the workloads around the hot path: the pre-grown configs[2] tumour, the configs[4]
batch at its full resident size, robustness sweeps (NEXT-4), the normality run (NEXT-2)
and long-horizon statistical parity against the fp64 oracle's committed ensemble (north_star tolerance 3)."""
import os

import numpy as np
import pytest

from oracle import ca_oracle as o
from paper_2303_08123_b200 import binding, pregrow, stats, workloads as w
from tests._parity import (oracle_from_snapshot, assert_ints_equal, assert_fields_close, assert_fields_bitwise,
                           assert_close_to_f64_up_to_threshold_flips)

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "reduced_c2_ensemble.txt")


def _free_gb():
    import torch
    torch.cuda.empty_cache()                 # earlier tests' workspaces sit in torch's caching allocator
    return torch.cuda.mem_get_info()[0] / 1e9


def test_c3_pregrown_spheroid_has_the_radial_structure_and_its_full_batch_window_matches_the_oracle():
    """BASELINE configs[2] as it states it: one simulation grown on the GPU from a single cell until the occupied set is 64
    sites across, snapshot broadcast to 512 simulations with ca_set_state, then a 50-step window with a fraction inside.
    The grown tumour has what a seeded ball lacks -- DEAD cells, quiescent cells, lysed sites, blocked READY parents -- on
    the 96^2-plane kernels; first / middle / last simulation are compared with the fp32 and fp64 oracles."""
    cfg = w.config(3)
    p = w.default_params()
    dims = cfg["dims"]
    snap, hours = pregrow.grow(dims, p, cfg["init"], cfg["rng_seed"], target_extent=cfg["pregrow_diameter"], check_h=24.0)
    prof = pregrow.radial_profile(snap)
    assert pregrow.extent(snap["state"]) >= 64
    # pin P12 at configs[2] size: proliferating rim outside the quiescent shell outside the necrotic core, core lysing
    assert prof["proliferating"][0] > 20000 and prof["quiescent"][0] > 5000 and prof["dead"][0] > 500
    assert prof["proliferating"][1] > prof["quiescent"][1] + 3 > prof["dead"][1] + 5
    assert prof["empty_inside_half_radius"] > 1000
    ready = ((snap["state"] & 0x27) == 0x24).sum()
    assert ready > 1000                                          # blocked READY parents inside the rim
    B = cfg["batch"]
    g = binding.CaBatch(B, *dims, p, max_frac=10)
    g.set_state(0, B, state=snap["state"], clock=snap["clock"], damage=snap["damage"], o2=snap["o2"], glc=snap["glc"], h=snap["h"], step=snap["step"])
    g.set_rng(cfg["rng_seed"], 0)
    dose = cfg["dose"].copy(); delay = cfg["delay"].copy()
    delay[:, 0] = 20.0 / p["steps_per_hour"]                      # first fraction 20 steps into the window
    g.set_protocols(dose, delay, cfg["nfrac"], t0_h=hours)
    g.step(50)
    cnt = g.counts()
    assert cnt[:, 1].min() > 0                                    # the fraction doomed cells everywhere
    for b in (0, B // 2 + 1, B - 1):
        gs = g.get_state(b)
        for prec in ("f32", "f64"):
            r = oracle_from_snapshot(snap, p, dims, cfg["rng_seed"], b, precision=prec)
            r.set_protocol(dose[b], delay[b], t0_h=hours)
            r.step(50)
            if prec == "f32":                                  # every decision in the kernel's precision: bit for bit
                assert_ints_equal(gs, r.get_state(), "f32 sim %d" % b)
                assert_fields_bitwise(gs, r.get_state(), "f32 sim %d" % b)
                assert cnt[b].tolist() == r.counts().tolist()
            else:                                              # 70 000 cells, some within rounding of a mode threshold
                assert_close_to_f64_up_to_threshold_flips(gs, r.get_state(), p, int(cnt[b][0]), "f64 sim %d" % b)
    g.close()


def test_c5_full_resident_batch_16384_sims():
    """The batch bench.py times for BASELINE configs[4]: 16 384 x 64^3 = 4.3e9 sites (125 GB), past 2^32 sites.  The saved
    tumour is broadcast, every simulation gets its own id and protocol; first, a middle and the last simulation of a
    24-step window (one fraction inside) must match the fp32 oracle bit for bit, fitness included."""
    if _free_gb() < 135:
        pytest.skip("needs 135 GB of free HBM")
    p = w.default_params()
    cfg = w.config(5)
    dims = cfg["dims"]
    B = 16384
    one = binding.CaBatch(1, *dims, p)
    one.seed(rng_seed=cfg["rng_seed"], **cfg["init"])
    one.step(40)
    snap = one.get_state(0)
    one.close()
    g = binding.CaBatch(B, *dims, p, max_frac=10)
    g.set_state(0, B, state=snap["state"], clock=snap["clock"], damage=snap["damage"], o2=snap["o2"], glc=snap["glc"], h=snap["h"], step=snap["step"])
    g.set_rng(cfg["rng_seed"], 0)
    dose = np.full((B, 1), 2.0); dose[B - 1, 0] = 5.0
    delay = np.full((B, 1), 8.0 / p["steps_per_hour"])
    g.set_protocols(dose, delay, t0_h=40.0 / p["steps_per_hour"])
    g.step(24)
    fit = g.fitness()
    for b in (0, 8193, B - 1):
        r = oracle_from_snapshot(snap, p, dims, cfg["rng_seed"], b, precision="f32")
        r.set_protocol(dose[b], delay[b], t0_h=40.0 / p["steps_per_hour"])
        r.step(24)
        gs = g.get_state(b)
        assert_ints_equal(gs, r.get_state(), "sim %d" % b)
        assert_fields_bitwise(gs, r.get_state(), "sim %d" % b)
        assert fit[b] == r.fitness()
    g.close()


def test_next4_robustness_sweep_rows_through_the_batched_path_match_the_oracle():
    """NEXT-4: every variant of one protocol with a fraction dropped or shifted, evaluated as ONE batch.
    Stress parameters and a BMII-shaped protocol on a minutes scale so that the oracle can follow every row to the end."""
    p = w.stress_params()
    base_dose = [2.0] * 5
    base_delay = [0.0, 0.04, 0.04, 0.04, 0.04]                     # 24-step spacing: BMII's 24 h scaled by 1/600
    dose, delay, nfrac, labels = w.robustness_sweep(base_dose, base_delay, shifts_h=(-0.01, 0.01), step_h=0.005)
    assert sum(l.startswith("drop") for l in labels) == 5
    B, n = len(nfrac), 24
    g = binding.CaBatch(B, n, n, n, p, max_frac=dose.shape[1])
    g.seed("ball", radius=4.0, rng_seed=99, sim_id_base=0, shared_init=True)
    g.set_protocols(dose, delay, nfrac)
    g.step(160)
    fit = g.fitness()
    cnt = g.counts()
    rows = [0] + [i for i, l in enumerate(labels) if l.startswith("drop")] + [B - 1]
    for b in rows:
        r = o.OracleSim(n, n, n, p)
        r.seed("ball", radius=4.0, rng_seed=99, sim_id=b, shared_init=True)
        r.set_protocol(dose[b][:nfrac[b]], delay[b][:nfrac[b]])
        r.step(160)
        assert_ints_equal(g.get_state(b), r.get_state(), labels[b])
        assert fit[b] == r.fitness() and cnt[b].tolist() == r.counts().tolist()
    # dropping a fraction leaves more survivors than the full protocol (doomed counts are what the dose did)
    assert all(cnt[b][1] <= cnt[0][1] + 60 for b in rows[1:-1])
    g.close()


def test_next2_final_count_over_2000_seeds_is_close_to_normal():
    """NEXT-2 (PAPER.md l.252 and Fig. 3D l.357: 2000 evaluations of one protocol, histogram against the normal
    distribution): BASELINE configs[0] run whole for 2000 seeds (global ids 0..1999) in one batch.  The oracle's own
    run of simulation 0 must be one of them, bit for bit in its counts (fp32 build)."""
    cfg = w.config(1)
    p = w.default_params()
    B = 2000
    g = binding.CaBatch(B, *cfg["dims"], p, max_frac=1)
    g.seed(rng_seed=cfg["rng_seed"], sim_id_base=0, **cfg["init"])
    g.set_protocols(np.repeat(cfg["dose"], B, 0), np.repeat(cfg["delay"], B, 0), t0_h=cfg["t0_h"])
    g.run(cfg["horizon_h"])
    cnt = g.counts()
    occ = cnt[:, 12].astype(np.float64)
    d, pval = stats.ks_normality(occ, discrete=True)              # integer counts, sd of a few cells: binned comparison
    mean, sd = occ.mean(), occ.std(ddof=1)
    assert sd > 0 and 0.02 < sd / mean < 0.5, (mean, sd)
    assert d < 0.04 and pval > 1e-3, (d, pval, mean, sd)
    skew = float(((occ - mean) ** 3).mean() / sd ** 3)
    assert abs(skew) < 0.6, skew
    r = o.OracleSim(*cfg["dims"], p, precision="f32")
    r.seed(cfg["init"]["kind"], center=cfg["init"]["center"], rng_seed=cfg["rng_seed"], sim_id=0)
    r.set_protocol(cfg["dose"][0], cfg["delay"][0], t0_h=cfg["t0_h"])
    r.run(cfg["horizon_h"])
    assert cnt[0].tolist() == r.counts().tolist()
    g.close()


def test_long_horizon_statistical_parity_with_the_fp64_oracle_ensemble():
    """north_star tolerance 3 / SURVEY 8(c) protocol (3) / the paper's own validation of its GPU port (PAPER.md l.69,
    l.250, Fig. 3 l.357): the reduced configs[1] job -- 8 protocols x 30 seeds, 5 simulated days after a 6 h warm-up --
    run on the GPU with the same global ids the fp64 oracle used for tests/golden/reduced_c2_ensemble.txt (written by
    tests/golden/make_reduced_c2_ensemble.py from oracle/ alone).  Per protocol: the GPU mean lies within 1 % of the
    oracle's or inside its seed-to-seed 95 % interval; neither the t-test nor KS tells the two samples apart; the
    t-test p-values over the protocols are not piled up below 0.05."""
    if not os.path.exists(GOLDEN):
        pytest.skip("golden ensemble not generated")
    rows = np.array([[int(x) for x in line.split()] for line in open(GOLDEN) if line.strip() and not line.startswith("#")])
    cfg = w.reduced_c2()
    p = w.default_params()
    npro, spp = cfg["population"], cfg["seeds_per_protocol"]
    assert len(rows) == npro * spp
    ref_occ = rows[:, 5].reshape(npro, spp).astype(np.float64)
    ref_live = rows[:, 2].reshape(npro, spp).astype(np.float64)
    B = npro * spp
    g = binding.CaBatch(B, *cfg["dims"], p, max_frac=cfg["dose"].shape[1])
    g.seed(rng_seed=cfg["rng_seed"], sim_id_base=0, **cfg["init"])      # shared_init: identical spheroid, own id for the dynamics
    pro = np.arange(B) // spp
    g.set_protocols(cfg["dose"][pro], cfg["delay"][pro], cfg["nfrac"][pro], t0_h=cfg["t0_h"])
    g.run(cfg["t0_h"] + cfg["horizon_h"])
    cnt = g.counts()
    g.close()
    gpu_occ = cnt[:, 12].reshape(npro, spp).astype(np.float64)
    gpu_live = cnt[:, 0].reshape(npro, spp).astype(np.float64)
    for name, x, y in (("occupied", gpu_occ, ref_occ), ("live", gpu_live, ref_live)):
        cmp = stats.compare_implementations(x, y)
        for k in range(npro):
            within_1pct = abs(cmp["mean_x"][k] - cmp["mean_y"][k]) <= 0.01 * cmp["mean_y"][k]
            lo, hi = np.percentile(y[k], [2.5, 97.5])
            assert within_1pct or lo <= cmp["mean_x"][k] <= hi, (name, k, cmp["mean_x"][k], cmp["mean_y"][k], lo, hi)
            assert stats.same_distribution(x[k], y[k]), (name, k, cmp["p_t"][k], cmp["p_ks"][k])
        assert stats.pvalues_not_piled_up(cmp["p_t"]), (name, cmp["p_t"])
    # the trajectories share their random streams: most simulations still agree exactly with the fp64 oracle after 75 600 steps
    # (measured in round 2: all 240 agree exactly, live and occupied; a threshold flip would show up here first)
    same = float((gpu_occ == ref_occ).mean())
    assert same > 0.9, same


def test_next3_paper_geometry_library_fitness_methodology_and_whole_run_parity():
    """NEXT-3: the paper-shaped workload -- one-plane lattice of <= 1500 sites, a library
    of 10 tumours grown for 10 days from a ~10-site seed, every protocol scored on every tumour x 8 seeds over 5 days of
    treatment + 5 days of regrowth, fitness = 1500 - n (Eq. 1), ITS against the untreated control (Eq. 2).  One of the 240
    simulations is re-run WHOLE (144 000 steps) by the fp32 build of the oracle from the same library snapshot: same counts."""
    from paper_2303_08123_b200 import ga
    cfg = w.paper_geometry()
    p = w.default_params(N_ref=cfg["n_ref"], well_mixed_medium=1)     # "well-mixed replenished substrate" (l.244): EMPTY sites are medium
    dims = cfg["dims"]
    lib = pregrow.grow_library(dims, p, cfg["init"], cfg["rng_seed"], cfg["n_tumours"], cfg["grow_h"])
    occ0 = np.array([int((((s["state"] & 7) >= 1) & ((s["state"] & 7) <= 5)).sum()) for s in lib])
    assert len(set(occ0.tolist())) > 3 and occ0.min() > 60 and occ0.max() < 1200, occ0       # ten different tumours that fit the plane
    T, S, npro = cfg["n_tumours"], cfg["seeds_per_tumour"], len(cfg["nfrac"])
    g = binding.CaBatch(npro * T * S, *dims, p, max_frac=cfg["dose"].shape[1])
    mean_fit, fit = ga.evaluate_on_library(g, lib, cfg["dose"], cfg["delay"], cfg["nfrac"], S, cfg["rng_seed"], cfg["horizon_h"])
    cnt = g.counts()
    assert fit.shape == (npro, T, S) and g.step_index == int(round((cfg["grow_h"] + cfg["horizon_h"]) * 600))
    n_mean = stats.occupied_from_fitness(mean_fit, cfg["n_ref"])
    assert (fit <= 1500).all() and (fit >= 1500 - 38 * 38).all()
    assert n_mean[0] > n_mean[1] and n_mean[0] > n_mean[2], n_mean                              # both benchmarks beat no treatment
    assert stats.its(n_mean[1], n_mean[0]) > 0.02 and stats.its(n_mean[2], n_mean[0]) > 0.02
    sd = fit.reshape(npro, -1).std(axis=1, ddof=1)
    assert (sd > 0).all()
    # whole-run parity of one simulation (BMII, tumour 3, seed 5)
    pr, j, s = 2, 3, 5
    b = (pr * T + j) * S + s
    r = oracle_from_snapshot(lib[j], p, dims, cfg["rng_seed"], b, precision="f32")
    r.set_protocol(cfg["dose"][pr][:cfg["nfrac"][pr]], cfg["delay"][pr][:cfg["nfrac"][pr]], t0_h=cfg["grow_h"])
    r.run(cfg["grow_h"] + cfg["horizon_h"])
    assert cnt[b].tolist() == r.counts().tolist()
    assert fit[pr, j, s] == r.fitness()
    g.close()


@pytest.mark.parametrize("dims", [(20, 14, 9), (40, 40, 3)])
def test_well_mixed_medium_flag_matches_the_oracle(dims):
    """The alternative reading of G2 (EMPTY sites held at the medium values) on the GPU: a 60-step stress window with
    irradiation, divisions, deaths and lysis, bit for bit against the fp32 build of the oracle and <= 1e-4 against fp64."""
    p = w.stress_params(well_mixed_medium=1)
    seed = 0x5EED77
    g = binding.CaBatch(3, *dims, p, max_frac=2)
    assert g.get_option("diffusion_kernel") == 0                   # served by the per-sub-step kernel
    c = (dims[0] // 2, dims[1] // 2, dims[2] // 2)
    g.seed("ball", center=c, radius=3.0, rng_seed=seed, sim_id_base=4)
    dose = np.array([[3.0, 2.0], [6.0, 1.5], [0.5, 4.0]])
    delay = np.array([[0.01, 0.03], [0.0, 0.05], [0.02, 0.02]])
    g.set_protocols(dose, delay)
    g.step(60)
    for b in range(3):
        gs = g.get_state(b)
        for prec in ("f32", "f64"):
            r = o.OracleSim(*dims, p, precision=prec)
            r.seed("ball", center=c, radius=3.0, rng_seed=seed, sim_id=4 + b)
            r.set_protocol(dose[b], delay[b])
            r.step(60)
            assert_ints_equal(gs, r.get_state(), "%s sim %d" % (prec, b))
            if prec == "f32":
                assert_fields_bitwise(gs, r.get_state(), "f32 sim %d" % b)
            else:
                assert_fields_close(gs, r.get_state(), p, 1e-4, "f64 sim %d" % b)
    st = g.get_state(0)
    assert np.all(st["glc"][(st["state"] & 7) == 0] == np.float32(p["boundary"][1]))      # EMPTY sites: exactly the medium value
    g.close()
