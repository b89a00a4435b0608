"""Long-horizon and full-size parity: BASELINE configs[0] run whole; configs[1] in the launch
configuration bench.py times, compared on snapshot windows the oracle can afford."""
import numpy as np
import pytest

from oracle import ca_oracle as o
from paper_2303_08123_b200 import binding, workloads as w
from tests._parity import oracle_from_snapshot, assert_ints_equal, assert_fields_close, assert_fields_bitwise

pytestmark = pytest.mark.gpu


def test_c1_whole_run_final_counts():
    """configs[0]: 32^3, 48 h, one 2 Gy fraction at 24 h.  Final counts within 1 % of the fp64 oracle
    (north_star); the fp32 diagnostic oracle must agree bitwise at the end of the whole run."""
    cfg = w.config(1)
    p = w.default_params()
    g = binding.CaBatch(1, *cfg["dims"], p)
    g.seed(rng_seed=cfg["rng_seed"], **cfg["init"])
    g.set_protocols(cfg["dose"], cfg["delay"], cfg["nfrac"], t0_h=cfg["t0_h"])
    g.run(cfg["horizon_h"])
    gs = g.get_state()
    gc = g.counts()[0]
    refs = {}
    for prec in ("f64", "f32"):
        r = o.OracleSim(*cfg["dims"], p, precision=prec)
        r.seed(cfg["init"]["kind"], center=cfg["init"]["center"], rng_seed=cfg["rng_seed"], sim_id=0)
        r.set_protocol(cfg["dose"][0], cfg["delay"][0], t0_h=cfg["t0_h"])
        r.run(cfg["horizon_h"])
        refs[prec] = r
    assert gs["step"] == 28800
    assert_ints_equal(gs, refs["f32"].get_state(), "c1 end, f32 oracle")
    assert_fields_bitwise(gs, refs["f32"].get_state(), "c1 end, f32 oracle")
    rc = refs["f64"].counts()
    assert gc[0] > 7 and gc[3] > 0                          # it grew, and cells doomed by the fraction at 24 h died
    for k in (0, 12):
        assert abs(int(gc[k]) - int(rc[k])) <= max(1, 0.01 * rc[k]), (k, gc.tolist(), rc.tolist())
    assert_fields_close(gs, refs["f64"].get_state(), p, 1e-4, "c1 end")
    assert g.fitness()[0] == float(30 ** 3 - gc[12])
    g.close()


def test_c2_full_size_snapshot_windows():
    """configs[1] at full size (64 sims x 64^3, the configuration bench.py times): run to checkpoints
    (quasi-steady warm-up; just after the first fraction), export sampled simulations, let the oracle
    advance each snapshot 50 steps, compare (SURVEY 8(c) comparison protocol (2))."""
    cfg = w.config(2)
    p = w.default_params()
    dims = cfg["dims"]
    g = binding.CaBatch(cfg["batch"], *dims, p, max_frac=10)
    g.seed(rng_seed=cfg["rng_seed"], sim_id_base=cfg["sim_id_base"], **cfg["init"])
    g.set_protocols(cfg["dose"], cfg["delay"], cfg["nfrac"], t0_h=cfg["t0_h"])
    first_fire = int(round((cfg["t0_h"] + cfg["delay"][:, 0].min()) * 600))
    b_first = int(np.argmin(cfg["delay"][:, 0]))
    for checkpoint, sims in ((600, (0, 63)), (first_fire - 20, (b_first, 17))):
        g.step(checkpoint - g.step_index)
        snaps = {b: g.get_state(b) for b in sims}
        g.step(50)
        for b in sims:
            after = g.get_state(b)
            for prec in ("f64", "f32"):
                r = oracle_from_snapshot(snaps[b], p, dims, cfg["rng_seed"], cfg["sim_id_base"] + b, prec)
                nf = int(cfg["nfrac"][b])
                # remaining fractions of this simulation, re-expressed from the snapshot's step
                t = cfg["t0_h"] + np.cumsum(cfg["delay"][b, :nf])
                keep = t * 600 >= snaps[b]["step"] - 1e-6
                if keep.any():
                    d = cfg["dose"][b, :nf][keep]
                    tt = t[keep]
                    r.set_protocol(d, np.diff(np.concatenate([[0.0], tt])), t0_h=0.0)
                r.step(50)
                ref = r.get_state()
                assert_ints_equal(after, ref, "c2 sim %d @%d %s" % (b, checkpoint, prec))
                if prec == "f32":
                    assert_fields_bitwise(after, ref, "c2 sim %d @%d" % (b, checkpoint))
                else:
                    assert_fields_close(after, ref, p, 1e-4, "c2 sim %d @%d" % (b, checkpoint))
    st = g.get_state(b_first)
    assert (st["damage"] > 0).any()                          # the first fraction fired inside the second window
    g.close()


def test_c2_shape_100_hours_fast_path_equals_generic_path():
    """configs[1] lattice and protocols, 4 simulations, 100 simulated hours (60 000 CA steps, several fractions fire):
    the fast path (fused diffusion, clustered S2+S3 with its blocked-parent memory, CUDA graphs) and the generic path
    (one launch per sub-step, scan kernels, no graphs) must end in bit-identical lattices and fields."""
    cfg = w.config(2)
    p = w.default_params()
    B = 4
    out = []
    for fast in (1, 0):
        g = binding.CaBatch(B, *cfg["dims"], p, max_frac=10)
        g.set_option("fused", fast); g.set_option("cell_path", fast)
        if not fast:
            g.set_option("graph_steps", 0)
        g.seed(rng_seed=cfg["rng_seed"], sim_id_base=0, **cfg["init"])
        g.set_protocols(cfg["dose"][:B], cfg["delay"][:B], cfg["nfrac"][:B], t0_h=0.0)
        g.run(100.0)
        out.append(([g.get_state(b) for b in range(B)], g.counts()))
        g.close()
    (sa, ca_), (sb, cb) = out
    assert np.array_equal(ca_, cb), (ca_[:, :4], cb[:, :4])
    assert ca_[:, 1].sum() > 0 and ca_[:, 0].min() > 3000          # doomed cells exist, tumours grew
    for b in range(B):
        for k in ("state", "clock", "damage", "o2", "glc", "h"):
            assert np.array_equal(sa[b][k], sb[b][k]), (b, k)


@pytest.mark.parametrize("k,batch,dims", [(3, 512, (96, 96, 96)), (4, 1024, (80, 80, 80))])
def test_c3_c4_full_batch_size_window_against_the_oracle(k, batch, dims):
    """configs[2] / configs[3] at their FULL batch size (13 / 15 GB of lattice state: 64-bit indexing, tiled diffusion
    kernel, occupancy map, clusters): a 30-step window from ca_seed with one fraction inside, first / middle / last
    simulation against the fp32 and fp64 oracles."""
    p = w.default_params()
    cfg = w.config(k)
    g = binding.CaBatch(batch, *dims, p, max_frac=8)
    g.seed("ball", radius=12.0, rng_seed=cfg["rng_seed"], sim_id_base=0, shared_init=False)
    dose = np.full((batch, 1), 2.0); dose[-1, 0] = 6.0
    delay = np.full((batch, 1), 10.0 / p["steps_per_hour"])
    g.set_protocols(dose, delay)
    g.step(30)
    cnt = g.counts()
    assert cnt[:, 0].min() > 6000 and cnt[:, 1].min() > 0
    for b in (0, batch // 2 + 1, batch - 1):
        gs = g.get_state(b)
        for prec in ("f32", "f64"):
            r = o.OracleSim(*dims, p, precision=prec)
            r.seed("ball", radius=12.0, rng_seed=cfg["rng_seed"], sim_id=b)
            r.set_protocol(dose[b], delay[b])
            r.step(30)
            assert_ints_equal(gs, r.get_state(), "%s sim %d" % (prec, b))
            if prec == "f32":
                assert_fields_bitwise(gs, r.get_state(), "f32 sim %d" % b)
                assert cnt[b].tolist() == r.counts().tolist()
            else:
                assert_fields_close(gs, r.get_state(), p, 1e-4, "f64 sim %d" % b)
    g.close()


def test_c5_sized_batch_4096_sims():
    """A configs[4]-sized batch (4096 x 64^3 = 1.07e9 sites, 31 GB): first, a middle and the last simulation of a 24-step
    window against the fp32 oracle -- 64-bit indexing of every kernel at the size the streaming driver uses."""
    p = w.default_params()
    cfg = w.config(5)
    B = 4096
    g = binding.CaBatch(B, 64, 64, 64, p, max_frac=10)
    g.seed(rng_seed=cfg["rng_seed"], sim_id_base=0, kind="ball", radius=9.0, shared_init=False)
    dose = np.tile(np.array([[2.0]]), (B, 1)); delay = np.full((B, 1), 8.0 / p["steps_per_hour"])
    g.set_protocols(dose, delay)
    g.step(24)
    fit = g.fitness()
    for b in (0, 2049, B - 1):
        r = o.OracleSim(64, 64, 64, p, precision="f32")
        r.seed("ball", radius=9.0, rng_seed=cfg["rng_seed"], sim_id=b)
        r.set_protocol(dose[b], delay[b])
        r.step(24)
        gs = g.get_state(b)
        assert_ints_equal(gs, r.get_state(), "sim %d" % b)
        assert_fields_bitwise(gs, r.get_state(), "sim %d" % b)
        assert fit[b] == r.fitness()
    g.close()


@pytest.mark.parametrize("k,batch", [(4, 512), (3, 512)])
def test_full_batch_runs_are_deterministic_and_match_the_generic_path(k, batch):
    """Two identical fast-path contexts and one fully generic one (per-sub-step diffusion, scan kernels) of the configs[3] /
    configs[2] job at a batch with thousands of work units per diffusion launch, 1800 CA steps from the saved tumour: every
    count of every simulation must agree, and the complete state of a few simulations bit for bit.  Regression test for a
    race in k_diffuse_rows (the bulk store of a segment's last plane read its descriptor after the next segment's had been
    written): about one simulation in 500 was corrupted within 1200 steps, which no 60-step parity window ever saw."""
    p = w.default_params()
    cfg = w.config(k)
    dims = cfg["dims"]
    one = binding.CaBatch(1, *dims, p, max_frac=1)
    one.seed("ball", center=tuple(d // 2 for d in dims), radius=9.0, rng_seed=cfg["rng_seed"], shared_init=True)
    one.step(600)
    snap = one.get_state(0)
    one.close()
    res, ctxs = [], []
    for opts in ({}, {}, {"fused": 0, "cell_path": 0}):
        g = binding.CaBatch(batch, *dims, p, max_frac=cfg["dose"].shape[1])
        for name, v in opts.items():
            g.set_option(name, v)
        g.set_state(0, batch, state=snap["state"], clock=snap["clock"], damage=snap["damage"], o2=snap["o2"], glc=snap["glc"], h=snap["h"], step=snap["step"])
        g.set_rng(cfg["rng_seed"], 0)
        dose = cfg["dose"][:batch].copy(); delay = cfg["delay"][:batch].copy()
        delay[:, 0] = 1.0 + (np.arange(batch) % 3) * 0.5          # first fractions inside the window, at three different steps
        g.set_protocols(dose, delay, cfg["nfrac"][:batch], t0_h=1.0)
        g.step(1800)
        res.append(g.counts())
        ctxs.append(g)
    assert res[0][:, 1].min() > 0                                  # every simulation was irradiated
    for i in (1, 2):
        bad = np.argwhere((res[i] != res[0]).any(axis=1)).ravel()
        assert len(bad) == 0, (i, bad[:8].tolist(), res[i][bad[0]].tolist(), res[0][bad[0]].tolist())
    for b in (0, batch // 3, batch - 1):
        ref = ctxs[2].get_state(b)
        for g in ctxs[:2]:
            out = g.get_state(b)
            for name in ("state", "clock", "damage", "o2", "glc", "h"):
                assert np.array_equal(out[name], ref[name]), (b, name)
    for g in ctxs:
        g.close()
