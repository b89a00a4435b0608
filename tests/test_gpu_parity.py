"""GPU parity tests proper: the CUDA path (through the C ABI) against the oracle, element by element
on the same seeded inputs.  Bars (BASELINE.json north_star): integer lattices bit-exact for the first
50 steps, fields within 1e-4 relative at fp32, final counts within 1 %.  In addition the fp32
diagnostic build of the oracle must match BITWISE (fields included) over the whole window."""
import numpy as np
import pytest

from oracle import ca_oracle as o
from paper_2303_08123_b200 import binding, workloads as w
from tests._parity import (oracle_from_snapshot, assert_ints_equal, assert_fields_close, assert_fields_bitwise,
                           field_rel_err)
from tests._helpers import blank_state, const_fields, live, kind, K_G1, K_M, ST_READY

pytestmark = pytest.mark.gpu


def _gpu(batch, dims, params, **kw):
    return binding.CaBatch(batch, dims[0], dims[1], dims[2], params, **kw)


@pytest.mark.parametrize("fused", [0, 1])
def test_c1_first_50_steps_bit_exact(fused):
    """BASELINE configs[0]: 32^3, 7-cell cluster, state exported EVERY step for 50 steps."""
    cfg = w.config(1)
    p = w.default_params()
    g = _gpu(1, cfg["dims"], p)
    g.set_option("fused", fused)
    g.set_option("graph_steps", 0)
    g.seed(rng_seed=cfg["rng_seed"], **cfg["init"])
    g.set_protocols(cfg["dose"], cfg["delay"], cfg["nfrac"], t0_h=cfg["t0_h"])
    r64 = o.OracleSim(*cfg["dims"], p)
    r32 = o.OracleSim(*cfg["dims"], p, precision="f32")
    for r in (r64, r32):
        r.seed(cfg["init"]["kind"], center=cfg["init"]["center"], rng_seed=cfg["rng_seed"], sim_id=0)
        r.set_protocol(cfg["dose"][0], cfg["delay"][0], t0_h=cfg["t0_h"])
    assert_ints_equal(g.get_state(), r64.get_state(), "seed")
    for s in range(1, 51):
        g.step(1); r64.step(1); r32.step(1)
        gs = g.get_state()
        assert_ints_equal(gs, r64.get_state(), "f64 step %d" % s)
        assert_fields_close(gs, r64.get_state(), p, 1e-4, "f64 step %d" % s)
        assert_ints_equal(gs, r32.get_state(), "f32 step %d" % s)
        assert_fields_bitwise(gs, r32.get_state(), "f32 step %d" % s)
    g.close()


@pytest.mark.parametrize("fused", [0, 1])
@pytest.mark.parametrize("dims", [(20, 14, 9), (37, 21, 18), (40, 40, 24)])
def test_stress_window_with_irradiation_divisions_and_deaths(dims, fused):
    """Ragged lattices, short cell cycle (many phase changes, divisions, conflicts, mitotic deaths, lysis)
    and two fractions inside the window; batch of 3 simulations with their own ids and protocols."""
    p = w.stress_params()
    seed, base = 0xC0FFEE1234, 11
    g = _gpu(3, dims, p, max_frac=4)
    g.set_option("fused", fused)
    g.seed("ball", radius=3.3, rng_seed=seed, sim_id_base=base)
    dose = np.array([[3.0, 2.0, 0.0], [6.0, 0.0, 1.5], [0.5, 4.0, 2.0]])
    delay = np.array([[0.01, 0.03, 0.01], [0.0, 0.05, 0.0], [0.02, 0.02, 0.02]])
    nfrac = np.array([3, 3, 2], np.int32)
    g.set_protocols(dose, delay, nfrac)
    refs = []
    for b in range(3):
        pair = []
        for prec in ("f64", "f32"):
            r = o.OracleSim(*dims, p, precision=prec)
            r.seed("ball", radius=3.3, rng_seed=seed, sim_id=base + b)
            r.set_protocol(dose[b, :nfrac[b]], delay[b, :nfrac[b]])
            pair.append(r)
        refs.append(pair)
    for s in range(10, 131, 10):           # the paper's every-10-steps cadence
        g.step(10)
        for b in range(3):
            r64, r32 = refs[b]
            r64.step(10); r32.step(10)
            gs = g.get_state(b)
            assert_ints_equal(gs, r32.get_state(), "f32 sim %d step %d" % (b, s))
            assert_fields_bitwise(gs, r32.get_state(), "f32 sim %d step %d" % (b, s))
            if s <= 50:
                assert_ints_equal(gs, r64.get_state(), "f64 sim %d step %d" % (b, s))
            assert_fields_close(gs, r64.get_state(), p, 1e-4, "f64 sim %d step %d" % (b, s))
    cnt = g.counts()
    for b in range(3):
        assert cnt[b].tolist() == refs[b][1].counts().tolist()
        assert abs(int(cnt[b][12]) - int(refs[b][0].counts()[12])) <= max(2, 0.01 * cnt[b][12])
    assert cnt[:, 0].sum() > 3 * 60 and cnt[:, 3].sum() > 0 and cnt[:, 1].sum() > 0     # grew, died, doomed: paths exercised
    fit = g.fitness()
    for b in range(3):
        assert fit[b] == refs[b][1].fitness()
    g.close()


def test_single_stages_against_oracle_stages():
    """The paper's 'single step tests' per stage: same snapshot in, same snapshot out."""
    dims = (24, 20, 16)
    p = w.stress_params()
    seed = 77
    base = o.OracleSim(*dims, p)
    base.seed("ball", radius=4.0, rng_seed=seed, sim_id=2)
    base.set_protocol([2.0], [0.1])
    base.step(60)                                            # fraction fires at step 60: next stage_irradiate
    snap = base.get_state()
    g = _gpu(2, dims, p)
    g.set_state(0, 2, state=snap["state"], clock=snap["clock"], damage=snap["damage"],
                o2=snap["o2"], glc=snap["glc"], h=snap["h"], step=snap["step"])
    g.set_rng(seed, 1)                                       # sim 1 of the batch has global id 2
    g.set_protocols(np.array([[2.0], [2.0]]), np.array([[0.0], [0.0]]), t0_h=0.1)
    r32 = oracle_from_snapshot({k: (v.astype(np.float32) if k in ("o2", "glc", "h") else v) for k, v in snap.items()},
                               p, dims, seed, 2, "f32")
    r32.set_protocol([2.0], [0.0], t0_h=0.1)
    for stage, fn in ((0, r32.stage_irradiate), (1, r32.stage_diffuse), (2, r32.stage_cells), (3, r32.stage_divide)):
        g.stage(stage); fn()
        gs = g.get_state(1)
        gs["step"] = r32.get_state()["step"]
        assert_ints_equal(gs, r32.get_state(), "stage %d" % stage)
        assert_fields_bitwise(gs, r32.get_state(), "stage %d" % stage)
    assert (g.get_state(1)["damage"] > 0).any()
    g.close()


@pytest.mark.parametrize("fused", [0, 1])
def test_diffusion_closed_form_and_uniform_invariance_on_gpu(fused):
    """Pins P3 and P5 applied directly to the CUDA stencil (fp32): discrete sine mode decays by g^m;
    a uniform field stays bitwise constant."""
    dims = (32, 32, 32)
    nx, ny, nz = dims
    p = w.default_params()
    shape = (nz, ny, nx)
    b = np.asarray(p["boundary"], np.float32).astype(np.float64)
    lam = np.asarray(p["lambda"], np.float32).astype(np.float64)
    ax = [np.sin(np.pi * np.arange(n) / (n - 1)) for n in (nz, ny, nx)]
    mode = ax[0][:, None, None] * ax[1][None, :, None] * ax[2][None, None, :]
    for a in (mode[0], mode[-1], mode[:, 0], mode[:, -1], mode[:, :, 0], mode[:, :, -1]):
        a[...] = 0
    f = [(b[s] + 0.25 * b[s] * mode).astype(np.float32) for s in range(3)]
    g = _gpu(1, dims, p)
    g.set_option("fused", fused)
    z16 = np.zeros(shape, np.uint16)
    g.set_state(0, 1, state=blank_state(nx, ny, nz), clock=z16, damage=z16, o2=f[0], glc=f[1], h=f[2], step=0)
    steps = 250
    for _ in range(steps):
        g.stage(1)                                           # n_sub = 4 sub-steps each
    out = g.get_state()
    geo = 3 * (1 - np.cos(np.pi / 31))
    for s, name in enumerate(("o2", "glc", "h")):
        expect = b[s] + 0.25 * b[s] * (1 - 2 * lam[s] * geo) ** (steps * p["n_sub"]) * mode
        assert (np.abs(out[name] - expect) / b[s]).max() < 1e-5, name
    cf = const_fields(p, shape, np.float32)
    g.set_state(0, 1, o2=cf[0], glc=cf[1], h=cf[2])
    g.step(100)
    out = g.get_state()
    for s, name in enumerate(("o2", "glc", "h")):
        assert (out[name] == cf[s]).all()
    g.close()


def test_p13_batch_independence_and_graph_equivalence():
    """A simulation's trajectory is bitwise the same alone, inside a batch, and with or without CUDA graphs;
    ca_run(a); ca_run(b) == ca_run(b)."""
    dims = (22, 22, 22)
    p = w.stress_params()
    seed = 99
    dose = np.array([[2.0, 1.0]]); delay = np.array([[0.05, 0.05]])
    outs = []
    for batch, base, graph, split in ((1, 5, 0, False), (4, 2, 20, False), (4, 2, 6, True)):
        g = _gpu(batch, dims, p, max_frac=2)
        g.set_option("graph_steps", graph)
        g.seed("cluster7", rng_seed=seed, sim_id_base=base)
        g.set_protocols(np.repeat(dose, batch, 0), np.repeat(delay, batch, 0))
        if split:
            g.run(0.05); g.run(0.11); g.run(0.25)
        else:
            g.run(0.25)
        outs.append(g.get_state(5 - base))
        assert g.step_index == 150
        g.close()
    for other in outs[1:]:
        for k in ("state", "clock", "damage", "o2", "glc", "h"):
            assert np.array_equal(outs[0][k], other[k]), k
    assert live(outs[0]["state"]).sum() > 7


def test_state_roundtrip_broadcast_and_errors():
    dims = (12, 10, 9)
    p = w.default_params()
    g = _gpu(3, dims, p, max_frac=3)
    with pytest.raises(binding.CaError) as e:
        g.step(1)
    assert e.value.code == binding.CA_ESTATE
    r = o.OracleSim(*dims, p)
    r.seed("ball", radius=2.5, rng_seed=4, sim_id=0)
    snap = r.get_state()
    rng = np.random.default_rng(0)
    snap["damage"] = (rng.integers(0, 5000, snap["damage"].shape) * live(snap["state"])).astype(np.uint16)
    g.set_state(0, 3, state=snap["state"], clock=snap["clock"], damage=snap["damage"], o2=snap["o2"], glc=snap["glc"], h=snap["h"], step=123)
    for b in range(3):
        out = g.get_state(b)
        assert out["step"] == 123
        for k in ("state", "clock", "damage"):
            assert np.array_equal(out[k], snap[k])
        for k in ("o2", "glc", "h"):
            assert np.array_equal(out[k], snap[k].astype(np.float32))
    bad = snap["state"].copy(); bad[0, 0, 0] = 0
    with pytest.raises(binding.CaError) as e:
        g.set_state(0, 1, state=bad)
    assert e.value.code == binding.CA_EINVAL
    for dose, delay in (([[-1.0]] * 3, [[1.0]] * 3), ([[1.0]] * 3, [[1.0 / 7]] * 3), ([[1.0]] * 3, [[0.0]] * 3)):
        with pytest.raises(binding.CaError) as e:           # negative dose / misaligned delay / in the past (step 123)
            g.set_protocols(np.array(dose), np.array(delay))
        assert e.value.code == binding.CA_EPROTO
    with pytest.raises(binding.CaError):
        g.set_protocols(np.zeros((3, 4)), np.zeros((3, 4)), t0_h=1.0)          # exceeds max_frac
    with pytest.raises(binding.CaError):
        g.run(0.0)                                                              # in the past
    cnt = g.counts()
    assert (cnt == np.asarray(r.counts())[None, :]).all()
    g.close()


@pytest.mark.parametrize("dims,n_sub,opts", [
    ((32, 32, 12), 4, {}),                                   # fixed 32x32 kernel, map from the diffusion kernel, default cluster
    ((64, 64, 10), 4, {"cluster": 1}),                       # fixed 64x64 kernel
    ((64, 64, 10), 4, {"cluster": 2, "graph_steps": 4}),     # clustered S2+S3 across 2 CTAs, inside CUDA graphs
    ((64, 64, 10), 4, {"graph_steps": 4}),                   # short CUDA graphs
    ((64, 64, 10), 4, {"cell_path": 0}),                     # generic scan kernels next to the fused diffusion
    ((32, 32, 12), 3, {}),                                   # 3 fused levels
    ((32, 32, 12), 6, {"graph_steps": 4}),                   # 3 + 3 levels, two passes (buffer flips twice per step)
    ((32, 32, 12), 5, {"graph_steps": 2}),                   # 3 + 2: odd number of flips per step
    ((48, 32, 9), 2, {}),                                    # run-time-dims fused kernel, map built by k_occ_map
    ((96, 96, 9), 4, {}),                                    # configs[2] plane: k_diffuse_rows, 4 y-slabs of 32 rows, spheroid on the cuts
    ((96, 96, 9), 4, {"rows_rp": 1, "rows_cluster": 3, "graph_steps": 4}), # the same plane on clusters of 3 CTAs: boundary rows through distributed shared memory
    ((96, 96, 9), 4, {"rows_rp": 1}),                        # the same plane with two rows per lane (16 warps; four rows per lane is the default)
    ((96, 40, 7), 3, {"rows_rp": 1, "graph_steps": 2}),      # ... on a non-square plane with a short last slab, 3 levels
    ((80, 80, 9), 4, {"graph_steps": 6}),                    # configs[3] plane: k_diffuse_rows, 2 y-slabs of 44 rows
    ((96, 40, 7), 4, {}),                                    # k_diffuse_rows on a plane that is not square: 2 slabs, map from k_occ_map
    ((80, 52, 6), 2, {}),                                    # k_diffuse_rows, 2 levels, a short second slab (duplicate row pairs)
    ((128, 72, 8), 3, {}),                                   # k_diffuse_slab: 2 column blocks with an x-seam, 3 y-slabs
])
def test_fast_path_variants_against_the_oracle(dims, n_sub, opts):
    """Every launch configuration of the fast path gives the oracle's lattice: bit-exact integers and (against the
    fp32 build) bit-exact fields over a 60-step window with irradiation, divisions, deaths and lysis; batch of 4."""
    p = w.stress_params(n_sub=n_sub)
    seed, base, B = 0xABCD0123, 5, 4
    g = _gpu(B, dims, p, max_frac=2)
    for k, v in opts.items():
        g.set_option(k, v)
    g.seed("ball", radius=3.4, rng_seed=seed, sim_id_base=base)
    dose = np.array([[3.0, 2.0], [6.0, 0.5], [0.5, 4.0], [1.0, 1.0]])
    delay = np.array([[0.01, 0.03], [0.0, 0.05], [0.02, 0.02], [0.03, 0.04]])
    g.set_protocols(dose, delay)
    refs = []
    for b in range(B):
        pair = []
        for prec in ("f64", "f32"):
            r = o.OracleSim(*dims, p, precision=prec)
            r.seed("ball", radius=3.4, rng_seed=seed, sim_id=base + b)
            r.set_protocol(dose[b], delay[b])
            pair.append(r)
        refs.append(pair)
    for s in (7, 20, 40, 60):                                 # uneven strides: graphs + single steps + irradiation splits
        g.run(s / p["steps_per_hour"])
        for b in range(B):
            r64, r32 = refs[b]
            r64.run(s / p["steps_per_hour"]); r32.run(s / p["steps_per_hour"])
            gs = g.get_state(b)
            assert_ints_equal(gs, r32.get_state(), "f32 sim %d step %d" % (b, s))
            assert_fields_bitwise(gs, r32.get_state(), "f32 sim %d step %d" % (b, s))
            if s <= 50:
                assert_ints_equal(gs, r64.get_state(), "f64 sim %d step %d" % (b, s))
            assert_fields_close(gs, r64.get_state(), p, 1e-4, "f64 sim %d step %d" % (b, s))
    cnt = g.counts()
    for b in range(B):
        assert cnt[b].tolist() == refs[b][1].counts().tolist()
    assert cnt[:, 0].sum() > B * 60 and cnt[:, 1].sum() > 0
    g.close()


def test_streamed_population_evaluation_is_batch_size_independent():
    """configs[4] driver: protocols x seeds streamed through a fixed-size batch give, simulation by simulation, the
    same fitness whatever the batch size, and the same as the oracle started from the same saved tumour."""
    from paper_2303_08123_b200 import ga
    p = w.stress_params()
    dims, seed = (32, 32, 12), 99
    g0 = _gpu(1, dims, p, max_frac=2)
    g0.seed("ball", radius=3.0, rng_seed=seed, sim_id_base=0)
    g0.step(12)
    snap = g0.get_state(0)
    g0.close()
    rng = np.random.default_rng(4)
    npro, spp = 5, 3
    dose = rng.choice([0.5, 2.0, 4.0], (npro, 2)); delay = rng.choice([0.01, 0.02, 0.03], (npro, 2)); nfrac = np.full(npro, 2, np.int32)
    t0 = snap["step"] / p["steps_per_hour"]
    t_end = t0 + 60 / p["steps_per_hour"]
    res = []
    for B in (4, 15, 7):
        g = _gpu(B, dims, p, max_frac=2)
        mean, per_sim = ga.evaluate_population(g, snap, dose, delay, nfrac, spp, seed, t0, t_end)
        res.append(per_sim)
        g.close()
    assert np.array_equal(res[0], res[1]) and np.array_equal(res[0], res[2])
    for sim in (0, 7, 14):                                    # spot-check against the oracle (fp32 build: identical decisions)
        r = oracle_from_snapshot(snap, p, dims, seed, sim, precision="f32")
        r.set_protocol(dose[sim // spp], delay[sim // spp], t0_h=t0)
        r.run(t_end)
        assert res[0][sim] == r.fitness(), sim


def test_dense_starving_tumour_long_window_all_cell_paths_agree():
    """A dense spheroid with strong uptake: quiescent READY cells, starvation deaths, lysis, blocked parents that become
    unblocked -- the situations the blocked-parent memory of the clustered kernel has to get right.  The oracle (fp32
    build) is followed for 240 steps, the generic and the clustered GPU paths are compared bit for bit over 900."""
    p = w.stress_params(lysis_steps=25)
    p["rate"] = [[-4e-3, 0.0, -2e-3, 0.0], [-2.4e-2, -7e-2, -1.2e-2, -3.5e-2], [1.5e-7, 6e-7, 0.75e-7, 3e-7]]
    dims, seed, B = (32, 32, 32), 777, 3
    dose = np.array([[2.0, 3.0]] * B); delay = np.array([[0.25, 0.5]] * B)
    runs = []
    for cell_path in (1, 0):
        g = _gpu(B, dims, p, max_frac=2)
        g.set_option("cell_path", cell_path)
        g.seed("ball", radius=8.5, rng_seed=seed, sim_id_base=40)
        g.set_protocols(dose, delay)
        snaps = []
        for s in (240, 600, 900):
            g.run(s / p["steps_per_hour"])
            snaps.append([g.get_state(b) for b in range(B)])
        runs.append((snaps, g.counts()))
        g.close()
    (sa, ca_), (sb_, cb) = runs
    assert np.array_equal(ca_, cb)
    for k in range(3):
        for b in range(B):
            assert_ints_equal(sa[k][b], sb_[k][b], "paths, window %d sim %d" % (k, b))
            assert_fields_bitwise(sa[k][b], sb_[k][b], "paths, window %d sim %d" % (k, b))
    c = ca_.sum(0)
    assert c[3] > 0 and c[2] > 0 and (c[10] + c[11]) > 0, c          # dead cells, READY cells, quiescent cells all present
    r = o.OracleSim(*dims, p, precision="f32")
    r.seed("ball", radius=8.5, rng_seed=seed, sim_id=41)
    r.set_protocol(dose[1], delay[1])
    r.run(240 / p["steps_per_hour"])
    assert_ints_equal(sa[0][1], r.get_state(), "oracle f32, 240 steps")
    assert_fields_bitwise(sa[0][1], r.get_state(), "oracle f32, 240 steps")


@pytest.mark.parametrize("dims", [(3, 3, 3), (4, 4, 3), (6, 8, 3), (64, 64, 3), (64, 4, 5), (4, 64, 4), (96, 4, 3), (8, 68, 4)])
def test_degenerate_lattices(dims):
    """Smallest and thinnest lattices: one interior plane, one interior row, a single interior site; a lone cell, then
    (where there is room) its first divisions.  Integers and fields bit-identical to the fp32 oracle, fp64 within 1e-4."""
    p = w.stress_params()
    seed = 31
    g = _gpu(2, dims, p, max_frac=1)
    g.seed("single", rng_seed=seed, sim_id_base=7)
    g.set_protocols(np.array([[1.0], [0.0]]), np.array([[5 / p["steps_per_hour"]], [0.0]]), np.array([1, 0], np.int32))
    refs = []
    for b in range(2):
        pair = []
        for prec in ("f32", "f64"):
            r = o.OracleSim(*dims, p, precision=prec)
            r.seed("single", rng_seed=seed, sim_id=7 + b)
            if b == 0:
                r.set_protocol([1.0], [5 / p["steps_per_hour"]])
            pair.append(r)
        refs.append(pair)
    for s in (1, 11, 50, 120):
        g.run(s / p["steps_per_hour"])
        for b in range(2):
            gs = g.get_state(b)
            for r in refs[b]:
                r.run(s / p["steps_per_hour"])
            assert_ints_equal(gs, refs[b][0].get_state(), "f32 sim %d step %d" % (b, s))
            assert_fields_bitwise(gs, refs[b][0].get_state(), "f32 sim %d step %d" % (b, s))
            if s <= 50:
                assert_ints_equal(gs, refs[b][1].get_state(), "f64 sim %d step %d" % (b, s))
            assert_fields_close(gs, refs[b][1].get_state(), p, 1e-4, "f64 sim %d step %d" % (b, s))
    assert g.fitness().tolist() == [refs[0][0].fitness(), refs[1][0].fitness()]
    g.close()
