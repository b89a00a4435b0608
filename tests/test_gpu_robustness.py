"""Error behaviour and guards of the C ABI on the GPU (include/ca.h "Errors"), plus the winner-list spill path."""
import numpy as np
import pytest

from oracle import ca_oracle as o
from paper_2303_08123_b200 import binding, workloads as w
from tests._parity import oracle_from_snapshot, assert_ints_equal
from tests._helpers import blank_state, const_fields, K_M, ST_READY

pytestmark = pytest.mark.gpu


def _parents_lattice(n, spacing, params):
    """READY parents in proliferating mode on a sub-lattice of the interior, EMPTY elsewhere; fields at medium values"""
    st = blank_state(n, n, n)
    ck = np.zeros(st.shape, np.uint16)
    dm = np.zeros(st.shape, np.uint16)
    sl = slice(2, n - 2, spacing)
    st[sl, sl, sl] = K_M | ST_READY
    dm[sl, sl, sl] = 37
    f = const_fields(params, st.shape, np.float32)
    return st, ck, dm, f


def test_more_winners_than_the_shared_list_spill_and_match_the_oracle():
    """3375 uncontested or contested parents of ONE simulation divide on one step: more than the 2048 winners a CTA
    keeps in shared memory (cluster = 1), so the rest goes through the per-simulation spill list.  Result = oracle."""
    p = w.stress_params()
    n, seed = 32, 4242
    st, ck, dm, f = _parents_lattice(n, 2, p)
    assert int((st == (K_M | ST_READY)).sum()) > 2048
    for cluster in (1, 2):
        g = binding.CaBatch(2, n, n, n, p)
        g.set_option("cluster", cluster)
        g.set_rng(seed, 5)
        g.set_state(0, 2, state=st, clock=ck, damage=dm, o2=f[0], glc=f[1], h=f[2], step=0)
        g.step(3)
        for b in range(2):
            r = o.OracleSim(n, n, n, p)
            r.set_state(state=st, clock=ck, damage=dm, o2=f[0].astype(np.float64), glc=f[1].astype(np.float64), h=f[2].astype(np.float64), step=0)
            r.set_rng(seed, 5 + b)
            r.step(3)
            assert_ints_equal(g.get_state(b), r.get_state(), "cluster %d sim %d" % (cluster, b))
        assert g.counts()[0, 0] > 2 * 2048
        g.close()


def test_overflow_beyond_the_spill_list_is_reported_not_silent():
    """A 3-D checkerboard of parents gives ~0.3 n births on one step, more than the n/8 spill capacity:
    the library must say CA_EOVERFLOW at the next synchronising call, and a fresh ca_set_state clears it."""
    p = w.stress_params()
    n = 32
    st = blank_state(n, n, n)
    z, y, x = np.indices(st.shape)
    par = ((x + y + z) % 2 == 0) & (st == 0)
    st[par] = K_M | ST_READY
    ck = np.zeros(st.shape, np.uint16)
    dm = np.zeros(st.shape, np.uint16)
    f = const_fields(p, st.shape, np.float32)
    B = 32                                      # spill capacity per simulation = max(65536, B*n/8) / B = n/8 = 4096 here
    g = binding.CaBatch(B, n, n, n, p)
    g.set_option("cluster", 1)
    g.set_rng(1, 0)
    g.set_state(0, B, state=st, clock=ck, damage=dm, o2=f[0], glc=f[1], h=f[2], step=0)
    g.step(1)
    with pytest.raises(binding.CaError) as ei:
        g.sync()
    assert ei.value.code == binding.CA_EOVERFLOW
    st2, ck2, dm2, f2 = _parents_lattice(n, 4, p)
    g.set_state(0, B, state=st2, clock=ck2, damage=dm2, o2=f2[0], glc=f2[1], h=f2[2], step=0)
    g.step(1)
    g.sync()                                    # no stale error
    g.close()


def test_failed_kernel_launch_stops_the_run_with_an_error():
    """a failed diffusion launch must not be followed by S2/S3 on undiffused fields and CA_OK."""
    p = w.stress_params()
    for graph_steps in (0, 20):
        g = binding.CaBatch(2, 24, 24, 24, p)
        g.set_option("graph_steps", graph_steps)
        g.seed("ball", radius=3.0, rng_seed=9, sim_id_base=0)
        g.step(20)
        before = g.get_state(1)
        g.set_option("inject_launch_error", 1)
        with pytest.raises(binding.CaError) as ei:
            g.step(20)
        assert ei.value.code == binding.CA_ECUDA
        assert g.step_index == 20
        after = g.get_state(1)
        if graph_steps == 0:
            for k in ("state", "clock", "damage"):
                assert np.array_equal(before[k], after[k])
        g.close()
    # stage call too
    g = binding.CaBatch(1, 24, 24, 24, p)
    g.seed("ball", radius=3.0, rng_seed=9)
    g.set_option("inject_launch_error", 1)
    with pytest.raises(binding.CaError):
        g.stage(2)
    g.stage(2)                                  # the injected error is consumed
    g.close()


def test_step_aligned_fp32_delays_are_accepted_and_fire_on_the_oracle_steps():
    """0.35 h, 0.7 h, 6.1 h are whole numbers of steps but not exact in fp32 (209.9999964 ...)."""
    p = w.default_params()
    g = binding.CaBatch(1, 16, 16, 16, p, max_frac=4)
    g.seed("single", rng_seed=1)
    dose = np.array([[1.0, 1.0, 1.0, 1.0]])
    delay = np.array([[0.35, 0.7, 6.1, 0.005]])
    g.set_protocols(dose, delay)
    r = o.OracleSim(16, 16, 16, p)
    r.seed("single", rng_seed=1)
    r.set_protocol(dose[0], delay[0])
    assert r.fire_steps().tolist() == [210, 630, 4290, 4293]
    g.step(215)                                  # crosses the first fraction
    r.step(215)
    assert_ints_equal(g.get_state(0), r.get_state(), "after fraction 0")
    with pytest.raises(binding.CaError) as ei:
        g.set_protocols(np.array([[1.0]]), np.array([[0.3501]]))
    assert ei.value.code == binding.CA_EPROTO
    g.close()


def test_bad_arguments_are_rejected():
    p = w.default_params()
    with pytest.raises(binding.CaError):
        binding.CaBatch(70000, 8, 8, 8, p)
    g = binding.CaBatch(1, 16, 16, 16, p)
    g.seed("single", rng_seed=1)
    with pytest.raises(binding.CaError) as ei:
        g.run(float("nan"))
    assert ei.value.code == binding.CA_EINVAL
    with pytest.raises(binding.CaError):
        g.run(float("inf"))
    g.close()


def test_the_callers_current_device_is_left_alone():
    import torch
    p = w.default_params()
    g = binding.CaBatch(1, 16, 16, 16, p, device=0)
    g.seed("single", rng_seed=1)
    g.step(2)
    assert torch.cuda.current_device() == 0
    g.close()


def test_get_option_reports_the_diffusion_kernel_that_serves_a_lattice():
    """ca_get_option: 1 k_diffuse_fused (planes <= 64^2), 3 k_diffuse_rows (96- / 80-wide), 2 k_diffuse_slab (other widths that are
    multiples of 16), 0 the per-sub-step fallback; knobs read back what was set."""
    p = w.default_params()
    for dims, kern in (((64, 64, 8), 1), ((32, 32, 8), 1), ((96, 96, 8), 3), ((80, 80, 8), 3), ((96, 40, 8), 3), ((128, 72, 8), 2), ((37, 21, 8), 0), ((100, 100, 8), 0)):
        g = binding.CaBatch(1, *dims, p)
        assert g.get_option("diffusion_kernel") == kern, (dims, g.get_option("diffusion_kernel"))
        g.set_option("fused", 0)
        assert g.get_option("diffusion_kernel") == 0
        g.close()
    g = binding.CaBatch(2, 96, 96, 8, p)
    assert g.get_option("rows_cluster") == 0 and g.get_option("graph_steps") == 20
    g.set_option("rows_cluster", 3)
    g.set_option("graph_steps", 4)
    assert g.get_option("rows_cluster") == 3 and g.get_option("graph_steps") == 4
    with pytest.raises(binding.CaError):
        g.get_option("no_such_option")
    g.close()
    g = binding.CaBatch(1, 80, 80, 8, p)
    assert g.get_option("rows_rp") == 1              # 5 sites per lane: four rows per lane would need more than 255 registers
    with pytest.raises(binding.CaError):
        g.set_option("rows_cluster", 3)              # clusters of 3 exist for 96 x 96 planes only
    with pytest.raises(binding.CaError):
        g.set_option("rows_rp", 2)                   # ... and four rows per lane for 96-wide planes only
    g.close()
    g = binding.CaBatch(1, 96, 40, 8, p)
    assert g.get_option("rows_rp") == 2              # the default on 96-wide planes
    g.set_option("rows_rp", 1)
    assert g.get_option("rows_rp") == 1
    with pytest.raises(binding.CaError):
        g.set_option("rows_rp", 3)
    g.close()
    g = binding.CaBatch(1, 64, 64, 8, p)
    assert g.get_option("rows_rp") == 0              # not a k_diffuse_rows lattice
    g.close()


def test_two_contexts_driven_by_two_host_threads_agree_with_serial_runs():
    """kernel attributes and the work-split cache used to be process-wide statics; ctypes releases the GIL, so two
    host threads can drive two contexts at once.  Two contexts with DIFFERENT lattices (different diffusion kernels, different
    split tables) stepped concurrently must end exactly where the same contexts end when stepped one after the other."""
    import threading
    p = w.stress_params()
    specs = [((64, 64, 10), 11), ((96, 96, 8), 12), ((32, 32, 12), 13)]

    def make(dims, seed):
        g = binding.CaBatch(3, *dims, p, max_frac=2)
        g.set_option("graph_steps", 4)
        g.seed("ball", radius=3.0, rng_seed=seed, sim_id_base=1)
        g.set_protocols(np.full((3, 1), 3.0), np.full((3, 1), 0.02))
        return g

    serial = []
    for dims, seed in specs:
        g = make(dims, seed)
        g.step(48)
        serial.append([g.get_state(b) for b in range(3)])
        g.close()
    ctxs = [make(dims, seed) for dims, seed in specs]
    errs = []

    def drive(g):
        try:
            for _ in range(12):
                g.step(4)
            g.sync()
        except Exception as e:                                   # noqa: BLE001
            errs.append(e)

    ts = [threading.Thread(target=drive, args=(g,)) for g in ctxs]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errs, errs
    for g, ref in zip(ctxs, serial):
        for b in range(3):
            out = g.get_state(b)
            for k in ("state", "clock", "damage", "o2", "glc", "h"):
                assert np.array_equal(out[k], ref[b][k]), (g.nx, b, k)
        g.close()
