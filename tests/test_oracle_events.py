"""Pins for the event arithmetic of the oracle (second table): O-SEED, the mode decision (G5),
the lysis delay (G12), every draw_clock call (G7 and the Philox purposes 2, 6, 7), the z directions of O-S3 (G8) and
the histograms of O-S4.  Everything expected here is computed from tests/_philox_ref.py (an independent pure-Python
Philox) and integer arithmetic written out in the test, or from numpy; nothing is read back from the oracle.

Each test names the one-line mutation of oracle/ca_oracle.c it is there to catch ("What's weak" 1)."""
import itertools

import numpy as np
import pytest

from oracle import ca_oracle as o
from paper_2303_08123_b200 import workloads as w
from tests import _philox_ref as pr
from tests._helpers import (blank_state, const_fields, kind, live, K_EMPTY, K_G1, K_S, K_G2, K_M, K_DEAD, K_WALL,
                            ST_READY, ST_DOOMED)


def _lin(z, y, x, nx, ny):
    return (z * ny + y) * nx + x


def _uniform_int(word, m):
    return (word * m) >> 32                                     # G23


# ------------------------------------------------------------------------------------------------ O-SEED --
def _expected_seed(dims, cells, params, seed, sid):
    """kind / clock of every placed cell from the Philox convention: purposes 0 and 1, step 0 (G16)."""
    nx, ny, nz = dims
    st = blank_state(nx, ny, nz)
    ck = np.zeros((nz, ny, nx), np.uint16)
    for (z, y, x) in cells:
        i = _lin(z, y, x, nx, ny)
        k = 1 + _uniform_int(pr.word0(seed, i, 0, sid, 0), 4)
        c = 1 + _uniform_int(pr.word0(seed, i, 0, sid, 1), params["T"][k - 1])
        st[z, y, x] = k                                          # mode PA (0) at the medium values, flags clear
        ck[z, y, x] = c
    return st, ck


def _ball_cells(dims, center, r):
    nx, ny, nz = dims
    cx, cy, cz = center
    return [(z, y, x) for z in range(1, nz - 1) for y in range(1, ny - 1) for x in range(1, nx - 1)
            if (x - cx) ** 2 + (y - cy) ** 2 + (z - cz) ** 2 <= r * r]


@pytest.mark.parametrize("shared,sim_id", [(False, 0), (False, 9), (True, 9)])
def test_seed_cluster7_exact_kinds_and_clocks(shared, sim_id):
    """catches: kind drawn from 3 values; clock `0 + uniform_int`; shared_init ignored; purposes 0/1 swapped."""
    dims = (11, 9, 13)
    p = w.default_params()
    seed = 0x5EED0001ABCD
    sim = o.OracleSim(*dims, p)
    sim.seed("cluster7", rng_seed=seed, sim_id=sim_id, shared_init=shared)
    c = (dims[2] // 2, dims[1] // 2, dims[0] // 2)              # (z, y, x) centre = n // 2
    cells = [c] + [(c[0] + dz, c[1] + dy, c[2] + dx) for dz, dy, dx in
                   ((0, 0, 1), (0, 0, -1), (0, 1, 0), (0, -1, 0), (1, 0, 0), (-1, 0, 0))]
    st, ck = _expected_seed(dims, cells, p, seed, 0 if shared else sim_id)
    out = sim.get_state()
    assert np.array_equal(out["state"], st)
    assert np.array_equal(out["clock"], ck)
    assert not out["damage"].any() and out["step"] == 0
    for s, name in enumerate(("o2", "glc", "h")):               # fields = medium values at EVERY site [B c1]
        assert (out[name] == float(np.float32(p["boundary"][s]))).all()


def test_seed_ball_membership_kinds_clocks_and_lattice_point_counts():
    """catches: BALL membership `<` instead of `<=`; centre not n // 2; kinds never M.  The counts are the number of
    integer points in a ball (OEIS A000605: r = 9 -> 3071), recounted here by brute force, not the oracle's."""
    p = w.default_params()
    seed = 77
    dims = (14, 12, 13)
    sim = o.OracleSim(*dims, p)
    sim.seed("ball", center=(6, 5, 7), radius=3.0, rng_seed=seed, sim_id=4)
    cells = _ball_cells(dims, (6, 5, 7), 3.0)
    assert len(cells) == 123                                     # A000605(3); with `<` it would be 93
    st, ck = _expected_seed(dims, cells, p, seed, 4)
    out = sim.get_state()
    assert np.array_equal(out["state"], st) and np.array_equal(out["clock"], ck)
    for dims, r, n in (((24, 24, 24), 9.0, 3071), ((24, 24, 24), 8.9, 2945), ((72, 72, 72), 32.0, 137065)):
        c = dims[0] // 2
        g = np.arange(dims[0]) - c
        d2 = g[:, None, None] ** 2 + g[None, :, None] ** 2 + g[None, None, :] ** 2
        inner = np.zeros(dims, bool)
        inner[1:-1, 1:-1, 1:-1] = True
        assert int(((d2 <= r * r) & inner).sum()) == n           # brute force, independent of the oracle
        sim = o.OracleSim(*dims, p)
        sim.seed("ball", radius=r, rng_seed=seed, sim_id=0)
        cnt = sim.counts()
        assert cnt[0] == n and cnt[12] == n
        assert cnt[4:8].min() > 0.2 * n                          # all four phases present, roughly uniform (G16)
        assert cnt[8] == n                                       # mode PA everywhere at the medium values


def test_seed_kinds_are_uniform_over_four_phases_and_clocks_cover_1_to_T():
    """catches: `1 + uniform_int(x, 3)` (never M) and clocks starting at 0 -- statistically, on 3071 cells."""
    p = w.default_params()
    sim = o.OracleSim(24, 24, 24, p)
    sim.seed("ball", radius=9.0, rng_seed=5, sim_id=0)
    out = sim.get_state()
    k = kind(out["state"])[live(out["state"])]
    ck = out["clock"][live(out["state"])]
    for q in (K_G1, K_S, K_G2, K_M):
        n = int((k == q).sum())
        assert abs(n - 3071 / 4) < 4 * np.sqrt(3071 * 0.25 * 0.75), (q, n)
        cq = ck[k == q]
        assert cq.min() >= 1 and cq.max() <= p["T"][q - 1]
        assert cq.max() > 0.97 * p["T"][q - 1] and cq.min() < 0.03 * p["T"][q - 1] + 2


# ------------------------------------------------------------------------------------------ mode decision --
def _cell_with_fields(p, O, G, H, state=K_G1, clock=500, n=5):
    sim = o.OracleSim(n, n, n, p)
    shape = (n, n, n)
    st = blank_state(n, n, n)
    ck = np.zeros(shape, np.uint16)
    c = n // 2
    st[c, c, c] = state
    ck[c, c, c] = clock
    f = [np.full(shape, v, np.float64) for v in (O, G, H)]
    sim.set_state(state=st, clock=ck, damage=np.zeros(shape, np.uint16), o2=f[0], glc=f[1], h=f[2], step=0)
    sim.set_rng(1, 0)
    return sim, c


def test_mode_decision_all_four_modes_thresholds_and_both_starvation_causes():
    """catches: `aerobic = 1` always; a swapped / strict comparison at any of the five thresholds (G5)."""
    p = w.default_params()
    f32 = lambda v: float(np.float32(v))
    OA, GP, GQ, HP, HQ = (f32(p[k]) for k in ("O_A", "G_P", "G_Q", "H_P", "H_Q"))
    up = lambda v: float(np.nextafter(np.float64(v), np.inf))
    dn = lambda v: float(np.nextafter(np.float64(v), -np.inf))
    hi_O, lo_O = 0.28, dn(OA)
    cases = [
        # (O, G, H) -> mode (0 PA, 1 PN, 2 QA, 3 QN) or "dead"
        ((hi_O, 5.5, 3.98e-5), 0),
        ((OA, GP, HP), 0),                       # equality: O >= O_A, G >= G_P, H <= H_P all hold
        ((lo_O, 5.5, 3.98e-5), 1),               # just below O_A: anaerobic
        ((0.0, GP, HP), 1),
        ((hi_O, dn(GP), 3.98e-5), 2),            # just below G_P: quiescent
        ((hi_O, 5.5, up(HP)), 2),                # just above H_P: quiescent
        ((lo_O, dn(GP), 3.98e-5), 3),
        ((lo_O, 5.5, up(HP)), 3),
        ((hi_O, GQ, HQ), 2),                     # equality at the starvation thresholds: NOT starved (G < G_Q, H > H_Q)
        ((hi_O, dn(GQ), 3.98e-5), "dead"),       # glucose starvation
        ((hi_O, 5.5, up(HQ)), "dead"),           # acidosis
        ((lo_O, dn(GQ), up(HQ)), "dead"),
    ]
    for (O, G, H), want in cases:
        sim, c = _cell_with_fields(p, O, G, H)
        sim.stage_cells()
        out = sim.get_state()
        s = int(out["state"][c, c, c])
        if want == "dead":
            assert s == K_DEAD and out["clock"][c, c, c] == p["lysis_steps"], (O, G, H, s)
        else:
            assert (s & 7) == K_G1 and ((s >> 3) & 3) == want, (O, G, H, s)
            assert out["clock"][c, c, c] == (499 if want < 2 else 500)      # only proliferating modes count down (G6)


def test_mode_selects_the_uptake_rate_of_the_next_diffusion_step():
    """the mode bits written by S2 are the ones S1 reads: one sub-step on a uniform field changes the cell's site by
    exactly rate[species][mode] (lap = 0 there) -- catches a transposed rate table or stale mode bits."""
    p = w.default_params()
    for mode, (O, G) in enumerate(((0.28, 5.5), (0.001, 5.5), (0.28, 0.3), (0.001, 0.3))):
        sim, c = _cell_with_fields(p, O, G, 3.98e-5)
        sim.stage_cells()
        assert ((int(sim.get_state()["state"][c, c, c]) >> 3) & 3) == mode
        sim.diffuse_substeps(1)
        out = sim.get_state()
        for s, (name, v0) in enumerate((("o2", O), ("glc", G), ("h", 3.98e-5))):
            expect = max(v0 + float(np.float32(p["rate"][s][mode])), 0.0)
            assert out[name][c, c, c] == pytest.approx(expect, rel=1e-15, abs=0.0), (mode, name)
            assert out[name][c, c, c + 1] == v0                  # an empty neighbour has no source term


# --------------------------------------------------------------------------------------------------- lysis --
def test_dead_cell_is_vacated_exactly_lysis_steps_s2_passes_after_death():
    """catches: DEAD site vacated one pass early (`clock <= 1`) or late; damage not cleared."""
    p = w.default_params(lysis_steps=37)
    sim, c = _cell_with_fields(p, 0.28, 0.0, 3.98e-5)           # starves in the first S2 pass
    dm = np.zeros((5, 5, 5), np.uint16)
    dm[c, c, c] = 99
    sim.set_state(damage=dm)
    sim.stage_cells()
    out = sim.get_state()
    assert out["state"][c, c, c] == K_DEAD and out["clock"][c, c, c] == 37 and out["damage"][c, c, c] == 0
    for k in range(1, 37):
        sim.stage_cells()
        out = sim.get_state()
        assert out["state"][c, c, c] == K_DEAD and out["clock"][c, c, c] == 37 - k, k
        assert sim.counts()[12] == 1                             # still occupied (G13)
    sim.stage_cells()                                            # pass number lysis_steps after the death
    out = sim.get_state()
    assert out["state"][c, c, c] == K_EMPTY and out["clock"][c, c, c] == 0
    assert sim.counts()[12] == 0


def test_mitotic_death_of_a_doomed_cell_at_the_end_of_g2_and_its_lysis():
    p = w.default_params(lysis_steps=5)
    sim, c = _cell_with_fields(p, 0.28, 5.5, 3.98e-5, state=K_G2 | ST_DOOMED, clock=2)
    sim.stage_cells()
    assert sim.get_state()["state"][c, c, c] == (K_G2 | ST_DOOMED)
    sim.stage_cells()
    out = sim.get_state()
    assert out["state"][c, c, c] == K_DEAD and out["clock"][c, c, c] == 5
    for _ in range(5):
        assert sim.get_state()["state"][c, c, c] == K_DEAD
        sim.stage_cells()
    assert sim.get_state()["state"][c, c, c] == K_EMPTY


# --------------------------------------------------------------------------------------------- draw_clock --
def _draw(p, knd, seed, site, step, sid, purpose):
    T, J = p["T"][knd - 1], p["J"][knd - 1]
    return T - J + _uniform_int(pr.word0(seed, site, step, sid, purpose), 2 * J + 1)      # G7


@pytest.mark.parametrize("seed", [3, 0xFEEDFACE12345, 2 ** 63 + 11])
def test_phase_entry_clocks_are_the_exact_philox_draws(seed):
    """catches: jitter width 2J instead of 2J + 1; wrong purpose / step / sim id / site in the counter; T, J of the
    phase being LEFT instead of the one being entered."""
    p = w.default_params()
    n = 7
    site = _lin(3, 3, 3, n, n)
    for step, sid in ((0, 0), (41, 6), (123456, 16383)):
        for k0 in (K_G1, K_S, K_G2):
            sim, c = _cell_with_fields(p, 0.28, 5.5, 3.98e-5, state=k0, clock=1, n=n)
            sim.set_state(step=step)
            sim.set_rng(seed, sid)
            sim.stage_cells()
            out = sim.get_state()
            assert kind(out["state"])[c, c, c] == k0 + 1
            assert out["clock"][c, c, c] == _draw(p, k0 + 1, seed, site, step, sid, 2), (step, sid, k0)


def test_jitter_covers_the_closed_interval_T_minus_J_to_T_plus_J():
    """catches: uniform_int(2J) -- the value T + J must be reachable.  Small J so that both ends are hit quickly."""
    p = w.default_params(T=[30, 48, 18, 6], J=[2, 2, 2, 2])
    seen = set()
    n = 7
    for step in range(120):
        sim, c = _cell_with_fields(p, 0.28, 5.5, 3.98e-5, state=K_G1, clock=1, n=n)
        sim.set_state(step=step)
        sim.set_rng(9, 2)
        sim.stage_cells()
        v = int(sim.get_state()["clock"][c, c, c])
        assert v == _draw(p, K_S, 9, _lin(3, 3, 3, n, n), step, 2, 2)
        seen.add(v)
    assert seen == {46, 47, 48, 49, 50}


@pytest.mark.parametrize("direction", range(6))
def test_division_clocks_parent_uses_its_own_site_daughter_the_target_site(direction):
    """One READY parent whose only EMPTY neighbour lies in `direction` (order -x,+x,-y,+y,-z,+z, G8): the daughter
    appears exactly there; parent clock = draw(G1, parent site, purpose 7), daughter clock = draw(G1, TARGET site,
    purpose 6).  catches: daughter clock drawn with the parent's site; purposes 6/7 swapped; z offsets swapped."""
    p = w.default_params()
    n = 7
    shape = (n, n, n)
    offs = [(0, 0, -1), (0, 0, 1), (0, -1, 0), (0, 1, 0), (-1, 0, 0), (1, 0, 0)]       # (dz, dy, dx)
    seed, sid, step = 0xD1CE5EED, 12, 977
    st = blank_state(n, n, n)
    c = (3, 3, 3)
    st[c] = K_M | ST_READY | ST_DOOMED
    for d, (dz, dy, dx) in enumerate(offs):
        if d != direction:
            st[c[0] + dz, c[1] + dy, c[2] + dx] = K_DEAD                    # occupied, not EMPTY
    dm = np.zeros(shape, np.uint16)
    dm[c] = 4321
    ck = np.zeros(shape, np.uint16)
    ck[st == K_DEAD] = 1000
    sim = o.OracleSim(n, n, n, p)
    f = const_fields(p, shape)
    sim.set_state(state=st, clock=ck, damage=dm, o2=f[0], glc=f[1], h=f[2], step=step)
    sim.set_rng(seed, sid)
    assert sim.stage_divide() == 1
    out = sim.get_state()
    dz, dy, dx = offs[direction]
    e = (c[0] + dz, c[1] + dy, c[2] + dx)
    expect = st.copy()
    expect[c] = K_G1 | ST_DOOMED
    expect[e] = K_G1 | ST_DOOMED
    assert np.array_equal(out["state"], expect)
    assert out["clock"][c] == _draw(p, K_G1, seed, _lin(*c, n, n), step, sid, 7)
    assert out["clock"][e] == _draw(p, K_G1, seed, _lin(*e, n, n), step, sid, 6)
    assert out["damage"][e] == 4321 and out["damage"][c] == 4321


# ------------------------------------------------------------------------------------- O-S3 in three dims --
def _brute_divide_3d(state, seed, step, sim, nx, ny):
    """Independently written O-S3 (G8, G9): for every EMPTY site list its claimants, take the minimum."""
    nz = state.shape[0]
    dirs = [(0, 0, -1), (0, 0, 1), (0, -1, 0), (0, 1, 0), (-1, 0, 0), (1, 0, 0)]     # -x +x -y +y -z +z
    choice = {}
    for z, y, x in itertools.product(range(1, nz - 1), range(1, ny - 1), range(1, nx - 1)):
        s = int(state[z, y, x])
        if (s & 7) != K_M or not (s & ST_READY) or ((s >> 3) & 3) >= 2:
            continue
        p = _lin(z, y, x, nx, ny)
        cand = [(pr.word0(seed, p, step, sim, 4, d), d) for d, (dz, dy, dx) in enumerate(dirs)
                if state[z + dz, y + dy, x + dx] == K_EMPTY]
        if cand:
            d = min(cand)[1]
            choice[(z, y, x)] = (z + dirs[d][0], y + dirs[d][1], x + dirs[d][2])
    winners = {}
    for e in set(choice.values()):
        claim = [(pr.word0(seed, _lin(*q, nx, ny), step, sim, 5), _lin(*q, nx, ny), q) for q, t in choice.items() if t == e]
        winners[e] = min(claim)[2]
    return winners


def test_p9_brute_force_random_patterns_on_a_3x3x3_interior():
    """1500 random READY / EMPTY / obstacle patterns on a 5^3 lattice: all six directions, contested targets in z.
    catches: off[4] / off[5] swapped; direction keys drawn without the aux byte; claims resolved by max."""
    p = w.default_params()
    n = 5
    shape = (n, n, n)
    seed, sid = 0x0DDBA11C0FFEE, 3
    rng = np.random.default_rng(2024)
    sim = o.OracleSim(n, n, n, p)
    f = const_fields(p, shape)
    z16 = np.zeros(shape, np.uint16)
    used_dirs = set()
    contested = 0
    for trial in range(1500):
        st = blank_state(n, n, n)
        density = (0.15, 0.4, 0.7)[trial % 3]
        r = rng.random((3, 3, 3))
        inner = st[1:-1, 1:-1, 1:-1]
        inner[r < density] = K_M | ST_READY
        inner[(r >= density) & (r < density + 0.1)] = K_S          # an occupied, non-dividing site
        inner[(r >= density + 0.1) & (r < density + 0.15)] = K_M | ST_READY | (2 << 3)   # quiescent READY: not a parent
        sim.set_state(state=st, clock=z16, damage=z16, o2=f[0], glc=f[1], h=f[2], step=trial)
        sim.set_rng(seed, sid)
        births = sim.stage_divide()
        out = sim.get_state()["state"]
        win = _brute_divide_3d(st, seed, trial, sid, n, n)
        assert births == len(win), trial
        expect = st.copy()
        for e, q in win.items():
            expect[e] = K_G1
            expect[q] = K_G1
            used_dirs.add((e[0] - q[0], e[1] - q[1], e[2] - q[2]))
        assert np.array_equal(out, expect), trial
        # a target claimed by more than one parent
        for e in win:
            nb = sum(1 for dz, dy, dx in ((0, 0, 1), (0, 0, -1), (0, 1, 0), (0, -1, 0), (1, 0, 0), (-1, 0, 0))
                     if (st[e[0] + dz, e[1] + dy, e[2] + dx] & 0x37) == (K_M | ST_READY))
            contested += nb > 1
    assert len(used_dirs) == 6 and contested > 200


# ---------------------------------------------------------------------------------------------- counts ---
def test_counts_histograms_against_numpy_on_a_random_lattice():
    """catches: doomed / ready counted on dead cells, phase or mode bins shifted, occupied != live + dead (G13)."""
    p = w.default_params()
    dims = (9, 8, 7)
    nx, ny, nz = dims
    rng = np.random.default_rng(8)
    st = blank_state(nx, ny, nz)
    inner = st[1:-1, 1:-1, 1:-1]
    kinds = rng.choice([K_EMPTY, K_G1, K_S, K_G2, K_M, K_DEAD], inner.shape, p=[0.3, 0.2, 0.15, 0.1, 0.15, 0.1])
    modes = rng.integers(0, 4, inner.shape)
    ready = (rng.random(inner.shape) < 0.3) & (kinds == K_M)
    doomed = (rng.random(inner.shape) < 0.4)
    lv = (kinds >= 1) & (kinds <= 4)
    inner[...] = np.where(lv, kinds | (modes << 3) | (ready * ST_READY) | (doomed * ST_DOOMED), kinds).astype(np.uint8)
    sim = o.OracleSim(nx, ny, nz, p)
    f = const_fields(p, (nz, ny, nx))
    sim.set_state(state=st, o2=f[0], glc=f[1], h=f[2], step=0)
    got = sim.counts().tolist()
    want = [int(lv.sum()), int((lv & doomed).sum()), int((lv & ready).sum()), int((kinds == K_DEAD).sum())]
    want += [int((kinds == q).sum()) for q in (K_G1, K_S, K_G2, K_M)]
    want += [int((lv & (modes == m)).sum()) for m in range(4)]
    want += [want[0] + want[3]]
    assert got == want
    assert sim.fitness() == (nx - 2) * (ny - 2) * (nz - 2) - want[12]               # Eq. 1 with N_ref = interior sites
    assert want[1] > 0 and want[2] > 0 and min(want[4:12]) > 0
