"""Pins P7-P9, P12: cycle clock, division conservation, tie-breaks."""
import itertools

import numpy as np

from oracle import ca_oracle as o
from paper_2303_08123_b200 import workloads as w
from tests import _philox_ref as pr
from tests._helpers import (blank_state, const_fields, kind, live, K_EMPTY, K_G1, K_S, K_G2, K_M, K_DEAD,
                            ST_READY, ST_DOOMED)


def _one_cell_sim(n, params, clock0, seed=3):
    sim = o.OracleSim(n, n, n, params)
    shape = (n, n, n)
    st = blank_state(n, n, n)
    ck = np.zeros(shape, np.uint16)
    c = n // 2
    st[c, c, c] = K_G1
    ck[c, c, c] = clock0
    f = const_fields(params, shape)
    sim.set_state(state=st, clock=ck, damage=np.zeros(shape, np.uint16), o2=f[0], glc=f[1], h=f[2], step=0)
    sim.set_rng(seed, 0)
    return sim, c


def test_p7_phase_changes_at_exact_steps_without_jitter():
    """J = 0, one G1 cell with clock T_G1, ample nutrients: G1->S after T0 steps, S->G2 after T0+T1, ...,
    division exactly after sum(T) steps; 1 -> 2 -> 4 with doublings exactly sum(T) apart."""
    T = [30, 48, 18, 6]
    p = w.default_params(T=T, J=[0, 0, 0, 0])
    sim, c = _one_cell_sim(12, p, T[0])
    seen = {}
    total = sum(T)
    for s in range(1, 2 * total + 1):
        sim.step(1)
        st = sim.get_state()
        n_live = int(live(st["state"]).sum())
        seen[s] = (int(kind(st["state"])[c, c, c]), n_live)
    assert seen[T[0] - 1][0] == K_G1 and seen[T[0]][0] == K_S
    assert seen[T[0] + T[1] - 1][0] == K_S and seen[T[0] + T[1]][0] == K_G2
    assert seen[T[0] + T[1] + T[2]][0] == K_M
    assert seen[total - 1] == (K_M, 1)
    assert seen[total] == (K_G1, 2)                 # READY and divided within the same step (G15)
    assert seen[2 * total - 1][1] == 2
    assert seen[2 * total][1] == 4                  # two adjacent parents: disjoint empty neighbours


def test_p7_default_cycle_length_is_17h():
    p = w.default_params(J=[0, 0, 0, 0])
    assert sum(p["T"]) == 10200                     # 5 + 8 + 3 + 1 h at 600 steps/h (G7)
    sim, c = _one_cell_sim(8, p, p["T"][0])
    sim.step(10199)
    assert sim.counts()[0] == 1
    sim.step(1)
    assert sim.counts()[0] == 2


def test_p7_quiescent_cell_does_not_advance_and_starved_cell_dies():
    p = w.default_params(J=[0, 0, 0, 0])
    n = 8
    shape = (n, n, n)
    sim, c = _one_cell_sim(n, p, 100)
    f = const_fields(p, shape)
    f[1][:] = 0.3                                   # G_Q <= G < G_P : quiescent (G5, G6)
    sim.set_state(glc=f[1])
    sim.stage_cells()
    st = sim.get_state()
    assert st["clock"][c, c, c] == 100 and ((st["state"][c, c, c] >> 3) & 3) == 2   # QA, clock frozen
    f[1][:] = 0.01                                  # below G_Q: necrosis (G5, G12)
    sim.set_state(glc=f[1])
    sim.stage_cells()
    st = sim.get_state()
    assert st["state"][c, c, c] == K_DEAD and st["clock"][c, c, c] == p["lysis_steps"]


def test_p8_conservation_through_division_and_death():
    """Per step: births = sites EMPTY -> G1; each birth has exactly one face-adjacent parent that went
    M|READY -> G1; live' = live + births - deaths; occupied' = occupied + births - lysed."""
    n = 18
    p = w.stress_params()
    sim = o.OracleSim(n, n, n, p)
    sim.seed("ball", radius=4.0, rng_seed=99, sim_id=5)
    sim.set_protocol([6.0], [0.05], t0_h=0.0)       # one big fraction at step 30 -> mitotic deaths, lysis
    total_births = total_deaths = total_lysed = 0
    prev = sim.get_state()["state"]
    for s in range(400):
        sim.stage_irradiate()
        sim.stage_diffuse()
        sim.stage_cells()
        mid = sim.get_state()["state"]
        births_reported = sim.stage_divide()
        sim.set_state(step=s + 1)
        cur = sim.get_state()["state"]
        born = (kind(mid) == K_EMPTY) & (kind(cur) == K_G1)
        assert births_reported == int(born.sum())
        assert not ((kind(mid) != K_EMPTY) & (kind(mid) != kind(cur)) & ~((kind(mid) == K_M) & (kind(cur) == K_G1))).any()
        parents = (kind(mid) == K_M) & ((mid & ST_READY) != 0) & (kind(cur) == K_G1)
        assert int(parents.sum()) == int(born.sum())
        # every birth touches >= 1 reset parent, and the bipartite parent<->birth matching is perfect:
        nb = np.zeros_like(born, dtype=int)
        for ax in range(3):
            for sh in (1, -1):
                nb += np.roll(parents, sh, axis=ax)
        assert (nb[born] >= 1).all()
        deaths = int((live(prev) & (kind(cur) == K_DEAD)).sum())
        lysed = int(((kind(prev) == K_DEAD) & (kind(mid) == K_EMPTY)).sum())   # may be re-filled by a birth
        b = int(born.sum())
        assert int(live(cur).sum()) == int(live(prev).sum()) + b - deaths
        occ = lambda a: int((live(a) | (kind(a) == K_DEAD)).sum())
        assert occ(cur) == occ(prev) + b - lysed
        total_births += b; total_deaths += deaths; total_lysed += lysed
        prev = cur
    assert total_births > 50 and total_deaths > 20 and total_lysed > 5     # the test exercised every path


def _brute_divide(state, seed, step, sim, nx, ny):
    """Independently written O-S3: for every EMPTY site list its claimants, take the minimum."""
    nz = state.shape[0]
    lin = lambda z, y, x: (z * ny + y) * nx + x
    dirs = [(0, 0, -1), (0, 0, 1), (0, -1, 0), (0, 1, 0), (-1, 0, 0), (1, 0, 0)]     # -x +x -y +y -z +z
    choice = {}
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        s = int(state[z, y, x])
        if (s & 7) != K_M or not (s & ST_READY) or ((s >> 3) & 3) >= 2:
            continue
        cand = []
        for d, (dz, dy, dx) in enumerate(dirs):
            if state[z + dz, y + dy, x + dx] == K_EMPTY:
                cand.append((pr.word0(seed, lin(z, y, x), step, sim, 4, d), d))
        if cand:
            d = min(cand)[1]
            choice[(z, y, x)] = (z + dirs[d][0], y + dirs[d][1], x + dirs[d][2])
    winners = {}
    for e in set(choice.values()):
        claim = [(pr.word0(seed, lin(*q), step, sim, 5), lin(*q), q) for q, t in choice.items() if t == e]
        winners[e] = min(claim)[2]
    return winners


def test_p9_two_parents_one_empty_site_smaller_claim_key_wins():
    p = w.default_params()
    nx, ny, nz = 5, 3, 3
    shape = (nz, ny, nx)
    for seed in range(12):
        st = blank_state(nx, ny, nz)
        st[1, 1, 1] = K_M | ST_READY
        st[1, 1, 3] = K_M | ST_READY
        sim = o.OracleSim(nx, ny, nz, p)
        f = const_fields(p, shape)
        sim.set_state(state=st, clock=np.zeros(shape, np.uint16), damage=np.zeros(shape, np.uint16),
                      o2=f[0], glc=f[1], h=f[2], step=17)
        sim.set_rng(seed, 3)
        assert sim.stage_divide() == 1
        out = sim.get_state()["state"]
        lin = lambda z, y, x: (z * ny + y) * nx + x
        k1 = pr.word0(seed, lin(1, 1, 1), 17, 3, 5)
        k3 = pr.word0(seed, lin(1, 1, 3), 17, 3, 5)
        win_x, lose_x = (1, 3) if (k1, 1) < (k3, 3) else (3, 1)
        assert kind(out)[1, 1, 2] == K_G1 and kind(out)[1, 1, win_x] == K_G1
        assert out[1, 1, lose_x] == (K_M | ST_READY)          # loser untouched, retries next step


def test_p9_brute_force_all_patterns_on_a_3x3_sheet():
    p = w.default_params()
    nx, ny, nz = 5, 5, 3
    shape = (nz, ny, nx)
    cells = [(1, y, x) for y in (1, 2, 3) for x in (1, 2, 3)]
    sim = o.OracleSim(nx, ny, nz, p)
    f = const_fields(p, shape)
    for pattern in range(512):
        st = blank_state(nx, ny, nz)
        for b, q in enumerate(cells):
            if pattern >> b & 1:
                st[q] = K_M | ST_READY
        sim.set_state(state=st, clock=np.zeros(shape, np.uint16), damage=np.zeros(shape, np.uint16),
                      o2=f[0], glc=f[1], h=f[2], step=pattern)
        sim.set_rng(0xABCDEF0123, 7)
        births = sim.stage_divide()
        out = sim.get_state()["state"]
        win = _brute_divide(st, 0xABCDEF0123, pattern, 7, nx, ny)
        assert births == len(win)
        expect = st.copy()
        for e, q in win.items():
            expect[e] = K_G1
            expect[q] = K_G1
        assert np.array_equal(out, expect), pattern
    # full interior => no births ever


def test_p9_quiescent_ready_parent_waits_and_doomed_is_inherited():
    p = w.default_params()
    nx, ny, nz = 5, 3, 3
    shape = (nz, ny, nx)
    st = blank_state(nx, ny, nz)
    st[1, 1, 1] = K_M | ST_READY | (2 << 3)                   # mode QA: not a parent (O-S3 step 1)
    st[1, 1, 3] = K_M | ST_READY | ST_DOOMED
    dm = np.zeros(shape, np.uint16); dm[1, 1, 3] = 777
    sim = o.OracleSim(nx, ny, nz, p)
    f = const_fields(p, shape)
    sim.set_state(state=st, clock=np.zeros(shape, np.uint16), damage=dm, o2=f[0], glc=f[1], h=f[2], step=0)
    sim.set_rng(1, 1)
    assert sim.stage_divide() == 1
    out = sim.get_state()
    assert out["state"][1, 1, 1] == st[1, 1, 1]
    assert out["state"][1, 1, 2] == (K_G1 | ST_DOOMED) and out["state"][1, 1, 3] == (K_G1 | ST_DOOMED)
    assert out["damage"][1, 1, 2] == 777 and out["damage"][1, 1, 3] == 777
    T, J = p["T"][0], p["J"][0]
    for x in (2, 3):
        assert T - J <= out["clock"][1, 1, x] <= T + J


def test_p12_untreated_growth_is_monotone_and_compact():
    """Qualitative sanity only (parity unpinned: the paper prints no growth law)."""
    n = 20
    p = w.stress_params()
    sim = o.OracleSim(n, n, n, p)
    sim.seed("cluster7", rng_seed=2)
    last = 7
    for _ in range(6):
        sim.step(100)
        c = sim.counts()
        assert c[0] >= last and c[3] == 0
        last = int(c[0])
    assert last > 100
    occ = live(sim.get_state()["state"])
    zz, yy, xx = np.nonzero(occ)
    r = np.sqrt((zz - 10) ** 2 + (yy - 10) ** 2 + (xx - 10) ** 2)
    r_eq = (3 * last / (4 * np.pi)) ** (1 / 3)
    assert r.max() < 1.8 * r_eq + 2                  # roughly spherical, no streamers


def test_p12_radial_order_rim_quiescent_shell_necrotic_core():
    """Pin P12, qualitative (SURVEY c.7; "a proliferating rim", quiescence, "progression of necrosis"):
    an untreated spheroid that outgrows its nutrient supply shows, from outside to inside, proliferating cells, a
    quiescent shell and a necrotic core that hollows out by lysis.  Scaled-down scenario (short cycle, uptake x16, so
    the viable depth is ~5 sites on a 30^3 lattice); the same order is checked on the GPU at BASELINE configs[2] size
    (tests/test_gpu_long.py).  Numbers are not the paper's: parity unpinned, sanity only."""
    n = 30
    p = w.default_params(T=[60, 96, 36, 12], J=[6, 10, 4, 1], lysis_steps=400)
    p["rate"] = [[16.0 * r for r in row] for row in p["rate"]]
    sim = o.OracleSim(n, n, n, p)
    sim.seed("cluster7", rng_seed=77)
    sim.step(2400)
    st = sim.get_state()["state"]
    k = st & 7
    lv = (k >= 1) & (k <= 4)
    mode = (st >> 3) & 3
    zz, yy, xx = np.indices(st.shape)
    occ = lv | (k == 5)
    c = [a[occ].mean() for a in (zz, yy, xx)]
    r = np.sqrt((zz - c[0]) ** 2 + (yy - c[1]) ** 2 + (xx - c[2]) ** 2)
    prolif, quiet, dead = lv & (mode < 2), lv & (mode >= 2), k == 5
    assert prolif.sum() > 300 and quiet.sum() > 100 and dead.sum() > 50
    assert r[prolif].mean() > r[quiet].mean() + 0.8 > r[dead].mean() + 1.6
    anaerobic = lv & ((mode & 1) == 1)
    assert r[anaerobic].mean() < r[lv & ((mode & 1) == 0)].mean()                 # oxygen runs out from the inside
    assert ((k == 0) & (r < 0.4 * r[occ].max())).sum() > 20                       # lysed core
    assert abs(c[0] - 15) < 1.5 and abs(c[1] - 15) < 1.5 and abs(c[2] - 15) < 1.5  # stays centred
