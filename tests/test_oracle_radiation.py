"""Pins P10, P11, P14, P15: dose-response closed forms, incomplete repair,
scheduling, and Eq. 1 / Eq. 2 against values the paper prints."""
import math
import os

import numpy as np
import pytest

from oracle import ca_oracle as o
from paper_2303_08123_b200 import workloads as w
from tests._helpers import blank_state, const_fields, kind, live, K_G1, K_S, K_G2, K_M, K_DEAD, ST_DOOMED


def _filled(n, params, phase, clock=60000, o2=None):
    """Interior filled with one phase; uptake is whatever params say; fields at boundary values."""
    sim = o.OracleSim(n, n, n, params)
    shape = (n, n, n)
    st = blank_state(n, n, n)
    st[1:-1, 1:-1, 1:-1] = phase
    ck = np.zeros(shape, np.uint16)
    ck[1:-1, 1:-1, 1:-1] = clock
    f = const_fields(params, shape)
    if o2 is not None:
        f[0][:] = o2
    sim.set_state(state=st, clock=ck, damage=np.zeros(shape, np.uint16), o2=f[0], glc=f[1], h=f[2], step=0)
    sim.set_rng(2024, 1)
    return sim


def _doomed_fraction(sim):
    st = sim.get_state()["state"]
    lv = live(st)
    return float(((st & ST_DOOMED) != 0)[lv].mean()), int(lv.sum())


def _binom_ok(frac, p, n, z=4.0):
    return abs(frac - p) <= z * math.sqrt(max(p * (1 - p), 1e-12) / n) + 1e-12


@pytest.mark.parametrize("phase", [K_G1, K_S, K_G2, K_M])
def test_p10_lq_survival_on_a_uniform_population(phase):
    n = 32
    p = w.default_params(oer_m=1.0)                 # omf == 1 exactly
    sim = _filled(n, p, phase)
    sim.set_protocol([2.0], [0.0])
    sim.stage_irradiate()
    frac, cells = _doomed_fraction(sim)
    a = float(np.float32(p["alpha"][phase - 1])); b = float(np.float32(p["beta"][phase - 1]))
    expect = 1 - math.exp(-a * 2.0 - b * 4.0)
    assert cells == 27000 and _binom_ok(frac, expect, cells), (frac, expect)
    if phase == K_G1:
        assert abs(expect - 0.4621) < 5e-4          # the number SURVEY.md P10 prints for G1, d_e = 2
    dmg = sim.get_state()["damage"]
    assert (dmg[1:-1, 1:-1, 1:-1] == 2048).all()    # 1024 * d_e, G10 step 4


def test_p10_oxygen_modification_limits():
    n = 24
    p = w.default_params()
    m, K = float(np.float32(p["oer_m"])), float(np.float32(p["oer_K"]))
    a, b = float(np.float32(p["alpha"][0])), float(np.float32(p["beta"][0]))
    # anoxic: d_e = d / m (textbook OER)
    sim = _filled(n, p, K_G1, o2=0.0)
    sim.set_protocol([3.0], [0.0]); sim.stage_irradiate()
    frac, cells = _doomed_fraction(sim)
    de = 3.0 / m
    assert _binom_ok(frac, 1 - math.exp(-a * de - b * de * de), cells)
    assert (sim.get_state()["damage"][1:-1, 1:-1, 1:-1] == 1024).all()
    # medium oxygen: omf(0.28) = 0.990610
    O = float(np.float32(0.28))
    omf = (m * O + K) / ((O + K) * m)
    assert abs(omf - 0.990610) < 1e-6
    sim = _filled(n, p, K_G1)
    sim.set_protocol([3.0], [0.0]); sim.stage_irradiate()
    frac, cells = _doomed_fraction(sim)
    de = 3.0 * omf
    assert _binom_ok(frac, 1 - math.exp(-a * de - b * de * de), cells)
    assert (sim.get_state()["damage"][1:-1, 1:-1, 1:-1] == math.floor(1024 * de + 0.5)).all()


def test_p10_zero_dose_is_a_no_op_and_20gy_sterilises():
    n = 14
    p = w.stress_params()
    runs = []
    for dose in (None, 0.0):
        sim = o.OracleSim(n, n, n, p)
        sim.seed("cluster7", rng_seed=5)
        if dose is not None:
            sim.set_protocol([dose], [0.05])
        sim.step(120)
        runs.append(sim.get_state())
    for k in ("state", "clock", "damage", "o2", "glc", "h"):
        assert np.array_equal(runs[0][k], runs[1][k])
    # single 20 Gy on an all-G1 population: kill probability 1 - 4e-8 per cell
    pd = w.default_params(oer_m=1.0)
    sim = _filled(16, pd, K_G1)
    sim.set_protocol(*w.PROTOCOL_SINGLE20)
    sim.stage_irradiate()
    frac, cells = _doomed_fraction(sim)
    assert frac == 1.0
    # ... and every doomed cell dies at the end of G2, then lyses: occupied reaches 0
    ps = w.stress_params(oer_m=1.0)
    sim = o.OracleSim(n, n, n, ps)
    sim.seed("ball", radius=3.0, rng_seed=5)
    sim.set_protocol([20.0], [0.0])
    sim.step(1)
    c = sim.counts()
    assert c[1] == c[0] > 0
    sim.step(2 * (sum(ps["T"]) + sum(ps["J"])) + ps["lysis_steps"] + 5)
    c = sim.counts()
    assert c[0] == 0 and c[12] == 0, c.tolist()


def _repair(D, events, shift):
    for _ in range(events):
        if D > 0:
            D -= max(1, D >> shift)
    return D


@pytest.mark.parametrize("gap", [0, 600, 3000])
def test_p11_incomplete_repair_two_fractions(gap):
    """survival = exp(-a(d1+d2) - b(d1^2 + d2^2 + 2 d1 d2 rho)), rho = D(gap)/(1024 d1); gap = 0 is LQ of
    d1+d2 (the fractions fire in list order on one step)."""
    n = 32
    d1, d2 = 2.0, 1.5
    p = w.default_params(oer_m=1.0, rate=[[0.0] * 4, [0.0] * 4, [0.0] * 4])
    a, b = float(np.float32(p["alpha"][0])), float(np.float32(p["beta"][0]))
    sim = _filled(n, p, K_G1)
    sim.set_protocol([d1, d2], [0.0, gap / 600.0])
    sim.step(gap + 1)
    frac, cells = _doomed_fraction(sim)
    events = gap // p["repair_period"]              # K2 repairs when (s+1) % period == 0, s = 0..gap-1
    D = _repair(2048, events, p["repair_shift"])
    rho = D / (1024.0 * d1)
    surv = math.exp(-a * (d1 + d2) - b * (d1 * d1 + d2 * d2 + 2 * d1 * d2 * rho))
    assert cells == 27000 and _binom_ok(frac, 1 - surv, cells), (frac, 1 - surv)
    if gap == 0:
        assert rho == 1.0 and abs(surv - math.exp(-a * 3.5 - b * 3.5 ** 2)) < 1e-15
    # distinguishability: the no-repair and full-repair predictions are outside the interval for gap=600
    if gap == 600:
        for bad_rho in (1.0, 0.0):
            bad = 1 - math.exp(-a * (d1 + d2) - b * (d1 * d1 + d2 * d2 + 2 * d1 * d2 * bad_rho))
            assert not _binom_ok(frac, bad, cells)


def test_p11_repair_half_time():
    """default rule: x15/16 every 60 steps -> half-time ln2/ln(16/15)*60 steps = 64.4 min."""
    p = w.default_params(oer_m=1.0, rate=[[0.0] * 4, [0.0] * 4, [0.0] * 4])
    sim = _filled(8, p, K_G1)
    sim.set_protocol([8.0], [0.0])                  # D = 8192
    sim.step(1)
    assert sim.get_state()["damage"][4, 4, 4] == 8192
    sim.step(643)                                   # 644 steps done -> 10 repair events (at s+1 = 60..600)
    assert sim.get_state()["damage"][4, 4, 4] == _repair(8192, 10, 4)
    sim.step(16)                                    # 660 steps -> 11 events: just below one half
    D = int(sim.get_state()["damage"][4, 4, 4])
    assert D == _repair(8192, 11, 4) and 0.47 < D / 8192 < 0.5
    assert abs(math.log(2) / math.log(16 / 15) * 60 / 10 - 64.4) < 0.05   # minutes


def test_p14_scheduling():
    p = w.default_params()
    sim = o.OracleSim(8, 8, 8, p)
    sim.seed("single", rng_seed=1)
    sim.set_protocol(*w.PROTOCOL_BMII)              # 5 x 2 Gy, 24 h apart, first at t = 0
    assert sim.fire_steps().tolist() == [0, 14400, 28800, 43200, 57600]
    sim.set_protocol(*w.PROTOCOL_BMI)               # 8 x 1.25 Gy: 0, 6, 24, 30, 48, 54, 72, 78 h
    assert sim.fire_steps().tolist() == [0, 3600, 14400, 18000, 28800, 32400, 43200, 46800]
    sim.set_protocol([2.0], [24.0])                 # BASELINE configs[0]
    assert sim.fire_steps().tolist() == [14400]
    sim.set_protocol([1.0, 1.0], [0.5, 0.0], t0_h=6.0)
    assert sim.fire_steps().tolist() == [3900, 3900]
    with pytest.raises(ValueError):
        sim.set_protocol([1.0], [1.0 / 7.0])        # not a whole number of steps
    with pytest.raises(ValueError):
        sim.set_protocol([-1.0], [1.0])
    sim.step(10)
    with pytest.raises(ValueError):
        sim.set_protocol([1.0], [0.0])              # already in the past


def test_p14_fraction_beyond_the_end_never_fires_and_run_is_resumable():
    p = w.stress_params()
    a = o.OracleSim(12, 12, 12, p); a.seed("cluster7", rng_seed=8); a.set_protocol([2.0, 2.0], [0.1, 1.0])
    b = o.OracleSim(12, 12, 12, p); b.seed("cluster7", rng_seed=8); b.set_protocol([2.0], [0.1])
    a.run(0.5); b.run(0.25); b.run(0.5)             # second fraction of `a` is at 1.1 h > 0.5 h
    sa, sb = a.get_state(), b.get_state()
    assert sa["step"] == sb["step"] == 300
    for k in ("state", "clock", "damage", "o2", "glc", "h"):
        assert np.array_equal(sa[k], sb[k])
    assert sa["damage"].max() > 0                   # the first fraction did fire


def test_p15_eq1_eq2_against_printed_values():
    gold = os.path.join(os.path.dirname(__file__), "golden", "paper_fitness_pairs.txt")
    p = w.default_params(N_ref=1500)                # the paper's constant
    n = 14
    shape = (n, n, n)
    rows = 0
    for line in open(gold):
        line = line.split("#")[0].strip()
        if not line:
            continue
        _, f_i, _, f_ref, printed = line.split()
        f_i, f_ref, printed = float(f_i), float(f_ref), float(printed)
        # Eq. 2 on n = 1500 - f reproduces the printed percentage to its printed precision
        its = ((1500 - f_ref) - (1500 - f_i)) / (1500 - f_ref) * 100
        assert abs(its - printed) < 0.051, (line, its)
        # Eq. 1 in the oracle: a lattice with round(n) occupied sites (live + dead) has f = 1500 - n
        occ = int(round(1500 - f_i))
        st = blank_state(n, n, n)
        flat = st[1:-1, 1:-1, 1:-1].reshape(-1)
        flat[: occ - 10] = K_G1
        flat[occ - 10: occ] = K_DEAD
        st[1:-1, 1:-1, 1:-1] = flat.reshape(n - 2, n - 2, n - 2)
        sim = o.OracleSim(n, n, n, p)
        f = const_fields(p, shape)
        sim.set_state(state=st, o2=f[0], glc=f[1], h=f[2], step=0)
        assert sim.fitness() == 1500 - occ
        assert sim.counts()[12] == occ
        rows += 1
    assert rows == 7
    # default N_ref = interior sites (G14)
    sim = o.OracleSim(n, n, n, w.default_params())
    sim.seed("cluster7", rng_seed=1)
    assert sim.fitness() == (n - 2) ** 3 - 7
