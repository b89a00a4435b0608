"""Seeded synthetic inputs shared by the CUDA path, the oracle, the tests and bench.py.

This module holds DATA ONLY: default model parameters, lattice/initial-state
recipes and protocol generators for BASELINE.json configs[0..4] (c1..c5).  None
of the method's arithmetic lives here (no stencil, no state machine, no RNG of
the method) -- it is the one module both sides may receive inputs from.

The paper's workload -- ten 10-day-old library tumours grown from 200 cells
 under protocols on a 0.25 Gy / 0.5 h grid within 120 h and
sum(dose) <= 10 Gy -- is NOT in this container (no library,
no calibrated parameter set).  The recipes below stand in for it, with the
shapes BASELINE.json's configs fix; DESIGN.md section 6 states them.
"""
import copy

import numpy as np

MASTER_SEED = 230308123

# Default parameter set ("O-PARAM").  Medium values are the
# paper's (glucose 5.5 mM, O2 0.28 mM, pH 7.4 -> [H+] 3.98e-5 mM);
# 600 steps/h is PAPER.md l.262.  Everything else is this build's reading.  The uptake / production rates were tuned once
# (round 2) against pin P12 at BASELINE configs[2] size -- a spheroid grown from one cell to 64 sites across on 96^3 shows a
# proliferating rim (mean radius 22.8 sites), a quiescent shell (16.2) and a necrotic, partly lysed core (dead cells at
# 12.5, ~6900 vacated sites inside half the radius) -- and are frozen since.
_DEFAULT = {
    "steps_per_hour": 600,
    "n_sub": 4,
    "lambda": [0.15, 0.05, 0.10],                  # O2, glucose, H+
    "boundary": [0.28, 5.5, 3.98e-5],
    # signed source per sub-step [species][mode PA, PN, QA, QN]
    "rate": [
        [-6e-4, 0.0, -3e-4, 0.0],                  # O2 uptake
        [-1.2e-3, -3.6e-3, -6e-4, -1.8e-3],        # glucose uptake
        [2.25e-8, 9e-8, 1.125e-8, 4.5e-8],         # H+ production
    ],
    "O_A": 0.02, "G_P": 0.5, "G_Q": 0.05, "H_P": 1.58e-4, "H_Q": 3.98e-4,
    "T": [3000, 4800, 1800, 600],                  # G1, S, G2, M  (17 h cycle, PAPER.md l.196/l.232 hint)
    "J": [300, 480, 180, 60],
    "alpha": [0.25, 0.12, 0.35, 0.50],
    "beta": [0.03, 0.015, 0.04, 0.06],
    "oer_m": 3.0, "oer_K": 0.004,
    "repair_period": 60, "repair_shift": 4,
    "lysis_steps": 14400,
    "N_ref": 0,
    "well_mixed_medium": 0,                        # 1: EMPTY sites held at the medium values (alternative reading of G2; NEXT-3)
}


def default_params(**overrides):
    p = copy.deepcopy(_DEFAULT)
    for k, v in overrides.items():
        if k not in p:
            raise KeyError(k)
        p[k] = copy.deepcopy(v)
    return p


def stress_params(**overrides):
    """Short cell cycle / fast lysis: many phase changes, divisions, conflicts and
    deaths inside a 50-step parity window.  Test input, not a model claim."""
    p = default_params(T=[30, 48, 18, 6], J=[10, 16, 6, 2], lysis_steps=40, repair_period=5)
    p.update(copy.deepcopy(overrides))
    return p


DOSE_ALPHABET = np.array([0.5, 1.0, 1.5, 2.0, 2.5])           # BASELINE configs[1], [4]
DELAY_ALPHABET = np.arange(1, 11) * 6.0                        # 6, 12, ..., 60 h


def protocols_alphabet(rng, batch, nfrac=10, dose_cap=None):
    """batch x nfrac protocols from the c2/c3/c5 alphabets; optional total-dose cap by rejection."""
    dose = np.zeros((batch, nfrac))
    delay = np.zeros((batch, nfrac))
    for b in range(batch):
        while True:
            d = DOSE_ALPHABET[rng.integers(0, len(DOSE_ALPHABET), nfrac)]
            if dose_cap is None or d.sum() <= dose_cap + 1e-9:
                break
        dose[b] = d
        delay[b] = DELAY_ALPHABET[rng.integers(0, len(DELAY_ALPHABET), nfrac)]
    return dose, delay, np.full(batch, nfrac, np.int32)


def protocols_hypofractionated(rng, batch, max_frac=8, dose_cap=30.0):
    """c4: 3-8 fractions, dose 2.0..6.0 on a 0.5 grid, delay 12..96 h on a 6 h grid, total <= cap."""
    dose = np.zeros((batch, max_frac))
    delay = np.zeros((batch, max_frac))
    nfrac = np.zeros(batch, np.int32)
    for b in range(batch):
        while True:
            k = int(3 + rng.integers(0, 6))
            d = 2.0 + 0.5 * rng.integers(0, 9, k)
            if d.sum() <= dose_cap + 1e-9:
                break
        dose[b, :k] = d
        delay[b, :k] = 12.0 + 6.0 * rng.integers(0, 15, k)
        nfrac[b] = k
    return dose, delay, nfrac


# BMII of the paper and the single 20 Gy shot: named test protocols
PROTOCOL_BMI = ([1.25] * 8, [0, 6, 18, 6, 18, 6, 18, 6])
PROTOCOL_BMII = ([2.0] * 5, [0, 24, 24, 24, 24])
PROTOCOL_SINGLE20 = ([20.0], [0])


def config(k):
    """Recipe for BASELINE.json configs[k-1] (k = 1..5).  Returns a dict of plain data."""
    seed = MASTER_SEED + k
    rng = np.random.default_rng(seed)
    if k == 1:
        return dict(name="c1", batch=1, dims=(32, 32, 32), rng_seed=seed, sim_id_base=0,
                    init=dict(kind="cluster7", center=(16, 16, 16), radius=0.0, shared_init=False),
                    warmup_h=0.0, t0_h=0.0, horizon_h=48.0,
                    dose=np.array([[2.0]]), delay=np.array([[24.0]]), nfrac=np.array([1], np.int32))
    if k == 2:
        dose, delay, nfrac = protocols_alphabet(rng, 64)
        return dict(name="c2", batch=64, dims=(64, 64, 64), rng_seed=seed, sim_id_base=0,
                    init=dict(kind="ball", center=(32, 32, 32), radius=9.0, shared_init=True),
                    warmup_h=6.0, t0_h=6.0, horizon_h=720.0, dose=dose, delay=delay, nfrac=nfrac)
    if k == 3:
        dose, delay, nfrac = protocols_alphabet(rng, 512, dose_cap=20.0)
        return dict(name="c3", batch=512, dims=(96, 96, 96), rng_seed=seed, sim_id_base=0,
                    init=dict(kind="single", center=(48, 48, 48), radius=0.0, shared_init=True),
                    pregrow_diameter=64, warmup_h=0.0, t0_h=None, horizon_h=720.0,
                    dose=dose, delay=delay, nfrac=nfrac)
    if k == 4:
        dose, delay, nfrac = protocols_hypofractionated(rng, 1024)
        return dict(name="c4", batch=1024, dims=(80, 80, 80), rng_seed=seed, sim_id_base=0,
                    init=dict(kind="ball", center=(40, 40, 40), radius=9.0, shared_init=True),
                    warmup_h=6.0, t0_h=6.0, horizon_h=960.0, dose=dose, delay=delay, nfrac=nfrac)
    if k == 5:
        dose, delay, nfrac = protocols_alphabet(rng, 4096)
        return dict(name="c5", population=4096, seeds_per_protocol=4, batch=16384, dims=(64, 64, 64),
                    rng_seed=seed, sim_id_base=0,
                    init=dict(kind="ball", center=(32, 32, 32), radius=9.0, shared_init=True),
                    warmup_h=6.0, t0_h=6.0, horizon_h=720.0, dose=dose, delay=delay, nfrac=nfrac)
    raise ValueError("config index must be 1..5")


def reduced_c2():
    """Reduced BASELINE configs[1] job for long-horizon statistical parity (SURVEY 8(c) protocol (3)): what the fp64 oracle
    can afford on the host cores.  32^3 lattice, shared BALL r = 4 (257 cells), 6 h warm-up, 8 protocols of 4 fractions
    (configs[1] dose alphabet, delays 6..24 h so that the treatment fits the 5-day horizon), 30 seeds each."""
    seed = MASTER_SEED + 12
    rng = np.random.default_rng(seed)
    npro, nfr = 8, 4
    dose = DOSE_ALPHABET[rng.integers(0, len(DOSE_ALPHABET), (npro, nfr))]
    delay = 6.0 * (1 + rng.integers(0, 4, (npro, nfr)))
    return dict(name="c2-reduced", population=npro, seeds_per_protocol=30, batch=npro * 30, dims=(32, 32, 32), rng_seed=seed,
                sim_id_base=0, init=dict(kind="ball", center=(16, 16, 16), radius=4.0, shared_init=True),
                warmup_h=6.0, t0_h=6.0, horizon_h=120.0, dose=dose, delay=delay, nfrac=np.full(npro, nfr, np.int32))


def paper_geometry():
    """NEXT-3: the workload in the PAPER's own shape rather than BASELINE's.  The paper's lattice is
    quasi-3-D with at most 1 500 occupiable sites, its tumours are grown for 10 days from 200 cells on
    10 sites and kept as a library of 10 (l.244), a protocol is scored on every library tumour several times (l.282) over a
    5-day treatment plus 5 days of regrowth (l.274), and fitness is 1500 - n (Eq. 1).  Here: a 40 x 40 x 3 lattice -- ONE
    interior plane of 38 x 38 = 1 444 sites between two planes of medium, so that every site touches the replenished
    medium (l.244) -- N_ref = 1500, a 9-site seed (BALL r = 1.5 in the plane), 10 tumours that differ by their simulation
    id, 240 h of growth, 240 h of evaluation, BMI and BMII of the paper (l.49) plus an untreated control, 8 seeds per
    tumour (80 samples per protocol, l.282); run with `well_mixed_medium = 1` (EMPTY sites are medium, l.244).  Not
    reproduced: ~20 cells per site (this build keeps one cell per site, G1) and the paper's calibrated
    parameters (it prints none)."""
    seed = MASTER_SEED + 30
    names = ["untreated", "BMI", "BMII"]
    F = 8
    dose, delay, nfrac = np.zeros((3, F)), np.zeros((3, F)), np.zeros(3, np.int32)
    for r, (d, t) in enumerate((([], []), PROTOCOL_BMI, PROTOCOL_BMII)):
        dose[r, :len(d)], delay[r, :len(d)], nfrac[r] = d, t, len(d)
    return dict(name="paper-geometry", dims=(40, 40, 3), rng_seed=seed, n_ref=1500, n_tumours=10, seeds_per_tumour=8,
                init=dict(kind="ball", center=(20, 20, 1), radius=1.5, shared_init=False),
                grow_h=240.0, horizon_h=240.0, protocol_names=names, dose=dose, delay=delay, nfrac=nfrac)


def robustness_sweep(base_dose, base_delay, shifts_h=(-1.0, -0.5, 0.5, 1.0), step_h=0.5):
    """NEXT-4 workload (how sensitive is a good protocol to delivery errors?): every variant of one
    protocol in which a single fraction is dropped, or delivered `shift` hours early / late (the following fraction
    keeps its absolute time).  Returns (dose, delay, nfrac, labels); row 0 is the unperturbed protocol.  Delays stay on
    the `step_h` grid and non-negative; variants that would leave it are skipped."""
    base_dose = np.asarray(base_dose, dtype=np.float64)
    base_delay = np.asarray(base_delay, dtype=np.float64)
    k = len(base_dose)
    rows, labels = [(base_dose.copy(), base_delay.copy(), k)], ["base"]
    for j in range(k):                                              # drop fraction j: its delay is added to the next one
        d = np.delete(base_dose, j)
        t = np.delete(base_delay, j)
        if j < k - 1:
            t[j] += base_delay[j]
        rows.append((np.append(d, 0.0), np.append(t, 0.0), k - 1))
        labels.append("drop%d" % j)
    for j in range(k):
        for s in shifts_h:
            t = base_delay.copy()
            t[j] += s
            if j < k - 1:
                t[j + 1] -= s
            if t.min() < 0 or abs(s / step_h - round(s / step_h)) > 1e-9:
                continue
            rows.append((base_dose.copy(), t, k))
            labels.append("shift%d%+.1fh" % (j, s))
    dose = np.stack([r[0] for r in rows])
    delay = np.stack([r[1] for r in rows])
    nfrac = np.array([r[2] for r in rows], np.int32)
    return dose, delay, nfrac, labels
