"""Host side of the search loop around the hot path (BASELINE configs[4] and SURVEY NEXT-1).

The paper's GA [P l.255-274, Fig. 4 l.361]: a generation is 40 protocols; each is scored by the mean fitness over
several stochastic simulations [P l.282]; the best 10 % (4) are copied unchanged, 40 % (16) are chosen as parents by
one of three selection operators (roulette, simple, tournament), and 36 children are formed from the parents by one
of three crossovers (single-point, two-point, uniform) followed by one of four mutations (swap, split, dose time,
dose value) [P l.272-274].  A protocol is a sparse vector of 240 dose values on a 30-minute grid over 120 h
[P l.262, l.268]; constraints: total dose <= 10 Gy, single dose 0.25 Gy .. d_max in 0.25 Gy steps, a minimum
interval between fractions (6 h in the dose search) [P l.264, l.61].

The paper names the operators and prints no pseudo-code for them; each function below states the reading it takes.
Everything here is host code: the simulations run in libca_b200 through `binding.CaBatch`.
"""
import numpy as np

from . import sharding
from . import workloads as w

N_SLOTS = 240            # 120 h on a 30-minute grid [P l.262, l.268]
SLOT_H = 0.5
DOSE_STEP = 0.25         # [P l.264]

SELECTIONS = ("roulette", "simple", "tournament")
CROSSOVERS = ("single_point", "two_point", "uniform")
MUTATIONS = ("swap", "split", "dose_time", "dose_value")


# ------------------------------------------------------------------ evaluation (the hot path's caller) --
def evaluate_population(batch_ctx, snapshot, dose, delay, nfrac, seeds_per_protocol, rng_seed, t0_h, t_end_h, dist=None):
    """Mean fitness per protocol over `seeds_per_protocol` simulations each, streamed through one CaBatch per rank.

    Simulation (protocol p, seed s) has the GLOBAL id p * seeds_per_protocol + s (same Philox key, different id =>
    different stream), so the result does not depend on how the population is cut into batches or over ranks.  Every
    batch starts from the same saved tumour (`snapshot`, a dict as returned by CaBatch.get_state).
    With an initialised `torch.distributed` module as `dist`, rank r evaluates the contiguous range of global ids
    `sharding.shard_range(total, world, r)` on its own context and every rank receives all fitness values (one
    all_gather of `total` floats); there is no other communication."""
    npro = len(nfrac)
    total = npro * seeds_per_protocol
    world, rank = 1, 0
    if dist is not None and dist.is_initialized():
        world, rank = dist.get_world_size(), dist.get_rank()
    lo, count = sharding.shard_range(total, world, rank)
    B = batch_ctx.batch
    local = np.zeros(count, np.float32)
    dose, delay, nfrac = np.asarray(dose), np.asarray(delay), np.asarray(nfrac)
    F = dose.shape[1]
    for first in range(lo, lo + count, B):
        n = min(B, lo + count - first)
        ids = first + np.arange(B)
        ids[n:] = first                                    # pad the last batch with copies (their results are dropped)
        pro = ids // seeds_per_protocol
        batch_ctx.set_state(0, B, state=snapshot["state"], clock=snapshot["clock"], damage=snapshot["damage"],
                            o2=snapshot["o2"], glc=snapshot["glc"], h=snapshot["h"], step=snapshot["step"])
        batch_ctx.set_rng(rng_seed, first)
        batch_ctx.set_protocols(dose[pro].reshape(B, F), delay[pro].reshape(B, F), nfrac[pro], t0_h=t0_h)
        batch_ctx.run(t_end_h)
        local[first - lo:first - lo + n] = batch_ctx.fitness()[:n]
    fit = sharding.gather_fitness(local, total, dist)
    return fit.reshape(npro, seeds_per_protocol).mean(axis=1), fit


def evaluate_on_library(batch_ctx, library, dose, delay, nfrac, seeds_per_tumour, rng_seed, t_end_h, sim_id_base=0):
    """The paper's fitness methodology: every protocol is run on every tumour of the library
    `seeds_per_tumour` times; its fitness is the mean over all those evaluations.  ONE batch holds protocols x tumours x
    seeds simulations, simulation (p, j, s) at index (p * T + j) * S + s with that global id (plus sim_id_base); tumour j's
    snapshot is loaded into its index ranges with ca_set_state.  `t_end_h` counts from the snapshots' own time.
    Returns (mean fitness per protocol, fitness[p][j][s])."""
    npro, T, S = len(nfrac), len(library), int(seeds_per_tumour)
    assert batch_ctx.batch == npro * T * S, (batch_ctx.batch, npro, T, S)
    t0_h = None
    for p in range(npro):
        for j, snap in enumerate(library):
            batch_ctx.set_state((p * T + j) * S, S, state=snap["state"], clock=snap["clock"], damage=snap["damage"],
                                o2=snap["o2"], glc=snap["glc"], h=snap["h"], step=snap["step"])
            t0_h = snap["step"]
    batch_ctx.set_rng(rng_seed, sim_id_base)
    sph = batch_ctx.params.steps_per_hour
    pro = np.arange(batch_ctx.batch) // (T * S)
    batch_ctx.set_protocols(np.asarray(dose)[pro], np.asarray(delay)[pro], np.asarray(nfrac)[pro], t0_h=t0_h / sph)
    batch_ctx.run(t0_h / sph + t_end_h)
    fit = batch_ctx.fitness().reshape(npro, T, S)
    return fit.reshape(npro, -1).mean(axis=1), fit


# ------------------------------------------------------------------ genotype <-> (dose, delay) list --
def genotype_to_list(g, max_frac=None):
    """240-slot dose vector -> (dose[k], delay[k]) with delay = wait since the previous fraction, the first one from the
    start of treatment [P l.49].  Slot i is t = 0.5 * i h, 0-based (G21)."""
    g = np.asarray(g, dtype=np.float64)
    idx = np.flatnonzero(g > 0)
    t = idx * SLOT_H
    delay = np.diff(np.concatenate([[0.0], t]))
    dose = g[idx]
    if max_frac is not None:
        assert len(idx) <= max_frac, (len(idx), max_frac)
    return dose, delay


def list_to_genotype(dose, delay, nfrac=None, n_slots=N_SLOTS):
    """Inverse of genotype_to_list.  Fractions that share a slot add up; times must lie on the 30-minute grid inside the window."""
    dose, delay = np.asarray(dose, np.float64), np.asarray(delay, np.float64)
    k = len(dose) if nfrac is None else int(nfrac)
    g = np.zeros(n_slots)
    t = 0.0
    for j in range(k):
        t += delay[j]
        i = t / SLOT_H
        if abs(i - round(i)) > 1e-9 or not 0 <= round(i) < n_slots:
            raise ValueError("fraction %d at t = %g h is not on the %g h grid inside %g h" % (j, t, SLOT_H, n_slots * SLOT_H))
        g[int(round(i))] += dose[j]
    return g


def population_to_table(G, max_frac):
    """genotypes [n][240] -> the (dose, delay, nfrac) table ca_set_protocols takes."""
    n = len(G)
    dose, delay, nfrac = np.zeros((n, max_frac)), np.zeros((n, max_frac)), np.zeros(n, np.int32)
    for r in range(n):
        d, t = genotype_to_list(G[r], max_frac)
        dose[r, :len(d)], delay[r, :len(d)], nfrac[r] = d, t, len(d)
    return dose, delay, nfrac


# ------------------------------------------------------------------ constraints --
def repair(rng, g, dose_cap=10.0, d_max=2.5, min_interval_h=6.0, d_min=DOSE_STEP):
    """Bring a genotype back into the feasible set [P l.264, l.61]: doses on the 0.25 Gy grid in [d_min, d_max]; fractions
    closer than the minimum interval are merged into the earlier one (the dose is kept, so the operator never loses
    dose silently; the sum is then clipped to d_max); while the total exceeds the cap, 0.25 Gy is taken from a random
    fraction (a fraction that reaches 0 disappears).  Returns a new vector."""
    g = np.round(np.asarray(g, np.float64) / DOSE_STEP) * DOSE_STEP
    g[g < 0] = 0.0
    gap = int(round(min_interval_h / SLOT_H))
    last = None
    for i in range(len(g)):
        if g[i] <= 0:
            continue
        if last is not None and i - last < gap:
            g[last] += g[i]
            g[i] = 0.0
        else:
            last = i
    nz = g > 0
    g[nz] = np.clip(g[nz], d_min, d_max)
    while g.sum() > dose_cap + 1e-9:
        idx = np.flatnonzero(g > 0)
        i = idx[rng.integers(0, len(idx))]
        g[i] -= DOSE_STEP
        if g[i] < d_min - 1e-9:
            g[i] = 0.0
    return g


def feasible(g, dose_cap=10.0, d_max=2.5, min_interval_h=6.0, d_min=DOSE_STEP):
    g = np.asarray(g, np.float64)
    idx = np.flatnonzero(g > 0)
    on_grid = np.allclose(g / DOSE_STEP, np.round(g / DOSE_STEP))
    gaps_ok = len(idx) < 2 or np.diff(idx).min() * SLOT_H >= min_interval_h - 1e-9
    return bool(on_grid and gaps_ok and g.sum() <= dose_cap + 1e-9 and (len(idx) == 0 or (g[idx].min() >= d_min - 1e-9 and g[idx].max() <= d_max + 1e-9)))


def random_genotype(rng, dose_cap=10.0, d_max=2.5, min_interval_h=6.0, n_slots=N_SLOTS):
    """A feasible random protocol: fractions at random slots at least the minimum interval apart, doses on the grid."""
    gap = int(round(min_interval_h / SLOT_H))
    kmax = (n_slots - 1) // gap + 1
    k = int(rng.integers(1, kmax + 1))
    g = np.zeros(n_slots)
    slots = np.sort(rng.choice(n_slots - (k - 1) * (gap - 1), size=k, replace=False)) + np.arange(k) * (gap - 1)   # gaps >= `gap`
    g[slots] = DOSE_STEP * rng.integers(1, int(round(d_max / DOSE_STEP)) + 1, k)
    return repair(rng, g, dose_cap, d_max, min_interval_h)


# ------------------------------------------------------------------ selection [P l.272, Fig. 4] --
def select_simple(rng, fitness, k):
    """"simple sort and take the top few"; ties -> lower index"""
    return np.argsort(-np.asarray(fitness, np.float64), kind="stable")[:k]


def select_roulette(rng, fitness, k):
    """"proportional chance by fitness": k draws with replacement, probability ~ fitness shifted to be positive
    (Eq. 1 fitness is positive by construction; the shift only matters for other score scales)."""
    f = np.asarray(fitness, np.float64)
    wgt = f - min(0.0, f.min())
    if wgt.sum() <= 0:
        wgt = np.ones_like(f)
    return rng.choice(len(f), size=k, replace=True, p=wgt / wgt.sum())


def select_tournament(rng, fitness, k):
    """"pair-wise competition on fitness": k times, two distinct random members meet and the fitter one becomes a parent
    (ties -> lower index)."""
    f = np.asarray(fitness, np.float64)
    out = np.zeros(k, np.int64)
    for i in range(k):
        a, b = rng.choice(len(f), size=2, replace=False) if len(f) > 1 else (0, 0)
        out[i] = a if (f[a], -a) >= (f[b], -b) else b
    return out


_SELECT = {"simple": select_simple, "roulette": select_roulette, "tournament": select_tournament}


# ------------------------------------------------------------------ crossover [P l.274] --
def crossover(rng, a, b, kind):
    """One child from two parent genotypes: single-point (head of a, tail of b), two-point (a with a middle segment of
    b), uniform (every slot from a or b with probability 1/2)."""
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    n = len(a)
    if kind == "single_point":
        c = int(rng.integers(1, n))
        return np.concatenate([a[:c], b[c:]])
    if kind == "two_point":
        c0, c1 = np.sort(rng.choice(np.arange(1, n), size=2, replace=False))
        return np.concatenate([a[:c0], b[c0:c1], a[c1:]])
    if kind == "uniform":
        return np.where(rng.integers(0, 2, n) == 0, a, b)
    raise ValueError(kind)


# ------------------------------------------------------------------ mutation [P l.274] --
def mutate(rng, g, kind, d_max=2.5):
    """swap: two fractions exchange their doses (a protocol with one fraction exchanges it with an empty slot, i.e. moves
    it); split: one fraction of >= 0.5 Gy is split into two parts on the 0.25 Gy grid, the second part going to a random
    empty slot; dose time: one fraction moves to a random empty slot; dose value: one fraction's dose is redrawn from
    {0.25, ..., d_max}.  An empty protocol gets one random fraction.  Constraints are restored by `repair` afterwards."""
    g = np.array(g, dtype=np.float64)
    idx = np.flatnonzero(g > 0)
    empty = np.flatnonzero(g <= 0)
    nlev = int(round(d_max / DOSE_STEP))
    if len(idx) == 0:
        g[rng.integers(0, len(g))] = DOSE_STEP * rng.integers(1, nlev + 1)
        return g
    if kind == "swap":
        if len(idx) >= 2:
            i, j = rng.choice(idx, size=2, replace=False)
        else:
            i, j = idx[0], empty[rng.integers(0, len(empty))]
        g[i], g[j] = g[j], g[i]
    elif kind == "split":
        big = idx[g[idx] >= 2 * DOSE_STEP - 1e-9]
        if len(big) and len(empty):
            i = big[rng.integers(0, len(big))]
            units = int(round(g[i] / DOSE_STEP))
            part = int(rng.integers(1, units))
            j = empty[rng.integers(0, len(empty))]
            g[i] = (units - part) * DOSE_STEP
            g[j] = part * DOSE_STEP
    elif kind == "dose_time":
        if len(empty):
            i = idx[rng.integers(0, len(idx))]
            j = empty[rng.integers(0, len(empty))]
            g[j], g[i] = g[i], 0.0
    elif kind == "dose_value":
        i = idx[rng.integers(0, len(idx))]
        g[i] = DOSE_STEP * rng.integers(1, nlev + 1)
    else:
        raise ValueError(kind)
    return g


# ------------------------------------------------------------------ one generation [P l.272-274, Fig. 4] --
def next_generation_genotypes(rng, G, fitness, selection="tournament", crossover_kind="uniform", mutation="dose_value",
                              elite_frac=0.1, parent_frac=0.4, dose_cap=10.0, d_max=2.5, min_interval_h=6.0):
    """Generation T -> T + 1: the best 10 % are copied unchanged (simple selection), 40 % become parents through
    `selection`, and the remaining children are formed from two random distinct parents by `crossover_kind`, then
    `mutation`, then constraint repair.  Higher fitness is better (Eq. 1)."""
    G = np.asarray(G, np.float64)
    n = len(G)
    n_elite = max(1, int(round(elite_frac * n)))
    n_par = max(2, int(round(parent_frac * n)))
    out = np.zeros_like(G)
    out[:n_elite] = G[select_simple(rng, fitness, n_elite)]
    parents = _SELECT[selection](rng, fitness, n_par)
    for c in range(n_elite, n):
        ia, ib = rng.choice(len(parents), size=2, replace=False)
        child = crossover(rng, G[parents[ia]], G[parents[ib]], crossover_kind)
        child = mutate(rng, child, mutation, d_max)
        out[c] = repair(rng, child, dose_cap, d_max, min_interval_h)
    return out


def next_generation(rng, dose, delay, nfrac, fitness, elite_frac=0.1, dose_alphabet=w.DOSE_ALPHABET, delay_alphabet=w.DELAY_ALPHABET):
    """BASELINE configs[4] form (fixed 10-fraction lists on the configs[1] alphabets): elitism + binary tournament + one
    mutation per child (dose value or dose time).  Higher fitness is better."""
    n = len(fitness)
    order = np.argsort(-np.asarray(fitness), kind="stable")
    n_elite = max(1, int(round(elite_frac * n)))
    nd, nt, nf = dose.copy(), delay.copy(), nfrac.copy()
    nd[:n_elite], nt[:n_elite], nf[:n_elite] = dose[order[:n_elite]], delay[order[:n_elite]], nfrac[order[:n_elite]]
    for c in range(n_elite, n):
        a, b = rng.integers(0, n, 2)
        win = a if (fitness[a], -a) >= (fitness[b], -b) else b          # ties: lower index, so the result is reproducible
        nd[c], nt[c], nf[c] = dose[win], delay[win], nfrac[win]
        j = int(rng.integers(0, max(1, nf[c])))
        if rng.integers(0, 2) == 0:
            nd[c, j] = dose_alphabet[rng.integers(0, len(dose_alphabet))]      # "dose value" mutation
        else:
            nt[c, j] = delay_alphabet[rng.integers(0, len(delay_alphabet))]    # "dose time" mutation
    return nd, nt, nf


def run_ga(batch_ctx, snapshot, dose, delay, nfrac, generations, seeds_per_protocol, rng_seed, t0_h, t_end_h, ga_seed=0, dist=None):
    """`generations` rounds of evaluate -> select/mutate on fixed-length lists (configs[4]).  With `dist`, the population is
    evaluated over all ranks; rank 0's next generation is broadcast so that every rank works on the same table.
    Returns the per-generation best and mean fitness and the final population."""
    rng = np.random.default_rng(ga_seed)
    history = []
    for g in range(generations):
        fit, _ = evaluate_population(batch_ctx, snapshot, dose, delay, nfrac, seeds_per_protocol, rng_seed, t0_h, t_end_h, dist=dist)
        history.append((float(fit.max()), float(fit.mean())))
        if g + 1 < generations:
            dose, delay, nfrac = next_generation(rng, dose, delay, nfrac, fit)
            dose, delay, nfrac = sharding.broadcast_protocols(dose, delay, nfrac, dist)
    return history, (dose, delay, nfrac), fit


def run_ga_genotypes(batch_ctx, snapshot, G, generations, seeds_per_protocol, rng_seed, t0_h, t_end_h, ga_seed=0, dist=None,
                     max_frac=20, **operators):
    """The paper's loop on 240-slot genotypes [P l.268-274]: evaluate, copy the elite, select, cross, mutate, repair."""
    rng = np.random.default_rng(ga_seed)
    history = []
    G = np.asarray(G, np.float64)
    for g in range(generations):
        dose, delay, nfrac = population_to_table(G, max_frac)
        fit, _ = evaluate_population(batch_ctx, snapshot, dose, delay, nfrac, seeds_per_protocol, rng_seed, t0_h, t_end_h, dist=dist)
        history.append((float(fit.max()), float(fit.mean())))
        if g + 1 < generations:
            G = next_generation_genotypes(rng, G, fit, **operators)
            if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
                obj = [G if dist.get_rank() == 0 else None]
                dist.broadcast_object_list(obj, src=0)
                G = obj[0]
    return history, G, fit
