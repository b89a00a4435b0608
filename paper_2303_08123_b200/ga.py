"""Host side of the search loop around the hot path (BASELINE configs[4]).

The paper's GA [P l.262-274, l.361] keeps a population of protocols, scores each by the mean fitness over several
stochastic simulations [P l.282], copies the best 10 % unchanged [P l.272], fills the rest by pair-wise
competition on fitness [P l.361] and applies one mutation per child, either to a dose value or to a dose time
[P l.274].  Only what the streaming evaluation of configs[4] needs is here (tournament + mutation on the
configs[1] alphabets); the paper's full operator set is NEXT-1.  Everything in this module is host code: the
simulations run in libca_b200 through `binding.CaBatch`.
"""
import numpy as np

from . import workloads as w


def evaluate_population(batch_ctx, snapshot, dose, delay, nfrac, seeds_per_protocol, rng_seed, t0_h, t_end_h):
    """Mean fitness per protocol over `seeds_per_protocol` simulations each, streamed through one CaBatch.

    Simulation (protocol p, seed s) has the GLOBAL id p * seeds_per_protocol + s (same Philox key, different id =>
    different stream), so the result does not depend on how the population is cut into batches.  Every batch starts
    from the same saved tumour (`snapshot`, a dict as returned by CaBatch.get_state)."""
    npro = len(nfrac)
    total = npro * seeds_per_protocol
    B = batch_ctx.batch
    fit = np.zeros(total, np.float32)
    F = dose.shape[1]
    for first in range(0, total, B):
        n = min(B, total - first)
        ids = first + np.arange(B)
        ids[n:] = first                                    # pad the last batch with copies (their results are dropped)
        pro = ids // seeds_per_protocol
        batch_ctx.set_state(0, B, state=snapshot["state"], clock=snapshot["clock"], damage=snapshot["damage"],
                            o2=snapshot["o2"], glc=snapshot["glc"], h=snapshot["h"], step=snapshot["step"])
        batch_ctx.set_rng(rng_seed, first)
        batch_ctx.set_protocols(dose[pro].reshape(B, F), delay[pro].reshape(B, F), nfrac[pro], t0_h=t0_h)
        batch_ctx.run(t_end_h)
        fit[first:first + n] = batch_ctx.fitness()[:n]
    return fit.reshape(npro, seeds_per_protocol).mean(axis=1), fit


def next_generation(rng, dose, delay, nfrac, fitness, elite_frac=0.1, dose_alphabet=w.DOSE_ALPHABET, delay_alphabet=w.DELAY_ALPHABET):
    """Elitism + binary tournament + one mutation per child (dose value or dose time), higher fitness is better."""
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


def run_ga(batch_ctx, snapshot, dose, delay, nfrac, generations, seeds_per_protocol, rng_seed, t0_h, t_end_h, ga_seed=0):
    """`generations` rounds of evaluate -> select/mutate.  Returns the per-generation best and mean fitness and the final population."""
    rng = np.random.default_rng(ga_seed)
    history = []
    for g in range(generations):
        fit, _ = evaluate_population(batch_ctx, snapshot, dose, delay, nfrac, seeds_per_protocol, rng_seed, t0_h, t_end_h)
        history.append((float(fit.max()), float(fit.mean())))
        if g + 1 < generations:
            dose, delay, nfrac = next_generation(rng, dose, delay, nfrac, fit)
    return history, (dose, delay, nfrac), fit
