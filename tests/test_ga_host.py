"""Host GA operators (no GPU, no oracle): elitism, tournament, mutation stay on the alphabets and are reproducible."""
import numpy as np

from paper_2303_08123_b200 import ga, workloads as w


def _pop(n=40, seed=3):
    rng = np.random.default_rng(seed)
    return w.protocols_alphabet(rng, n)


def test_elites_are_copied_and_children_stay_on_the_alphabets():
    dose, delay, nfrac = _pop()
    fit = np.random.default_rng(1).normal(size=len(nfrac))
    nd, nt, nf = ga.next_generation(np.random.default_rng(7), dose, delay, nfrac, fit)
    order = np.argsort(-fit, kind="stable")
    assert np.array_equal(nd[:4], dose[order[:4]]) and np.array_equal(nt[:4], delay[order[:4]])      # 10 % of 40 [P l.272]
    assert np.isin(nd, w.DOSE_ALPHABET).all() and np.isin(nt, w.DELAY_ALPHABET).all()
    assert np.array_equal(nf, nfrac)
    # every child differs from some member of the old population in at most one gene [P l.274]
    for c in range(4, len(nf)):
        diffs = (nd[c][None, :] != dose).sum(1) + (nt[c][None, :] != delay).sum(1)
        assert diffs.min() <= 1


def test_selection_prefers_fitter_parents_and_is_reproducible():
    dose, delay, nfrac = _pop(200)
    fit = np.arange(200, dtype=float)                      # protocol i has fitness i
    a = ga.next_generation(np.random.default_rng(11), dose, delay, nfrac, fit)
    b = ga.next_generation(np.random.default_rng(11), dose, delay, nfrac, fit)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    # binary tournament: the expected rank of a winner is 2/3 of the way up; check that children resemble the upper half
    nd, nt, _ = a
    parent = [int(np.argmin((nd[c][None, :] != dose).sum(1) + (nt[c][None, :] != delay).sum(1))) for c in range(20, 200)]
    assert np.mean(parent) > 115


def test_robustness_sweep_keeps_absolute_times_of_untouched_fractions():
    dose, delay = w.PROTOCOL_BMII
    d, t, nf, labels = w.robustness_sweep(dose, delay)
    base_times = np.cumsum(delay)
    assert labels[0] == "base" and nf[0] == 5 and len(labels) == len(nf) == len(d)
    for row, lab in enumerate(labels):
        times = np.cumsum(t[row][:nf[row]])
        assert (t[row][:nf[row]] >= 0).all()
        if lab.startswith("drop"):
            j = int(lab[4:])
            assert np.allclose(times, np.delete(base_times, j)) and np.allclose(d[row][:nf[row]], np.delete(dose, j))
        elif lab.startswith("shift"):
            j = int(lab[5])
            diff = times - base_times
            assert abs(diff[j]) > 0 and np.allclose(np.delete(diff, j), 0.0)
    assert sum(l.startswith("drop") for l in labels) == 5 and sum(l.startswith("shift") for l in labels) >= 12
