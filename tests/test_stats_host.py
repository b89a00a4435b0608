"""Host statistics (no GPU): Eq. 2 against the values the paper prints, t-test / KS against scipy."""
import os

import numpy as np
from scipy import stats as st

from paper_2303_08123_b200 import stats

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_fitness_pairs.txt")


def test_eq2_reproduces_the_printed_percentages():
    n = 0
    for line in open(GOLDEN):
        line = line.split("#")[0].split()
        if len(line) < 5:
            continue
        f_i, f_ref, printed = float(line[1]), float(line[3]), float(line[4])
        n_i, n_ref = stats.occupied_from_fitness(f_i, 1500), stats.occupied_from_fitness(f_ref, 1500)
        assert abs(100.0 * stats.its(n_i, n_ref) - printed) < 0.051, line
        n += 1
    assert n >= 7


def test_welch_and_ks_match_scipy():
    rng = np.random.default_rng(2)
    for shift in (0.0, 0.4, 2.0):
        a, b = rng.normal(300.0, 40.0, 60), rng.normal(300.0 + 40.0 * shift, 55.0, 45)
        t, df, p = stats.welch_t(a, b)
        ref = st.ttest_ind(a, b, equal_var=False)
        assert abs(t - ref.statistic) < 1e-10 and abs(p - ref.pvalue) < 1e-10
        d, pk = stats.ks_2samp(a, b)
        refk = st.ks_2samp(a, b, method="asymp")
        assert abs(d - refk.statistic) < 1e-12
        assert abs(pk - refk.pvalue) < 0.02 + 0.2 * refk.pvalue                  # Stephens' small-sample correction vs scipy's asymptotic form
    same = rng.normal(0, 1, 200)
    assert stats.same_distribution(same[:100], same[100:])
    assert not stats.same_distribution(same[:100], same[100:] + 1.0)


def test_summarize_groups_seeds():
    f = np.arange(12.0)
    mean, sd = stats.summarize(f, 4)
    assert mean.tolist() == [1.5, 5.5, 9.5] and np.allclose(sd, np.std([0, 1, 2, 3], ddof=1))


def test_ks_normality_continuous_matches_scipy_and_discrete_handles_integer_counts():
    rng = np.random.default_rng(8)
    x = rng.normal(300.0, 40.0, 500)
    d, p = stats.ks_normality(x)
    ref = st.kstest((x - x.mean()) / x.std(ddof=1), "norm")
    assert abs(d - ref.statistic) < 1e-12 and abs(p - ref.pvalue) < 0.02
    assert stats.ks_normality(rng.exponential(1.0, 500))[1] < 1e-3            # clearly not normal
    k = np.round(rng.normal(36.0, 4.0, 2000))                                  # integer counts, sd of a few units
    assert stats.ks_normality(k)[0] > 0.04                                     # the plain statistic sees the steps ...
    assert stats.ks_normality(k, discrete=True)[0] < 0.03                      # ... the binned one does not
    assert stats.ks_normality(np.round(rng.exponential(6.0, 2000)), discrete=True)[1] < 1e-3


def test_compare_implementations_and_pvalue_pile_up():
    rng = np.random.default_rng(9)
    x = [rng.normal(300 + 5 * k, 30, 40) for k in range(60)]
    y = [rng.normal(300 + 5 * k, 30, 48) for k in range(60)]                   # same distributions: Fig. 3B of the paper
    cmp = stats.compare_implementations(x, y)
    assert stats.pvalues_not_piled_up(cmp["p_t"]) and (cmp["p_t"] < 0.05).mean() < 0.15
    assert np.all(np.abs(cmp["mean_x"] - cmp["mean_y"]) < 4 * (cmp["ci_x"] + cmp["ci_y"]))
    z = [rng.normal(330 + 5 * k, 30, 48) for k in range(60)]                   # shifted by one sd: must be noticed
    assert not stats.pvalues_not_piled_up(stats.compare_implementations(x, z)["p_t"])
    m, ci = stats.mean_ci95(np.arange(10.0))
    assert m == 4.5 and abs(ci - st.t.ppf(0.975, 9) * np.arange(10.0).std(ddof=1) / np.sqrt(10)) < 1e-12


def test_identical_samples_are_the_same_distribution():
    """D = 0 must give p = 1 (the alternating Kolmogorov series is 0 there if summed naively): a GPU run that reproduces
    the oracle's counts exactly is the best possible agreement, not a rejection."""
    x = np.array([1828.0, 1683.0, 1808.0, 1733.0, 1658.0])
    assert stats.ks_2samp(x, x.copy()) == (0.0, 1.0)
    assert stats.welch_t(x, x.copy())[2] == 1.0
    assert stats.same_distribution(x, x.copy())
    rng = np.random.default_rng(3)
    a, b = rng.normal(0, 1, 400), rng.normal(0.02, 1, 400)
    ref = st.ks_2samp(a, b)
    d, p = stats.ks_2samp(a, b)
    assert abs(d - ref.statistic) < 1e-12 and abs(p - ref.pvalue) < 0.05
