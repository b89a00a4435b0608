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
