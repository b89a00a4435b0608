"""Fitness methodology around the hot path (NEXT-2, host only): per-protocol statistics over seeds, the paper's
"improvement in treatment success" (Eq. 2) and the comparisons the paper uses to validate one
implementation against another (two-sided t-test and Kolmogorov-Smirnov on final counts, PAPER.md l.69, l.357;
normality of the final count over seeds).  Plain numpy; scipy is used when present for p-values."""
import math

import numpy as np


def occupied_from_fitness(fitness, n_ref):
    """Eq. 1 inverted: n = N_ref - f  (the paper's N_ref is 1500)."""
    return float(n_ref) - np.asarray(fitness, dtype=np.float64)


def its(n_i, n_ref):
    """Eq. 2: ITS = (n_ref - n_i) / n_ref, the relative reduction of the surviving tumour against a reference protocol."""
    return (float(n_ref) - float(n_i)) / float(n_ref)


def summarize(fitness_per_sim, seeds_per_protocol):
    """[protocols * seeds] -> per-protocol mean and sample sd over seeds (fitness = mean over runs)."""
    f = np.asarray(fitness_per_sim, dtype=np.float64).reshape(-1, seeds_per_protocol)
    sd = f.std(axis=1, ddof=1) if seeds_per_protocol > 1 else np.zeros(len(f))
    return f.mean(axis=1), sd


def welch_t(a, b):
    """Two-sided Welch t-test: (t, degrees of freedom, p).  p is None without scipy."""
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    va, vb = a.var(ddof=1) / len(a), b.var(ddof=1) / len(b)
    if va + vb == 0.0:
        return 0.0, float(len(a) + len(b) - 2), 1.0 if a.mean() == b.mean() else 0.0
    t = (a.mean() - b.mean()) / math.sqrt(va + vb)
    df = (va + vb) ** 2 / (va ** 2 / (len(a) - 1) + vb ** 2 / (len(b) - 1))
    try:
        from scipy import stats as st
        p = float(2.0 * st.t.sf(abs(t), df))
    except ImportError:
        p = None
    return float(t), float(df), p


def ks_2samp(a, b):
    """Two-sample Kolmogorov-Smirnov statistic D and its asymptotic p-value."""
    a, b = np.sort(np.asarray(a, np.float64)), np.sort(np.asarray(b, np.float64))
    allv = np.concatenate([a, b])
    cdfa = np.searchsorted(a, allv, side="right") / len(a)
    cdfb = np.searchsorted(b, allv, side="right") / len(b)
    d = float(np.abs(cdfa - cdfb).max())
    en = math.sqrt(len(a) * len(b) / (len(a) + len(b)))
    lam = (en + 0.12 + 0.11 / en) * d
    p = 2.0 * sum((-1) ** (k - 1) * math.exp(-2.0 * (k * lam) ** 2) for k in range(1, 101))
    return d, float(min(1.0, max(0.0, p)))


def same_distribution(a, b, alpha=0.01):
    """The acceptance rule used for long horizons, where near-threshold fp32 choices cascade and element-wise parity is
    not expected: neither the t-test nor KS rejects at level alpha."""
    _, _, pt = welch_t(a, b)
    _, pk = ks_2samp(a, b)
    return (pt is None or pt >= alpha) and pk >= alpha
