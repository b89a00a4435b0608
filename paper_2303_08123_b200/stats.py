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


def _kolmogorov_sf(lam):
    """Q_KS(lambda) = 2 * sum_{k>=1} (-1)^(k-1) exp(-2 k^2 lambda^2); the alternating series does not converge for small
    lambda (it is 1 there to every digit), so identical samples (D = 0) get p = 1, not the series' 0."""
    if lam < 0.3:
        return 1.0
    p = 2.0 * sum((-1) ** (k - 1) * math.exp(-2.0 * (k * lam) ** 2) for k in range(1, 101))
    return float(min(1.0, max(0.0, p)))


def ks_2samp(a, b):
    """Two-sample Kolmogorov-Smirnov statistic D and its asymptotic p-value."""
    a, b = np.sort(np.asarray(a, np.float64)), np.sort(np.asarray(b, np.float64))
    allv = np.concatenate([a, b])
    cdfa = np.searchsorted(a, allv, side="right") / len(a)
    cdfb = np.searchsorted(b, allv, side="right") / len(b)
    d = float(np.abs(cdfa - cdfb).max())
    en = math.sqrt(len(a) * len(b) / (len(a) + len(b)))
    lam = (en + 0.12 + 0.11 / en) * d
    return d, _kolmogorov_sf(lam)


def same_distribution(a, b, alpha=0.01):
    """The acceptance rule used for long horizons, where near-threshold fp32 choices cascade and element-wise parity is
    not expected: neither the t-test nor KS rejects at level alpha."""
    _, _, pt = welch_t(a, b)
    _, pk = ks_2samp(a, b)
    return (pt is None or pt >= alpha) and pk >= alpha


def normal_cdf(x):
    return 0.5 * (1.0 + np.vectorize(math.erf)(np.asarray(x, np.float64) / math.sqrt(2.0)))


def ks_normality(a, discrete=False):
    """One-sample Kolmogorov-Smirnov test of `a` against the normal distribution with the sample's own mean and sd
    (PAPER.md l.69 and Fig. 3C/D, l.357: "KS-test for the normality of the GPU evaluations"; l.252: the final count over
    seeds is close to normal).  Returns (D, asymptotic p).  The parameters are estimated from the sample, as in the
    paper's figure, so p is conservative (Lilliefors); it is used as a sanity threshold, not as an exact level."""
    a = np.sort(np.asarray(a, np.float64))
    n = len(a)
    sd = a.std(ddof=1)
    if sd == 0.0:
        return 1.0, 0.0
    if discrete:
        # integer counts with a small sd: compare with the normal distribution binned the same way (continuity correction),
        # P(X <= k) against Phi((k + 1/2 - mean) / sd), otherwise the steps of the empirical CDF alone exceed any KS bound
        vals = np.unique(a)
        ecdf = np.searchsorted(a, vals, side="right") / n
        d = float(np.abs(ecdf - normal_cdf((vals + 0.5 - a.mean()) / sd)).max())
    else:
        cdf = normal_cdf((a - a.mean()) / sd)
        d = float(max((np.arange(1, n + 1) / n - cdf).max(), (cdf - np.arange(0, n) / n).max()))
    en = math.sqrt(n)
    lam = (en + 0.12 + 0.11 / en) * d
    return d, _kolmogorov_sf(lam)


def mean_ci95(a):
    """mean and half-width of its 95 % confidence interval over replicates (Fig. 3A)"""
    a = np.asarray(a, np.float64)
    n = len(a)
    if n < 2:
        return float(a.mean()), float("inf")
    try:
        from scipy import stats as st
        tq = float(st.t.ppf(0.975, n - 1))
    except ImportError:
        tq = 1.96 + 2.4 / max(1, n - 1)
    return float(a.mean()), tq * float(a.std(ddof=1)) / math.sqrt(n)


def compare_implementations(x, y):
    """The paper's fidelity check between two implementations (Fig. 3A-B): `x`, `y` are
    [protocols][replicates] final counts (or fitness).  Per protocol: mean and 95 % half-width of each, two-sided
    Welch t-test p-value, two-sample KS p-value.  Returns a dict of arrays."""
    x, y = [np.asarray(r, np.float64) for r in x], [np.asarray(r, np.float64) for r in y]
    assert len(x) == len(y)
    out = {k: [] for k in ("mean_x", "ci_x", "mean_y", "ci_y", "p_t", "p_ks")}
    for a, b in zip(x, y):
        ma, ca = mean_ci95(a)
        mb, cb = mean_ci95(b)
        out["mean_x"].append(ma); out["ci_x"].append(ca); out["mean_y"].append(mb); out["ci_y"].append(cb)
        out["p_t"].append(welch_t(a, b)[2]); out["p_ks"].append(ks_2samp(a, b)[1])
    return {k: np.array(v, np.float64) for k, v in out.items()}


def pvalues_not_piled_up(p, level=0.05, slack=3.0):
    """Under the null hypothesis p-values are uniform: about `level` of them fall below `level`.  True unless the
    fraction below `level` exceeds `level` by more than `slack` binomial standard deviations (and at least 2 do)."""
    p = np.asarray(p, np.float64)
    n = len(p)
    k = int((p < level).sum())
    return k <= max(1.0, n * level + slack * math.sqrt(n * level * (1.0 - level)))
