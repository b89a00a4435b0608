"""Host logic of bench.py (no GPU): the protocol table the end-to-end arm re-uploads every step, and the slab / traffic helpers."""
import numpy as np

import bench
from paper_2303_08123_b200 import workloads as w


def test_remaining_table_keeps_indices_and_absolute_times():
    """Fractions already delivered become (0 Gy, 0 h) no-ops at t_now, later ones keep their list index (the irradiation draws
    are keyed by it) and their absolute fire time: the e2e arm must reproduce the device arm bit for bit."""
    rng = np.random.default_rng(4)
    dose, delay, nfrac = w.protocols_alphabet(rng, 16)
    nfrac = nfrac.copy(); nfrac[3] = 7
    t0 = 6.0
    T = t0 + np.cumsum(delay, axis=1)
    for t_now in (6.0, 6.1, 17.9, 18.0, 100.0, 1000.0):
        nd, nt = bench.remaining_table(dose, delay, nfrac, t0, t_now)
        T2 = t_now + np.cumsum(nt, axis=1)
        for b in range(16):
            for j in range(int(nfrac[b])):
                if T[b, j] < t_now - 1e-9:
                    assert nd[b, j] == 0.0 and nt[b, j] == 0.0                      # a no-op that fires "now"
                else:
                    assert nd[b, j] == dose[b, j] and abs(T2[b, j] - T[b, j]) < 1e-9
            assert (nt[b] >= 0).all()
            steps = nt[b, :nfrac[b]] * 600.0
            assert np.allclose(steps, np.round(steps), atol=1e-6)                   # still whole CA steps


def test_ncu_traffic_reads_the_committed_summaries():
    tot, src, batch = bench.ncu_traffic("r02_ncu_fused_c5*.txt")
    assert src.startswith("profiles/r02_ncu_fused") and batch == 2048
    alg = bench.B_ALG * batch * 64 ** 3
    assert 0.95 < tot / alg < 1.2                                                   # the fused kernel moves ~1.07 x the algorithmic bytes
    assert bench.ncu_traffic("no_such_file_*.txt") == (None, None, None)
