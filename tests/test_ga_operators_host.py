"""NEXT-1: the paper's GA operators on the 240-slot genotype (Fig. 4 l.361).  Host only."""
import numpy as np
import pytest

from paper_2303_08123_b200 import ga, workloads as w


def test_genotype_indexing_is_zero_based_half_hours():
    """G21: slot i <-> t = 0.5 * i h; BMI / BMII of the paper (l.49) round-trip through the 240-vector."""
    g = np.zeros(ga.N_SLOTS)
    g[4] = 1.25
    d, t = ga.genotype_to_list(g)
    assert d.tolist() == [1.25] and t.tolist() == [2.0]          # "four times 30 minutes" = 2 h  [P l.268]
    for dose, delay in (w.PROTOCOL_BMI, w.PROTOCOL_BMII):
        g = ga.list_to_genotype(dose, delay)
        assert g[0] == dose[0] and np.count_nonzero(g) == len(dose)
        d2, t2 = ga.genotype_to_list(g)
        assert np.allclose(d2, dose) and np.allclose(t2, delay)
        assert np.flatnonzero(g).tolist() == (np.cumsum(delay) * 2).astype(int).tolist()
    with pytest.raises(ValueError):
        ga.list_to_genotype([1.0], [0.25])                        # off the 30-minute grid
    with pytest.raises(ValueError):
        ga.list_to_genotype([1.0], [120.0])                       # outside the 120 h window


def test_population_to_table_matches_what_ca_set_protocols_takes():
    rng = np.random.default_rng(1)
    G = np.stack([ga.random_genotype(rng) for _ in range(40)])
    dose, delay, nfrac = ga.population_to_table(G, 20)
    for r in range(40):
        back = ga.list_to_genotype(dose[r], delay[r], nfrac[r])
        assert np.allclose(back, G[r])
        assert (delay[r, :nfrac[r]] * 600 % 300 == 0).all()       # whole 300-step units [P l.262]


def test_random_and_repaired_genotypes_are_feasible():
    rng = np.random.default_rng(2)
    for d_max in (1.25, 2.5, 4.5):
        for _ in range(100):
            g = ga.random_genotype(rng, d_max=d_max)
            assert ga.feasible(g, d_max=d_max)
    bad = np.zeros(ga.N_SLOTS)
    bad[[0, 3, 20, 21, 100]] = [3.0, 1.0, 0.6, 4.0, 5.0]
    fixed = ga.repair(rng, bad, dose_cap=10.0, d_max=2.5, min_interval_h=6.0)
    assert ga.feasible(fixed) and fixed.sum() <= 10.0
    assert fixed[3] == 0 and fixed[21] == 0                       # merged into the earlier neighbour
    ok = ga.random_genotype(rng)
    assert np.array_equal(ga.repair(rng, ok), ok)                 # feasible input is left alone


@pytest.mark.parametrize("kind", ga.CROSSOVERS)
def test_crossover_takes_every_slot_from_one_of_the_parents(kind):
    rng = np.random.default_rng(3)
    a, b = np.arange(1, 241, dtype=float), -np.arange(1, 241, dtype=float)
    for _ in range(50):
        c = ga.crossover(rng, a, b, kind)
        from_a = c > 0
        assert np.array_equal(np.abs(c), a)
        switches = int(np.count_nonzero(np.diff(from_a.astype(int))))
        if kind == "single_point":
            assert switches == 1 and from_a[0] and not from_a[-1]
        elif kind == "two_point":
            assert switches == 2 and from_a[0] and from_a[-1]
        else:
            assert 60 < from_a.sum() < 180


@pytest.mark.parametrize("kind", ga.MUTATIONS)
def test_mutations_do_what_their_names_say(kind):
    rng = np.random.default_rng(4)
    for _ in range(200):
        g = ga.random_genotype(rng)
        m = ga.mutate(rng, g, kind)
        i0, i1 = np.flatnonzero(g), np.flatnonzero(m)
        if kind == "swap":
            assert np.allclose(np.sort(g[i0]), np.sort(m[i1])) and np.isclose(g.sum(), m.sum())
            if len(i0) >= 2:
                assert np.array_equal(i0, i1)                     # times kept, doses exchanged
        elif kind == "split":
            assert np.isclose(g.sum(), m.sum()) and len(i1) in (len(i0), len(i0) + 1)
            if g[i0].max() >= 0.5:
                assert len(i1) == len(i0) + 1
        elif kind == "dose_time":
            assert len(i1) == len(i0) and np.allclose(np.sort(g[i0]), np.sort(m[i1])) and len(set(i0) ^ set(i1)) == 2
        else:
            assert np.array_equal(i0, i1) and (g != m).sum() <= 1 and m[i1].max() <= 2.5 and m[i1].min() >= 0.25
    empty = ga.mutate(rng, np.zeros(ga.N_SLOTS), kind)
    assert np.count_nonzero(empty) == 1


def test_selection_operators():
    rng = np.random.default_rng(5)
    fit = np.arange(40, dtype=float)
    assert ga.select_simple(rng, fit, 16).tolist() == list(range(39, 23, -1))
    tour = np.concatenate([ga.select_tournament(rng, fit, 16) for _ in range(200)])
    assert abs(tour.mean() - (2 * 39 / 3.0)) < 1.0                # E[max of two distinct of 0..39] = 26.33
    roul = np.concatenate([ga.select_roulette(rng, fit, 16) for _ in range(400)])
    assert abs(roul.mean() - (np.sum(fit * fit) / fit.sum())) < 0.6   # E = sum f^2 / sum f = 26.33
    assert (roul == 0).sum() == 0                                 # zero fitness, zero chance
    assert len(set(ga.select_roulette(rng, np.full(10, -3.0), 50))) > 5   # degenerate weights -> uniform


@pytest.mark.parametrize("selection", ga.SELECTIONS)
def test_one_generation_follows_fig4(selection):
    """40 protocols: 4 copied unchanged, 36 children from 16 parents, every child feasible [P l.272-274]."""
    rng = np.random.default_rng(6)
    G = np.stack([ga.random_genotype(rng) for _ in range(40)])
    fit = rng.normal(1000.0, 50.0, 40)
    for cx in ga.CROSSOVERS:
        for mu in ga.MUTATIONS:
            r1 = ga.next_generation_genotypes(np.random.default_rng(9), G, fit, selection, cx, mu)
            r2 = ga.next_generation_genotypes(np.random.default_rng(9), G, fit, selection, cx, mu)
            assert np.array_equal(r1, r2)
            assert np.array_equal(r1[:4], G[np.argsort(-fit, kind="stable")[:4]])
            assert all(ga.feasible(g) for g in r1)
            assert r1.shape == G.shape


def test_ga_improves_a_toy_fitness():
    """The loop as a whole climbs: fitness = -(distance of the total dose from 7 Gy) - 0.1 * number of fractions."""
    rng = np.random.default_rng(7)
    G = np.stack([ga.random_genotype(rng) for _ in range(40)])
    score = lambda P: np.array([-abs(g.sum() - 7.0) - 0.1 * np.count_nonzero(g) for g in P])
    first = score(G).max()
    for _ in range(30):
        G = ga.next_generation_genotypes(rng, G, score(G), "tournament", "two_point", "dose_value")
    assert score(G).max() >= first and score(G).max() > -0.6
