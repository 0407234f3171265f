"""Host-side GA / Monte-Carlo operators of PAPER.md App. B and C: pure numpy, no GPU."""
import numpy as np

from paper_1701_03549_b200 import search


def test_tournament_keeps_the_elite_and_prefers_fitter():
    rng = np.random.default_rng(0)
    fit = np.arange(100, dtype=np.float64)[::-1].copy()        # individual 99 is the best (fitness 0)
    idx = search.tournament_select(rng, fit, n_elite=3)
    assert list(idx[:3]) == [99, 98, 97]                       # elitism: the best survive as they are
    # the winner of a 2-way tournament is the fitter of two uniform draws: E[fitness] = (n - 1) / 3 for fitness 0..n-1
    big = np.concatenate([search.tournament_select(rng, fit, 0) for _ in range(200)])
    assert abs(fit[big].mean() - 99 / 3) < 1.0
    assert fit[big].mean() < fit.mean()


def test_one_point_crossover_swaps_tails():
    rng = np.random.default_rng(1)
    parents = np.stack([np.full(7, i, dtype=np.float64) for i in range(10)])
    child = search.one_point_crossover(rng, parents, n_elite=2)
    assert (child[:2] == parents[:2]).all()
    for i in range(2, 10, 2):
        a, b = child[i], child[i + 1]
        cut = int(np.argmax(a != a[0]))                        # first swapped gene
        assert 1 <= cut < 7
        assert (a[:cut] == i).all() and (a[cut:] == i + 1).all()
        assert (b[:cut] == i + 1).all() and (b[cut:] == i).all()
    # genes are only moved between the two parents of a pair, column by column
    assert np.allclose(np.sort(child, axis=0), np.sort(parents, axis=0))


def test_mutation_probability_decays_and_mutation_respects_bounds():
    p = [search.mutation_probability(g, 20) for g in range(20)]
    assert p[0] == 0.25 and abs(p[-1] - 0.02) < 1e-12 and all(x > y for x, y in zip(p, p[1:]))   # dynamic mutation
    rng = np.random.default_rng(2)
    lo, hi = np.array([-1.0, 0.0, 5.0]), np.array([1.0, 2.0, 6.0])
    pop = lo + rng.random((4000, 3)) * (hi - lo)
    out = search.mutate(rng, pop, 0.25, lo, hi, n_elite=5)
    assert (out[:5] == pop[:5]).all()
    assert (out >= lo).all() and (out <= hi).all()
    changed = (out != pop)[5:].mean()
    assert 0.2 < changed < 0.3
    assert (search.mutate(rng, pop, 0.0, lo, hi) == pop).all()


def test_ga_and_monte_carlo_minimise_a_known_function():
    target = np.array([0.3, -1.2, 2.0, 0.5, 0.0])
    lo, hi = np.full(5, -3.0), np.full(5, 3.0)
    f = lambda pop: ((np.asarray(pop) - target) ** 2).sum(axis=1)
    best, fit, hist = search.genetic_algorithm(f, lo, hi, pop_size=128, generations=40, n_elite=2, seed=3)
    assert fit < 0.05 and np.abs(best - target).max() < 0.25
    assert hist[-1][1] <= hist[0][1] and len(hist) == 40
    bests = [h[1] for h in hist]
    assert all(b2 <= b1 + 1e-12 for b1, b2 in zip(bests, bests[1:]))       # elitism: the best never gets worse on a deterministic function
    samples, fits = search.monte_carlo(f, lo, hi, n_samples=4096, batch=500, seed=4)
    assert (np.diff(fits) >= 0).all() and fits[0] < 1.0 and samples.shape == (4096, 5)


def test_scar_cells_initial_population_and_ensemble_estimate():
    """SURVEY 8 f2 host pieces: candidates come from the reference scar, the estimate and its error from the
    ensemble below a fitness cutoff."""
    mask = np.zeros((5, 40), bool)
    mask[1, 3] = mask[4, 33] = mask[2, 31] = mask[2, 32] = True
    Ww = 2
    words = np.zeros((5, Ww), np.uint32)
    for y, x in zip(*np.nonzero(mask)):
        words[y, x >> 5] |= np.uint32(1) << np.uint32(x & 31)
    cells = search.scar_cells(words, 40)
    assert sorted(map(tuple, cells.tolist())) == sorted([(3, 1), (33, 4), (31, 2), (32, 2)])
    rng = np.random.default_rng(0)
    lo, hi = np.array([-1.0, -2, -3, -4, -5, 0, 0]), np.array([1.0, 2, 3, 4, 5, 39, 4])
    pop = search.initial_population_with_ignition(rng, lo, hi, cells, 500)
    assert pop.shape == (500, 7) and (pop[:, :5] >= lo[:5]).all() and (pop[:, :5] <= hi[:5]).all()
    assert set(map(tuple, pop[:, 5:7].astype(int).tolist())) == set(map(tuple, cells.tolist()))      # every candidate is a scar cell
    ind = np.array([[0.0, 10], [1.0, 20], [2.0, 30], [3.0, 40]]); fit = np.array([0.5, 0.1, 0.2, np.inf])
    best, mean, sd, n = search.ensemble_estimate(ind, fit, cutoff=0.3)
    assert (best == [1.0, 20]).all() and n == 2 and np.allclose(mean, [1.5, 25]) and np.allclose(sd, np.std([[1.0, 20], [2.0, 30]], axis=0, ddof=1))
    assert search.ensemble_estimate(ind, fit, cutoff=0.01)[3] == 0


def test_ga_with_initial_population_and_archive():
    target = np.array([0.3, -1.2])
    f = lambda pop: ((np.asarray(pop) - target) ** 2).sum(axis=1)
    init = np.full((32, 2), 2.5)
    arch = []
    best, fit, hist = search.genetic_algorithm(f, [-3, -3], [3, 3], generations=30, n_elite=2, seed=1, init=init, archive=arch)
    assert len(arch) == 30 and arch[0][0].shape == (32, 2) and (arch[0][0] == 2.5).all()
    assert fit < f(init[:1])[0]
