"""Host-side search loops that drive the batch API (App. B and App. C).

The paper calibrates the five parameters of Eq. 1 with a genetic algorithm (2-way tournament selection
with elitism, one-point crossover, mutation whose probability decays as the run advances)
or with brute-force Monte Carlo sampling of a prior.  north_star keeps these loops on
the host: every generation is one pass of the hot path (fire_params_upload -> fire_simulate_batch ->
fire_fitness) and one small device-to-host copy of the scores.  The GA operators below are plain numpy
on a (population, genes) array; nothing here touches a kernel, and nothing here is on the timed path of
bench.py.

What the paper does not give (population size, number of generations, elitism count, mutation schedule,
replicates per individual) is chosen here and named in the arguments; DESIGN.md lists the choices.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


# ------------------------------------------------------------------------------------------ operators
def tournament_select(rng: np.random.Generator, fitness: np.ndarray, n_elite: int = 1) -> np.ndarray:
    """Indices of the next generation's parents: the `n_elite` best individuals are kept
    as they are (elitism); every other slot is the fitter of two individuals drawn at random.  Lower
    fitness is better (Eq. 2: 0 = perfect overlap)."""
    n = fitness.shape[0]
    order = np.argsort(fitness, kind="stable")
    out = np.empty(n, dtype=np.int64)
    out[:n_elite] = order[:n_elite]
    a = rng.integers(0, n, n - n_elite)
    b = rng.integers(0, n, n - n_elite)
    out[n_elite:] = np.where(fitness[a] <= fitness[b], a, b)
    return out


def one_point_crossover(rng: np.random.Generator, parents: np.ndarray, n_elite: int = 1) -> np.ndarray:
    """One-point crossover (Fig. B.7): consecutive pairs of parents swap everything beyond a
    random cross point.  The first `n_elite` rows pass through untouched."""
    child = parents.copy()
    n, g = parents.shape
    for i in range(n_elite + ((n - n_elite) & 1), n - 1, 2):
        cut = int(rng.integers(1, g))
        child[i, cut:], child[i + 1, cut:] = parents[i + 1, cut:], parents[i, cut:]
    return child


def mutation_probability(gen: int, n_gen: int, p_start: float = 0.25, p_end: float = 0.02) -> float:
    """Dynamic mutation: the per-gene mutation probability decreases as the GA advances."""
    if n_gen <= 1:
        return p_end
    return p_start + (p_end - p_start) * gen / (n_gen - 1)


def mutate(rng: np.random.Generator, pop: np.ndarray, p_mut: float, lo: np.ndarray, hi: np.ndarray,
           n_elite: int = 1, scale: float = 0.1) -> np.ndarray:
    """Each gene of each non-elite individual changes with probability `p_mut` by a normal step of
    `scale` x the gene's range ("a tiny random gene change", Fig. B.8), clipped to the bounds."""
    out = pop.copy()
    hit = rng.random(pop.shape) < p_mut
    hit[:n_elite] = False
    step = rng.standard_normal(pop.shape) * (hi - lo) * scale
    out[hit] += step[hit]
    return np.clip(out, lo, hi)


# ------------------------------------------------------------------------------------------ evaluation
@dataclass
class Evaluator:
    """One generation on the device: `betas` (P, 5) -> mean Eq. 2 fitness of every individual over
    `replicates` simulations from `ignition` against `reference` (bit-packed burnt map)."""
    L: object                       # libfire.Landscape
    reference: object               # torch int32 [H][Ww] on the device
    ignition: tuple
    replicates: int = 4
    metric: int = 0
    seed: int = 1
    calls: int = field(default=0, init=False)

    def __call__(self, betas: np.ndarray) -> np.ndarray:
        import torch
        from . import libfire as lf
        P, R = betas.shape[0], self.replicates
        S = P * R
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        lf.fire_params_upload(self.L, dev(betas.astype(np.float32)))
        ign = np.tile(np.asarray(self.ignition, np.int32), (S, 1))
        par = np.repeat(np.arange(P, dtype=np.int32), R)
        # new random streams every call: the seed carries the call number, the sim id is the slot
        seeds = (np.uint64(self.seed) << np.uint64(40)) | (np.uint64(self.calls) << np.uint64(20)) | np.arange(S, dtype=np.uint64)
        burned = torch.empty((S, self.L.H, self.L.Ww), dtype=torch.int32, device="cuda")
        lf.fire_simulate_batch(self.L, dev(ign), dev(par), dev(seeds.view(np.int64)), burned)
        score = torch.empty((S,), dtype=torch.float32, device="cuda")
        lf.fire_fitness(self.L, self.reference, burned, self.metric, score)
        self.calls += 1
        return score.cpu().numpy().astype(np.float64).reshape(P, R).mean(axis=1)


@dataclass
class IgnitionEvaluator:
    """The 7-parameter case: an individual is (beta_0 .. beta_4, x, y) and starts its fires
    from its own ignition cell (x, y rounded to the nearest cell and clipped to the lattice).  A cell that cannot burn burns
    nothing (R-12), so Eq. 2 gives that individual delta = 1.  Scores of the last call stay on the device in `last_counts`
    (u32 [P * replicates][2]) for fire_fitness_group_stats (a8: per-candidate mean and variance)."""
    L: object
    reference: object
    replicates: int = 4
    metric: int = 0
    seed: int = 1
    calls: int = field(default=0, init=False)
    last_counts: object = field(default=None, init=False)

    def cells_of(self, pop: np.ndarray) -> np.ndarray:
        xy = np.rint(np.asarray(pop, np.float64)[:, 5:7]).astype(np.int64)
        xy[:, 0] = np.clip(xy[:, 0], 0, self.L.W - 1)
        xy[:, 1] = np.clip(xy[:, 1], 0, self.L.H - 1)
        return xy.astype(np.int32)

    def __call__(self, pop: np.ndarray) -> np.ndarray:
        import torch
        from . import libfire as lf
        pop = np.asarray(pop, np.float64)
        P, R = pop.shape[0], self.replicates
        S = P * R
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        lf.fire_params_upload(self.L, dev(pop[:, :5].astype(np.float32)))
        ign = np.repeat(self.cells_of(pop), R, axis=0)
        par = np.repeat(np.arange(P, dtype=np.int32), R)
        seeds = (np.uint64(self.seed) << np.uint64(40)) | (np.uint64(self.calls) << np.uint64(20)) | np.arange(S, dtype=np.uint64)
        burned = torch.empty((S, self.L.H, self.L.Ww), dtype=torch.int32, device="cuda")
        lf.fire_simulate_batch(self.L, dev(ign), dev(par), dev(seeds.view(np.int64)), burned)
        score = torch.empty((S,), dtype=torch.float32, device="cuda")
        counts = torch.empty((S, 2), dtype=torch.int32, device="cuda")
        lf.fire_fitness(self.L, self.reference, burned, self.metric, score, counts)
        self.last_counts = counts
        self.calls += 1
        return score.cpu().numpy().astype(np.float64).reshape(P, R).mean(axis=1)


def scar_cells(reference_bitmap: np.ndarray, W: int) -> np.ndarray:
    """(x, y) of every burnt cell of a bit-packed map u32[H][ceil(W/32)]: the candidates the paper draws ignition points from
    ("a random ignition point within the reference fire burnt area")."""
    words = np.ascontiguousarray(reference_bitmap, dtype="<u4")
    bits = np.unpackbits(words.view(np.uint8), axis=-1, bitorder="little")[:, :W]
    ys, xs = np.nonzero(bits)
    return np.stack([xs, ys], 1).astype(np.int64)


def initial_population_with_ignition(rng: np.random.Generator, lo, hi, scar: np.ndarray, pop_size: int) -> np.ndarray:
    """Genes 0-4 uniform in [lo, hi]; genes 5-6 = a cell of the reference scar chosen at random."""
    lo, hi = np.asarray(lo, np.float64), np.asarray(hi, np.float64)
    pop = np.empty((pop_size, 7), np.float64)
    pop[:, :5] = lo[:5] + rng.random((pop_size, 5)) * (hi[:5] - lo[:5])
    pop[:, 5:7] = scar[rng.integers(0, scar.shape[0], pop_size)]
    return pop


def ensemble_estimate(individuals: np.ndarray, fitness: np.ndarray, cutoff: float):
    """The paper's reading of a finished search (Tables 2-3): the best individual is the one of minimum fitness; the
    estimate of every parameter is the mean, and its error the standard deviation, over the ensemble of simulated individuals
    whose fitness is below `cutoff`.  Returns (best, mean, sd, ensemble size)."""
    individuals, fitness = np.asarray(individuals, np.float64), np.asarray(fitness, np.float64)
    ok = np.isfinite(fitness)
    best = individuals[int(np.argmin(np.where(ok, fitness, np.inf)))].copy()
    sel = ok & (fitness < cutoff)
    if not sel.any():
        return best, np.full(individuals.shape[1], np.nan), np.full(individuals.shape[1], np.nan), 0
    ens = individuals[sel]
    return best, ens.mean(axis=0), ens.std(axis=0, ddof=1) if ens.shape[0] > 1 else np.zeros(individuals.shape[1]), int(sel.sum())


# ------------------------------------------------------------------------------------------ search loops
def genetic_algorithm(evaluate, lo, hi, pop_size: int = 64, generations: int = 20, n_elite: int = 2,
                      seed: int = 0, p_start: float = 0.25, p_end: float = 0.02, init: np.ndarray | None = None,
                      archive: list | None = None):
    """GA of PAPER.md App. B over the box [lo, hi].  `evaluate(pop) -> fitness` (lower is better).  `init`: first population
    (default: uniform in the box).  `archive`: if a list, every evaluated (population, fitness) pair is appended to it (the
    ensemble the paper's histograms and error bars are made of).
    Returns (best vector, best fitness, history of (generation, best, mean))."""
    rng = np.random.Generator(np.random.PCG64(seed))
    lo, hi = np.asarray(lo, np.float64), np.asarray(hi, np.float64)
    pop = lo + rng.random((pop_size, lo.shape[0])) * (hi - lo) if init is None else np.clip(np.asarray(init, np.float64), lo, hi)
    pop_size = pop.shape[0]
    history = []
    best_vec, best_fit = None, np.inf
    for gen in range(generations):
        fit = np.asarray(evaluate(pop), np.float64)
        fit = np.where(np.isfinite(fit), fit, np.inf)
        if archive is not None:
            archive.append((pop.copy(), fit.copy()))
        k = int(np.argmin(fit))
        if fit[k] < best_fit:
            best_vec, best_fit = pop[k].copy(), float(fit[k])
        history.append((gen, float(fit[k]), float(np.mean(fit[np.isfinite(fit)])) if np.isfinite(fit).any() else np.inf))
        if gen == generations - 1:
            break
        parents = pop[tournament_select(rng, fit, n_elite)]
        pop = mutate(rng, one_point_crossover(rng, parents, n_elite), mutation_probability(gen, generations, p_start, p_end),
                     lo, hi, n_elite)
    return best_vec, best_fit, history


def monte_carlo(evaluate, lo, hi, n_samples: int = 1024, batch: int = 256, seed: int = 0):
    """Brute-force Monte Carlo of PAPER.md App. C: sample the (uniform) prior, simulate everything, rank by
    fitness.  Returns (samples sorted by fitness, sorted fitness)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    lo, hi = np.asarray(lo, np.float64), np.asarray(hi, np.float64)
    samples = lo + rng.random((n_samples, lo.shape[0])) * (hi - lo)
    fit = np.concatenate([np.asarray(evaluate(samples[i:i + batch]), np.float64) for i in range(0, n_samples, batch)])
    order = np.argsort(np.where(np.isfinite(fit), fit, np.inf), kind="stable")
    return samples[order], fit[order]
