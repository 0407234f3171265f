"""Pins for the oracle's fitness (C-5, Eq. 2) and group statistics."""
import numpy as np
import pytest

from conftest import pack_bitmap


def rand_maps(rng, H, W, n):
    return [rng.random((H, W)) < rng.uniform(0.05, 0.6) for _ in range(n)]


def test_eq2_special_cases(orc):
    """PAPER.md:123 'This function is 0 when simulation and real maps are perfectly overlapped'."""
    rng = np.random.default_rng(0)
    A = rng.random((20, 45)) < 0.4
    a = pack_bitmap(A); N = int(A.sum())
    I, Ns, Nr = orc.fitness_counts(a, a, 45)
    assert (I, Ns, Nr) == (N, N, N)
    assert orc.fitness_score(I, Ns, Nr, 0) == 0.0 and orc.fitness_score(I, Ns, Nr, 1) == 1.0
    empty = pack_bitmap(np.zeros_like(A))
    I, Ns, Nr = orc.fitness_counts(a, empty, 45)                      # A* empty: delta = 1, J = 0
    assert (I, Ns) == (0, 0) and orc.fitness_score(I, Ns, Nr, 0) == 1.0 and orc.fitness_score(I, Ns, Nr, 1) == 0.0
    B = ~A & (rng.random(A.shape) < 0.5)                              # disjoint: delta = (N + N*) / N
    I, Ns, Nr = orc.fitness_counts(a, pack_bitmap(B), 45)
    assert I == 0 and orc.fitness_score(I, Ns, Nr, 0) == np.float32(N + B.sum()) / np.float32(N)
    with np.errstate(all="ignore"):
        assert np.isnan(orc.fitness_score(0, 0, 0, 0)) and np.isinf(orc.fitness_score(0, 5, 0, 0))   # N = 0: IEEE


def test_eq2_against_numpy_set_arithmetic(orc):
    rng = np.random.default_rng(1)
    for H, W in ((7, 31), (9, 32), (5, 33), (16, 100)):
        A = rand_maps(rng, H, W, 1)[0]
        for B in rand_maps(rng, H, W, 6):
            I, Ns, Nr = orc.fitness_counts(pack_bitmap(A), pack_bitmap(B), W)
            assert (I, Ns, Nr) == ((A & B).sum(), B.sum(), A.sum())
            union, inter = (A | B).sum(), (A & B).sum()
            delta = orc.fitness_score(I, Ns, Nr, 0)
            assert delta == np.float32(union - inter) / np.float32(A.sum())        # Eq. 2 literally
            assert float(delta) * A.sum() == pytest.approx(Nr + Ns - 2 * I, rel=1e-6)
            assert orc.fitness_score(I, Ns, Nr, 1) == np.float32(inter) / np.float32(union)


def test_group_stats_against_numpy(orc):
    rng = np.random.default_rng(2)
    G, R, N = 13, 16, 5000
    Ns = rng.integers(0, 9000, (G, R)); I = np.minimum(Ns, rng.integers(0, N, (G, R)))
    counts = np.stack([I, Ns], axis=-1).astype(np.uint32)
    sums, mv = orc.group_stats(counts, N, G, R)
    x = N + Ns - 2 * I
    assert (sums[:, 0] == x.sum(1)).all() and (sums[:, 1] == (x.astype(object) ** 2).sum(1)).all()
    delta = x / N
    assert mv[:, 0] == pytest.approx(delta.mean(1), rel=1e-12)
    assert mv[:, 1] == pytest.approx(delta.var(1, ddof=1), rel=1e-9)               # R-16: sample variance
    same = np.tile(counts[:1, :1], (1, R, 1))
    _, mv1 = orc.group_stats(same, N, 1, R)
    assert mv1[0, 1] == 0.0
