"""`-m "not gpu"`: pins of the oracle's fuel-dependent burn-out time variant (C-4', reading R-21; SURVEY 8 f3;
PAPER.md:91, :145, :68, :273).  None of them re-types the oracle's loop:

  * burn_time == 1 everywhere reproduces orc_simulate byte for byte (burnt map, steps, ignition times, counters);
  * p == 1: the burnt set is the burnable 8-connected component (scipy.ndimage.label), every cell ignites at its BFS depth
    whatever the burn times, and the run lasts max(depth + burn_time) steps;
  * p == 0: only the ignition burns, for burn_time[its class] steps;
  * lattices <= 3 x 3, burn times 1..3: exact law of the final burnt set by enumerating the Markov chain on
    (remaining active time per cell, burnt set) with rational probabilities (chi-square);
  * percolation identity with memory: every directed pair (s -> c) is tried burn_time(s) times unless c burns first, so the
    final burnt set has the law of "reachable from the ignition when edge (s -> c, d) is open with probability
    1 - (1 - p_cd)^burn_time(s)"; an independent numpy sampler + BFS must match the burnt-area distribution (KS).
"""
from fractions import Fraction
from itertools import product

import numpy as np
import pytest
from scipy import ndimage, stats

from conftest import OFFSETS, unpack_bitmap


def random_landscape(orc, rng, H, W, nonburn=0.25, nveg=4):
    veg = rng.choice(nveg, size=(H, W), p=[nonburn] + [(1 - nonburn) / (nveg - 1)] * (nveg - 1)).astype(np.uint8)
    ls = {"veg": veg, "slope": rng.uniform(0, 0.6, (H, W)).astype(np.float32),
          "aspect": rng.uniform(0, 2 * np.pi, (H, W)).astype(np.float32),
          "wind": rng.uniform(0, 2 * np.pi, (H, W)).astype(np.float32)}
    return ls, orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])


def test_burn_time_one_is_the_base_model_byte_for_byte(orc):
    rng = np.random.default_rng(7)
    for _ in range(12):
        H, W = int(rng.integers(1, 40)), int(rng.integers(1, 50))
        ls, L = random_landscape(orc, rng, H, W)
        beta = np.array([rng.uniform(-1.5, 0.5), -0.4, 0.2, 0.9, 0.6], np.float32)
        ign = (int(rng.integers(0, W)), int(rng.integers(0, H)))
        seed = int(rng.integers(0, 2 ** 62))
        ms = int(rng.choice([0, 0, 5]))
        a = orc.simulate(L, beta, ign, seed, sim=3, max_steps=ms, want_time=True)
        for bt in ([1, 1, 1, 1], [0, 1, 1, 1], [1]):                  # 0 and missing entries read as 1
            b = orc.simulate_burn_time(L, beta, bt + [1] * (4 - len(bt)), ign, seed, sim=3, max_steps=ms, want_time=True)
            assert (a["burned"] == b["burned"]).all() and (a["time"] == b["time"]).all()
            assert (a["steps"], a["trials"], a["cand_steps"], a["distinct"]) == (b["steps"], b["trials"], b["cand_steps"], b["distinct"])


def bfs_depth(burnable, ix, iy):
    H, W = burnable.shape
    depth = np.full((H, W), -1, np.int64)
    if not burnable[iy, ix]:
        return depth
    depth[iy, ix] = 0
    frontier = [(ix, iy)]
    while frontier:
        nxt = []
        for (x, y) in frontier:
            for dx, dy in OFFSETS:
                u, v = x + dx, y + dy
                if 0 <= u < W and 0 <= v < H and burnable[v, u] and depth[v, u] < 0:
                    depth[v, u] = depth[y, x] + 1
                    nxt.append((u, v))
        frontier = nxt
    return depth


def test_certain_spread_burns_the_component_at_bfs_depth_and_lasts_depth_plus_burn_time(orc):
    rng = np.random.default_rng(8)
    for _ in range(10):
        H, W = int(rng.integers(2, 30)), int(rng.integers(2, 30))
        ls, L = random_landscape(orc, rng, H, W, nonburn=0.4)
        burnable = ls["veg"] != 0
        ys, xs = np.nonzero(burnable)
        k = int(rng.integers(0, len(xs)))
        ign = (int(xs[k]), int(ys[k]))
        bt = [1] + [int(v) for v in rng.integers(1, 6, 3)]
        r = orc.simulate_burn_time(L, np.array([50, 0, 0, 0, 0], np.float32), bt, ign, 5, want_time=True)
        lab, _ = ndimage.label(burnable, structure=np.ones((3, 3)))
        comp = lab == lab[ign[1], ign[0]]
        assert (unpack_bitmap(r["burned"], W) == comp).all()
        depth = bfs_depth(burnable, *ign)
        assert (r["time"][comp] == depth[comp]).all() and (r["time"][~comp] == -1).all()
        assert r["steps"] == int((depth[comp] + np.asarray(bt)[ls["veg"][comp]]).max())


def test_no_spread_burns_the_ignition_for_its_burn_time(orc):
    rng = np.random.default_rng(9)
    ls, L = random_landscape(orc, rng, 9, 9, nonburn=0.0)
    for v, k in [(1, 4), (2, 1), (3, 7)]:
        ls["veg"][4, 4] = v
        L = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
        bt = [1, 4, 1, 7]
        r = orc.simulate_burn_time(L, np.array([-50, 0, 0, 0, 0], np.float32), bt, (4, 4), 1)
        assert r["steps"] == k and int(unpack_bitmap(r["burned"], 9).sum()) == 1
        assert r["trials"] == 8 * k                                    # every step it is active it tries its 8 neighbours again
        assert orc.simulate_burn_time(L, np.array([-50, 0, 0, 0, 0], np.float32), bt, (4, 4), 1, max_steps=2)["steps"] == min(k, 2)


def exact_final_distribution(T, burnable, veg, bt, ix, iy):
    """Exact law of the final burnt set: Markov chain on (frozenset of (cell, steps left), burnt set), rational probabilities."""
    H, W = burnable.shape
    cells = [(x, y) for y in range(H) for x in range(W)]

    def q(x, y, d):
        t = int(T[y, x, d])
        return Fraction(1) if t == 0xFFFFFFFF else Fraction(t, 2 ** 32)

    final = {}
    start = (frozenset([((ix, iy), bt[veg[iy, ix]])]), frozenset([(ix, iy)]))
    level = {start: Fraction(1)}
    while level:
        nxt = {}
        for (active, burned), pr in level.items():
            if not active:
                final[burned] = final.get(burned, 0) + pr
                continue
            act = {c for c, _ in active}
            cand = []
            for (x, y) in cells:
                if not burnable[y, x] or (x, y) in burned:
                    continue
                miss = Fraction(1); has = False
                for d, (dx, dy) in enumerate(OFFSETS):
                    if (x - dx, y - dy) in act:
                        miss *= 1 - q(x, y, d); has = True
                if has:
                    cand.append(((x, y), 1 - miss))
            stay = frozenset((c, left - 1) for c, left in active if left > 1)
            for pattern in product((0, 1), repeat=len(cand)):
                pp = pr
                for (c, pi), bit in zip(cand, pattern):
                    pp *= pi if bit else 1 - pi
                if pp == 0:
                    continue
                new = [c for (c, _), bit in zip(cand, pattern) if bit]
                key = (stay | frozenset((c, bt[veg[c[1], c[0]]]) for c in new), burned | frozenset(new))
                nxt[key] = nxt.get(key, 0) + pp
        level = nxt
    return final


@pytest.mark.parametrize("H,W,seed,bt", [(3, 3, 0, [1, 2, 1, 3]), (2, 3, 1, [1, 2, 2, 2]), (3, 2, 2, [1, 3, 1, 2])])
def test_tiny_lattice_exact_markov_enumeration_with_burn_times(orc, H, W, seed, bt):
    rng = np.random.default_rng(100 + seed)
    ls, L = random_landscape(orc, rng, H, W, nonburn=0.15)
    ls["veg"][H // 2, W // 2] = 1
    L = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    beta = np.array([-1.6, 0.4, 0.3, 0.8, 0.5], np.float32)
    T = orc.threshold_table(L, beta)
    ign = (W // 2, H // 2)
    exact = exact_final_distribution(T, ls["veg"] != 0, ls["veg"], bt, *ign)
    assert abs(sum(exact.values()) - 1) == 0
    n = 60000
    counts = {}
    for s in range(n):
        r = orc.simulate_burn_time(L, beta, bt, ign, seed=1234 + s, sim=s, table=T)
        m = unpack_bitmap(r["burned"], W)
        key = frozenset((int(x), int(y)) for y, x in zip(*np.nonzero(m)))
        counts[key] = counts.get(key, 0) + 1
    assert set(counts) <= set(exact)
    keys = [k for k in exact if exact[k] * n >= 5]
    obs = np.array([counts.get(k, 0) for k in keys], float)
    exp = np.array([float(exact[k]) * n for k in keys])
    rest_o, rest_e = n - obs.sum(), n - exp.sum()
    if rest_e >= 5:
        obs, exp = np.append(obs, rest_o), np.append(exp, rest_e)
    else:
        exp = exp * (obs.sum() / exp.sum())
    chi2, pval = stats.chisquare(obs, exp)
    assert pval > 1e-3, (chi2, pval, len(keys))
    # and it is NOT the law of the one-step model (the pin would not notice a burn time that is ignored otherwise)
    base = exact_final_distribution(T, ls["veg"] != 0, ls["veg"], [1, 1, 1, 1], *ign)
    tv = sum(abs(float(exact.get(k, 0)) - float(base.get(k, 0))) for k in set(exact) | set(base)) / 2
    assert tv > 0.02


def test_percolation_identity_with_burn_times(orc):
    """Reachability in a random digraph with edge probability 1 - (1 - p)^burn_time(source): independent sampler (PCG64), KS."""
    rng = np.random.default_rng(33)
    H, W = 24, 24
    ls, L = random_landscape(orc, rng, H, W, nonburn=0.1)
    ls["veg"][H // 2, W // 2] = 2
    L = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    bt = [1, 3, 1, 2]
    beta = np.array([-2.2, 0.3, 0.2, 0.7, 0.4], np.float32)
    T = orc.threshold_table(L, beta)
    p = np.where(T == 0xFFFFFFFF, 1.0, T.astype(np.float64) / 2.0 ** 32)         # [H][W][8], indexed by TARGET
    burnable = ls["veg"] != 0
    ign = (W // 2, H // 2)
    n = 1000
    a_or = np.array([unpack_bitmap(orc.simulate_burn_time(L, beta, bt, ign, seed=9000 + s, sim=s, table=T)["burned"], W).sum() for s in range(n)])
    k_src = np.asarray(bt)[ls["veg"]]
    a_pc = np.empty(n)
    for s in range(n):
        u = rng.random((H, W, 8))
        seen = np.zeros((H, W), bool); seen[ign[1], ign[0]] = True
        frontier = [ign]
        while frontier:
            nxt = []
            for (x, y) in frontier:
                for d, (dx, dy) in enumerate(OFFSETS):
                    tx, ty = x + dx, y + dy
                    if 0 <= tx < W and 0 <= ty < H and burnable[ty, tx] and not seen[ty, tx]:
                        if u[ty, tx, d] < 1.0 - (1.0 - p[ty, tx, d]) ** k_src[y, x]:
                            seen[ty, tx] = True; nxt.append((tx, ty))
            frontier = nxt
        a_pc[s] = seen.sum()
    ks = stats.ks_2samp(a_or, a_pc)
    assert ks.pvalue > 0.01, ks
    a_base = np.array([unpack_bitmap(orc.simulate(L, beta, ign, 9000 + s, sim=s, table=T)["burned"], W).sum() for s in range(n)])
    assert a_or.mean() > 1.2 * a_base.mean()                                     # longer burning spreads further
