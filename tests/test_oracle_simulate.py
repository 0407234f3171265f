"""Pins for the oracle's CA simulation (C-4): P-1 .. P-7 of DESIGN.md."""
from collections import deque
from fractions import Fraction
from itertools import product

import numpy as np
import pytest
from scipy import ndimage
from scipy.stats import chisquare, ks_2samp

from conftest import OFFSETS, unpack_bitmap

NEVER = (-50.0, 0, 0, 0, 0)       # p == 0 everywhere
ALWAYS = (50.0, 0, 0, 0, 0)       # p == 1 everywhere


def random_landscape(orc, rng, H, W, nonburn=0.25, nveg=4):
    veg = rng.choice(nveg, size=(H, W), p=[nonburn] + [(1 - nonburn) / (nveg - 1)] * (nveg - 1))
    return orc.Landscape(veg, rng.uniform(0, 0.7, (H, W)), rng.uniform(0, 2 * np.pi, (H, W)),
                         rng.uniform(0, 2 * np.pi, (H, W)))


def bfs_depth(burnable: np.ndarray, ix, iy):
    """Brute-force BFS over the 8-neighbourhood (the paper's neighbourhood, PAPER.md:85 '8 cells')."""
    H, W = burnable.shape
    depth = -np.ones((H, W), np.int64)
    if not burnable[iy, ix]:
        return depth
    depth[iy, ix] = 0
    q = deque([(ix, iy)])
    while q:
        x, y = q.popleft()
        for dx, dy in OFFSETS:
            u, v = x + dx, y + dy
            if 0 <= u < W and 0 <= v < H and burnable[v, u] and depth[v, u] < 0:
                depth[v, u] = depth[y, x] + 1
                q.append((u, v))
    return depth


# ------------------------------------------------------------------ P-1
def test_p_zero_burns_only_the_ignition_cell(orc):
    rng = np.random.default_rng(10)
    L = random_landscape(orc, rng, 40, 50)
    ys, xs = np.nonzero(L.veg)
    for k in range(5):
        ix, iy = int(xs[k * 7]), int(ys[k * 7])
        r = orc.simulate(L, NEVER, (ix, iy), seed=k)
        b = unpack_bitmap(r["burned"], L.W)
        assert b.sum() == 1 and b[iy, ix] and r["steps"] == 1


# ------------------------------------------------------------------ P-2
def test_p_one_burns_the_connected_component_in_bfs_order(orc):
    rng = np.random.default_rng(11)
    for trial in range(4):
        L = random_landscape(orc, rng, 48, 70, nonburn=0.45)
        burnable = L.veg != 0
        ys, xs = np.nonzero(burnable)
        ix, iy = int(xs[trial * 13]), int(ys[trial * 13])
        r = orc.simulate(L, ALWAYS, (ix, iy), seed=trial, want_time=True)
        b = unpack_bitmap(r["burned"], L.W)
        lab, _ = ndimage.label(burnable, structure=np.ones((3, 3)))
        assert (b == (lab == lab[iy, ix])).all()                      # textbook component
        depth = bfs_depth(burnable, ix, iy)
        assert (r["time"] == depth).all()                             # burn time = BFS depth
        assert r["steps"] == depth.max() + 1                          # eccentricity + 1


# ------------------------------------------------------------------ P-3, P-4
def test_invariants_every_step(orc):
    rng = np.random.default_rng(12)
    L = random_landscape(orc, rng, 64, 64, nonburn=0.1)
    beta = (-0.9, -0.3, 0.2, 0.6, 0.4)
    burnable = L.veg != 0
    ix, iy = 32, 32
    if not burnable[iy, ix]:
        L.veg[iy, ix] = 2; burnable = L.veg != 0
    full = orc.simulate(L, beta, (ix, iy), seed=5, want_time=True)
    bfull = unpack_bitmap(full["burned"], L.W)
    assert bfull.sum() > 50
    t = full["time"]
    assert ((t >= 0) == bfull).all() and t[iy, ix] == 0
    assert not (bfull & ~burnable).any()                              # burned subset of burnable
    assert full["steps"] == t.max() + 1                               # last burning set is non-empty then dies
    assert full["steps"] <= bfull.sum() <= burnable.sum()             # P-4 termination bound
    # burned after k steps (max_steps) is nested and equals {time <= k}: cells never revert, and a cell
    # burns for exactly one step (it is in 'burning' only at its own ignition time)
    prev = np.zeros_like(bfull)
    for k in range(1, full["steps"] + 1, max(1, full["steps"] // 12)):
        rk = orc.simulate(L, beta, (ix, iy), seed=5, max_steps=k)
        bk = unpack_bitmap(rk["burned"], L.W)
        assert (bk == ((t >= 0) & (t <= k))).all()
        assert not (prev & ~bk).any()
        prev = bk
    # every burned cell but the ignition was ignited by a neighbour burning exactly one step before
    for y, x in zip(*np.nonzero(t > 0)):
        assert any(0 <= x - dx < L.W and 0 <= y - dy < L.H and t[y - dy, x - dx] == t[y, x] - 1
                   for dx, dy in OFFSETS)
    lab, _ = ndimage.label(bfull, structure=np.ones((3, 3)))
    assert lab.max() == 1                                             # burned set is 8-connected


def test_counters_match_their_definition(orc):
    """trials = number of (target, direction) pairs enumerated in C-4 step 2, recounted from the time map."""
    rng = np.random.default_rng(13)
    L = random_landscape(orc, rng, 32, 32, nonburn=0.15)
    L.veg[16, 16] = 2
    r = orc.simulate(L, (-0.7, 0, 0, 0.5, 0), (16, 16), seed=3, want_time=True)
    t = r["time"]; burnable = L.veg != 0
    trials = cands = 0; targets = set()
    INF = 10**9
    tt = np.where(t >= 0, t, INF)
    for step in range(r["steps"]):
        for y, x in product(range(L.H), range(L.W)):
            if not burnable[y, x] or tt[y, x] <= step:               # already burned at time `step`
                continue
            n = sum(1 for dx, dy in OFFSETS
                    if 0 <= x - dx < L.W and 0 <= y - dy < L.H and t[y - dy, x - dx] == step)
            trials += n
            if n:
                cands += 1; targets.add((x, y))
    assert (r["trials"], r["cand_steps"], r["distinct"]) == (trials, cands, len(targets))


def test_ignition_outside_or_nonburnable_burns_nothing(orc):
    rng = np.random.default_rng(14)
    L = random_landscape(orc, rng, 16, 16)
    ys, xs = np.nonzero(L.veg == 0)
    for ign in ((-1, 3), (3, -1), (16, 3), (3, 16), (int(xs[0]), int(ys[0]))):
        r = orc.simulate(L, ALWAYS, ign, seed=1)
        assert r["burned"].sum() == 0 and r["steps"] == 0             # R-12


def test_determinism_and_seed_sim_sensitivity(orc):
    rng = np.random.default_rng(15)
    L = random_landscape(orc, rng, 48, 48, nonburn=0.05)
    L.veg[24, 24] = 2
    beta = (-0.8, 0, 0, 0.3, 0)
    a = orc.simulate(L, beta, (24, 24), seed=77, sim=2)
    b = orc.simulate(L, beta, (24, 24), seed=77, sim=2)
    assert (a["burned"] == b["burned"]).all() and a["steps"] == b["steps"]
    assert (orc.simulate(L, beta, (24, 24), seed=78, sim=2)["burned"] != a["burned"]).any()
    assert (orc.simulate(L, beta, (24, 24), seed=77, sim=3)["burned"] != a["burned"]).any()
    # batch == one by one, with explicit sim indices
    r = orc.simulate_batch(L, [beta], [(24, 24)] * 3, [0, 0, 0], [77, 77, 78], sim_index=[2, 3, 2])
    assert (r["burned"][0] == a["burned"]).all() and r["steps"][0] == a["steps"]
    tab = orc.threshold_table(L, beta)
    c = orc.simulate(L, beta, (24, 24), seed=77, sim=2, table=tab)
    assert (c["burned"] == a["burned"]).all()                         # table route == on-demand route


# ------------------------------------------------------------------ P-5
def test_one_dimensional_strip_closed_form(orc):
    """1 x W strip, uniform p, centre ignition: left/right extents are independent truncated geometric
    variables, P(extent >= k) = q^k with q = T / 2^32; chi^2 on the area pmf over 10^5 replicates."""
    W, x0, n = 41, 20, 100_000
    L = orc.Landscape(np.full((1, W), 2), np.zeros((1, W)), np.zeros((1, W)), np.zeros((1, W)))
    beta = (0.85, 0, 0, 0, 0)
    q = orc.threshold(beta, 2, 0, 0, 0, 2) / 2.0**32
    assert q == pytest.approx(0.70, abs=0.01)
    r = orc.simulate_batch(L, [beta], [(x0, 0)] * n, [0] * n, np.arange(n) + 1000)
    area = np.array([bin(int(w[0, 0]) | (int(w[0, 1]) << 32)).count("1") for w in r["burned"]])
    m = 20
    ext = np.array([q**k * (1 - q) for k in range(m)] + [q**m])       # P(extent = k), truncated at m
    pmf = np.convolve(ext, ext)                                        # area - 1 = left + right
    obs = np.bincount(area - 1, minlength=2 * m + 1)
    exp = pmf * n
    keep = exp >= 5
    obs_k = np.append(obs[keep], obs[~keep].sum()); exp_k = np.append(exp[keep], exp[~keep].sum())
    _, p = chisquare(obs_k, exp_k)
    assert p > 1e-3, p
    # steps = max(left, right) + 1 (+1 more when the longer side was stopped by a failed trial, not the edge)
    assert r["steps"].max() <= m + 1


# ------------------------------------------------------------------ P-6
def exact_final_distribution(T, burnable, ix, iy):
    """Exact law of the final burned set on a tiny lattice by enumerating the Markov chain on
    (burning, burned) with rational probabilities T/2^32 (T = 0xFFFFFFFF counts as 1)."""
    H, W = burnable.shape
    cells = [(x, y) for y in range(H) for x in range(W)]

    def q(x, y, d):
        t = int(T[y, x, d])
        return Fraction(1) if t == 0xFFFFFFFF else Fraction(t, 2**32)

    final = {}
    start = (frozenset([(ix, iy)]), frozenset([(ix, iy)]))
    level = {start: Fraction(1)}
    while level:
        nxt = {}
        for (burning, burned), pr in level.items():
            if not burning:
                final[burned] = final.get(burned, 0) + pr
                continue
            cand = []
            for (x, y) in cells:
                if not burnable[y, x] or (x, y) in burned:
                    continue
                miss = Fraction(1); has = False
                for d, (dx, dy) in enumerate(OFFSETS):
                    if (x - dx, y - dy) in burning:
                        miss *= 1 - q(x, y, d); has = True
                if has:
                    cand.append(((x, y), 1 - miss))
            for pattern in product((0, 1), repeat=len(cand)):
                pp = pr
                for (c, pi), bit in zip(cand, pattern):
                    pp *= pi if bit else 1 - pi
                if pp == 0:
                    continue
                new = frozenset(c for (c, _), bit in zip(cand, pattern) if bit)
                key = (new, burned | new)
                nxt[key] = nxt.get(key, 0) + pp
        level = nxt
    return final


@pytest.mark.parametrize("H,W,seed", [(3, 3, 0), (2, 3, 1), (3, 2, 2)])
def test_tiny_lattice_exact_markov_enumeration(orc, H, W, seed):
    rng = np.random.default_rng(100 + seed)
    veg = rng.integers(1, 4, (H, W)); veg[rng.integers(H), rng.integers(W)] = 0
    ix, iy = 1, 1
    veg[iy, ix] = 2
    L = orc.Landscape(veg, rng.uniform(0.0, 0.6, (H, W)), rng.uniform(0, 2 * np.pi, (H, W)),
                      rng.uniform(0, 2 * np.pi, (H, W)))
    beta = (-0.4, -0.6, 0.5, 1.2, 0.8)
    T = orc.threshold_table(L, beta)
    assert len(np.unique(T[veg != 0])) > 20                            # genuinely heterogeneous
    law = exact_final_distribution(T, veg != 0, ix, iy)
    assert sum(law.values()) == 1
    n = 200_000
    r = orc.simulate_batch(L, [beta], [(ix, iy)] * n, [0] * n, np.arange(n, dtype=np.uint64) + (seed << 32))
    codes = r["burned"].reshape(n, -1)[:, :H].copy()                   # one word per row (W <= 32)
    key = np.zeros(n, np.int64)
    for y in range(H):
        key |= codes[:, y].astype(np.int64) << (8 * y)
    obs = dict(zip(*np.unique(key, return_counts=True)))
    exp_keys, exp_p = [], []
    for burned, pr in law.items():
        k = 0
        for (x, y) in burned:
            k |= 1 << (8 * y + x)
        exp_keys.append(k); exp_p.append(float(pr))
    assert set(obs) <= set(exp_keys)                                   # nothing impossible happens
    e = np.array(exp_p) * n
    o = np.array([obs.get(k, 0) for k in exp_keys], float)
    big = e >= 5
    o2 = np.append(o[big], o[~big].sum()); e2 = np.append(e[big], e[~big].sum())
    if e2[-1] == 0:
        o2, e2 = o2[:-1], e2[:-1]
    _, p = chisquare(o2, e2 * o2.sum() / e2.sum())
    assert p > 1e-3, p


# ------------------------------------------------------------------ P-7
def percolation_sample(T, burnable, ix, iy, rng):
    """Independent sampler: open every directed edge (c - offset(d) -> c) up front w.p. T[c][d]/2^32
    with numpy's PCG64, then BFS.  Returns (burned mask, steps)."""
    H, W = burnable.shape
    open_ = rng.random((H, W, 8)) < np.where(T == 0xFFFFFFFF, 1.0, T / 2.0**32)
    burned = np.zeros((H, W), bool); burned[iy, ix] = True
    front = burned.copy(); steps = 0
    while front.any():
        new = np.zeros((H, W), bool)
        for d, (dx, dy) in enumerate(OFFSETS):
            src = np.zeros((H, W), bool)                               # src[y, x] = front[y - dy, x - dx]
            ys = slice(max(dy, 0), H + min(dy, 0)); yo = slice(max(-dy, 0), H + min(-dy, 0))
            xs = slice(max(dx, 0), W + min(dx, 0)); xo = slice(max(-dx, 0), W + min(-dx, 0))
            src[ys, xs] = front[yo, xo]
            new |= src & open_[:, :, d]
        new &= burnable & ~burned
        burned |= new; front = new; steps += 1
    return burned, steps


def test_percolation_identity_heterogeneous(orc):
    """Each directed pair is tried at most once, so the final burned set has the law of the cells reachable
    in a random digraph with independent edges; areas and durations must agree in distribution (KS)."""
    from paper_1701_03549_b200 import workloads as wl
    ls = wl.make_landscape(1)
    L = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    beta = wl.load_workload(1, landscape=ls).ref_beta
    T = orc.threshold_table(L, beta)
    n = 1000
    r = orc.simulate_batch(L, [beta], [(32, 32)] * n, [0] * n, np.arange(n, dtype=np.uint64) + 5000)
    area_o = np.array([unpack_bitmap(b, L.W).sum() for b in r["burned"]])
    rng = np.random.Generator(np.random.PCG64(4242))
    area_p, steps_p = [], []
    for _ in range(n):
        b, s = percolation_sample(T, L.veg != 0, 32, 32, rng)
        area_p.append(b.sum()); steps_p.append(s)
    assert area_o.std() > 10                                           # a non-degenerate distribution
    assert ks_2samp(area_o, area_p).pvalue > 0.01
    assert ks_2samp(r["steps"], steps_p).pvalue > 0.01
