"""`-m gpu`: parity of the CUDA path (through the C ABI) with the CPU oracle, element by element.

Layers:
  1. thresholds: GPU table vs oracle table; > 1 count apart = failure, <= 1-count differences are
     counted and reported (north_star).
  2. propagation with the oracle fed the GPU's OWN threshold table: bit-exact, no excuses.
  3. end to end, each side on its own thresholds: bit-exact burned maps, steps, trials and fitness
     on all five configs -- configs 3-5 at full size against values stored by
     oracle/make_workloads.py (oracle only), in the launch configuration bench.py times.
"""
import json

import numpy as np
import pytest

from conftest import GOLDEN, ROOT, unpack_bitmap
from paper_1701_03549_b200 import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():                       # collected on the CPU box too; never runs there
    pytest.skip("needs a CUDA device", allow_module_level=True)

import gpu_helpers as gh                                 # noqa: E402
from paper_1701_03549_b200 import libfire as lf          # noqa: E402


def small_landscape(rng, H, W, nonburn=0.2, nveg=4):
    veg = rng.choice(nveg, size=(H, W), p=[nonburn] + [(1 - nonburn) / (nveg - 1)] * (nveg - 1)).astype(np.uint8)
    return {"veg": veg, "slope": rng.uniform(0, 0.7, (H, W)).astype(np.float32),
            "aspect": rng.uniform(0, 2 * np.pi, (H, W)).astype(np.float32),
            "wind": rng.uniform(0, 2 * np.pi, (H, W)).astype(np.float32), "W": W, "H": H}


def orc_landscape(orc, ls):
    return orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])


def report(request, **kv):
    line = " ".join(f"{k}={v}" for k, v in kv.items())
    print(f"\n[parity] {request.node.name}: {line}")
    request.node.user_properties.append(("parity", line))


# ---------------------------------------------------------------------------------- layer 1
@pytest.mark.parametrize("cfg", [1, 2])
def test_thresholds_within_one_count(orc, request, cfg):
    w = wl.load_workload(cfg)
    Lo = orc_landscape(orc, w.landscape)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, np.vstack([w.betas, w.ref_beta[None, :]]))
    n_diff = n_tot = 0
    for p in range(w.P + 1):
        beta = w.betas[p] if p < w.P else w.ref_beta
        g = gh.thresholds(L, p).astype(np.int64)
        o = orc.threshold_table(Lo, beta).astype(np.int64)
        d = np.abs(g - o)
        assert d.max() <= 1, f"cfg{cfg} p={p}: threshold differs by {d.max()} counts at {np.unravel_index(d.argmax(), d.shape)}"
        assert ((g == 0) == (o == 0))[w.landscape["veg"] == 0].all()
        n_diff += int((d != 0).sum()); n_tot += d.size
    report(request, entries=n_tot, one_count_differences=n_diff, fraction=f"{n_diff / n_tot:.2e}")
    assert n_diff / n_tot < 1e-3
    L.close()


@pytest.mark.parametrize("cfg", [3, 5])
def test_full_size_tables_vs_oracle_counted(orc, request, cfg):
    """north_star: "any threshold that differs by more than 1 count in 2^32 is a failure, and <= 1-count boundary differences
    are counted and reported" -- on the headline config's whole table (256 vectors x 1024 x 1024 x 8 = 2.1e9 entries) and on
    config 5's (16 x 4096 x 4096 x 8), vector by vector against the oracle's table."""
    w = wl.load_workload(cfg)
    Lo = orc_landscape(orc, w.landscape)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, w.betas)
    n_diff = n_tot = 0
    worst = 0
    for p in range(w.P):
        g = gh.thresholds(L, p)
        o = orc.threshold_table(Lo, w.betas[p])
        ne = g != o
        k = int(ne.sum())
        if k:
            d = np.abs(g[ne].astype(np.int64) - o[ne].astype(np.int64))
            worst = max(worst, int(d.max()))
            assert worst <= 1, f"cfg{cfg} p={p}: threshold differs by {worst} counts"
        n_diff += k; n_tot += g.size
    report(request, entries=n_tot, one_count_differences=n_diff, fraction=f"{n_diff / n_tot:.2e}", worst=worst)
    assert n_diff / n_tot < 1e-3
    L.close()


def test_thresholds_extreme_and_special_values(orc, request):
    rng = np.random.default_rng(5)
    ls = small_landscape(rng, 37, 45)
    ls["slope"][0, :8] = [0.0, np.float32(5 * np.pi / 180), np.nextafter(np.float32(5 * np.pi / 180), np.float32(1)), 1.5, 1e-30, 0.3, 0.3, 0.3]
    ls["aspect"][0, :8] = [0.0, 0.0, np.float32(7 * np.pi / 4), np.float32(np.pi / 2), 0.0, np.float32(np.pi / 2), np.float32(np.pi), np.float32(2 * np.pi)]
    ls["wind"][1, :4] = [0.0, np.float32(np.pi / 4), np.float32(np.pi), np.float32(2 * np.pi)]
    betas = np.array([[0, 0, 0, 0, 0], [-50, 0, 0, 0, 0], [50, 0, 0, 0, 0], [-5, -10, 5, 18.1, -5], [23, 0, 0, 0, 0],
                      [-23, 0, 0, 0, 0], [30, -30, 30, -30, 30], [-1.5, 0.25, -0.75, 2.5, 1.25]], np.float32)
    L = gh.make_landscape(ls); Lo = orc_landscape(orc, ls)
    gh.upload(L, betas)
    n_diff = 0
    for p in range(len(betas)):
        g = gh.thresholds(L, p).astype(np.int64); o = orc.threshold_table(Lo, betas[p]).astype(np.int64)
        assert np.abs(g - o).max() <= 1, (p, np.abs(g - o).max())
        n_diff += int((g != o).sum())
    burn = ls["veg"] != 0
    assert (gh.thresholds(L, 0)[burn] == 2 ** 31).all()              # beta = 0 -> p = 1/2 exactly
    assert (gh.thresholds(L, 1) == 0).all()                          # p == 0
    assert (gh.thresholds(L, 2)[burn] == 0xFFFFFFFF).all()           # p == 1 (certain)
    assert (gh.thresholds(L, 2)[~burn] == 0).all()
    report(request, one_count_differences=n_diff)
    L.close()


# ---------------------------------------------------------------------------------- layer 2
@pytest.mark.parametrize("cfg", [1, 2])
def test_propagation_bit_exact_on_gpu_thresholds(orc, request, cfg):
    w = wl.load_workload(cfg)
    Lo = orc_landscape(orc, w.landscape)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, w.betas)
    g = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    tables = [gh.thresholds(L, p) for p in range(w.P)]
    o = orc.simulate_batch(Lo, w.betas, w.ignitions, w.sim_param, w.seeds, tables=tables)
    bad = [s for s in range(w.S) if not (g["burned"][s] == o["burned"][s]).all()]
    assert not bad, f"cfg{cfg}: burned maps differ for sims {bad[:10]}"
    assert (g["steps"] == o["steps"]).all() and (g["trials"] == o["trials"]).all()
    report(request, sims=w.S, trials=int(o["trials"].sum()), cells_burned=int(gh.popcount(o["burned"]).sum()))
    L.close()


# ---------------------------------------------------------------------------------- layer 3
@pytest.mark.parametrize("cfg", [1, 2, 4, 3, 5])
def test_end_to_end_matches_oracle_golden(request, cfg):
    """Full-size configs in bench.py's launch configuration vs values stored by oracle/make_workloads.py."""
    e = json.loads((GOLDEN / f"cfg{cfg}_expected.json").read_text())
    w = wl.load_workload(cfg)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, np.vstack([w.betas, w.ref_beta[None, :]]))      # the reference vector rides along as index P
    g = gh.simulate(L, w.ignitions, w.sim_param, w.seeds, keep_device=True)
    assert (g["steps"] == np.array(e["steps"], np.uint32)).all(), np.flatnonzero(g["steps"] != np.array(e["steps"]))[:10]
    assert (g["trials"] == np.array(e["trials"], np.uint64)).all()
    # reference fire: its own simulation (sim id 0) from the stored vector, ignition and seed
    ref = gh.simulate(L, [w.ref_ignition], [w.P], [w.ref_seed], sim_ids=[0])
    assert gh.digest(ref["burned"][0]) == e["ref_digest"] and int(ref["steps"][0]) == e["ref_steps"]
    counts, score, N = gh.fitness(L, ref["burned"][0], g["burned"], w.metric)
    assert N == e["ref_area"]
    assert (counts[:, 0] == np.array(e["intersection"], np.uint32)).all()
    assert (counts[:, 1] == np.array(e["area"], np.uint32)).all()
    # every burned map, bit for bit (digest of the canonical words), in slabs to bound host memory
    S = w.S
    slab = max(1, (256 << 20) // (L.H * L.Ww * 4))
    bad = []
    for s0 in range(0, S, slab):
        hb = g["burned"][s0:s0 + slab].cpu().numpy().view(np.uint32)
        bad += [s0 + i for i in range(hb.shape[0]) if gh.digest(hb[i]) != e["digest"][s0 + i]]
    assert not bad, f"cfg{cfg}: {len(bad)} burned maps differ, first {bad[:10]}"
    # scores: one IEEE divide of the exact integers, restated here in numpy float32
    I = counts[:, 0].astype(np.int64); A = counts[:, 1].astype(np.int64)
    with np.errstate(all="ignore"):
        want = ((N + A - 2 * I).astype(np.float32) / np.float32(N)) if w.metric == 0 else \
               (I.astype(np.float32) / (N + A - I).astype(np.float32))
    assert np.array_equal(score, want.astype(np.float32), equal_nan=True)
    if w.groups:
        G, R = w.groups
        sums, mv = gh.group_stats(counts, N, G, R)
        x = (N + A - 2 * I).reshape(G, R)
        assert (sums[:, 0] == x.sum(1)).all() and (sums[:, 1] == (x * x).sum(1)).all()
        d = x / N
        assert np.allclose(mv[:, 0], d.mean(1), rtol=1e-13) and np.allclose(mv[:, 1], d.var(1, ddof=1), rtol=1e-9, atol=1e-18)
    report(request, sims=S, trials=e["totals"]["trials"], burned_cells=e["totals"]["area"], launches=lf.fire_launch_count(L))
    L.close()


# ---------------------------------------------------------------------------------- edge cases
def test_limits_p0_p1_and_invalid_sims(orc):
    rng = np.random.default_rng(21)
    ls = small_landscape(rng, 50, 77, nonburn=0.4)          # width not a multiple of 32: ragged tail
    ls["veg"][0, 0] = 1; ls["veg"][49, 76] = 2              # burnable corners: fires that start on the lattice edge
    Lo = orc_landscape(orc, ls)
    L = gh.make_landscape(ls)
    betas = np.array([[-50, 0, 0, 0, 0], [50, 0, 0, 0, 0], [-1, 0, 0.2, 1, 0.5]], np.float32)
    gh.upload(L, betas)
    ys, xs = np.nonzero(ls["veg"]); nb_y, nb_x = np.nonzero(ls["veg"] == 0)
    ign = [[xs[3], ys[3]], [xs[3], ys[3]], [xs[40], ys[40]], [nb_x[0], nb_y[0]], [-1, 5], [77, 5], [5, 50], [5, -1],
           [xs[9], ys[9]], [xs[9], ys[9]], [0, 0], [76, 49]]
    par = [0, 1, 2, 1, 1, 1, 1, 1, 3, -1, 1, 1]
    seeds = np.arange(len(par), dtype=np.uint64) + 77
    g = gh.simulate(L, ign, par, seeds)
    o = orc.simulate_batch(Lo, betas, np.array(ign, np.int32), np.array(par, np.int32), seeds)
    assert (g["burned"] == o["burned"]).all() and (g["steps"] == o["steps"]).all() and (g["trials"] == o["trials"]).all()
    b = unpack_bitmap(g["burned"], 77)
    assert b[0].sum() == 1 and g["steps"][0] == 1                                   # p == 0: ignition only
    from scipy import ndimage
    lab, _ = ndimage.label(ls["veg"] != 0, structure=np.ones((3, 3)))
    assert (b[1] == (lab == lab[ys[3], xs[3]])).all()                               # p == 1: the 8-connected component
    for s in (3, 4, 5, 6, 7, 8, 9):
        assert b[s].sum() == 0 and g["steps"][s] == 0 and g["trials"][s] == 0       # R-12
    assert (g["burned"][:, :, -1] >> np.uint32(77 - 64)).max() == 0                  # tail bits stay zero
    L.close()


@pytest.mark.parametrize("H,W", [(1, 1), (1, 200), (130, 1), (3, 33), (64, 64), (97, 161)])
def test_odd_shapes_bit_exact(orc, H, W):
    rng = np.random.default_rng(H * 1000 + W)
    ls = small_landscape(rng, H, W, nonburn=0.1)
    Lo = orc_landscape(orc, ls); L = gh.make_landscape(ls)
    betas = np.array([[0.3, -0.5, 0.3, 1.0, 0.5], [-0.6, 0, 0, 0.5, 0], [50, 0, 0, 0, 0]], np.float32)
    gh.upload(L, betas)
    S = 24
    ign = np.stack([rng.integers(0, W, S), rng.integers(0, H, S)], 1).astype(np.int32)
    par = (np.arange(S) % 3).astype(np.int32); seeds = rng.integers(0, 2 ** 63, S).astype(np.uint64)
    g = gh.simulate(L, ign, par, seeds)
    tables = [gh.thresholds(L, p) for p in range(3)]
    o = orc.simulate_batch(Lo, betas, ign, par, seeds, tables=tables)
    assert (g["burned"] == o["burned"]).all() and (g["steps"] == o["steps"]).all() and (g["trials"] == o["trials"]).all()
    L.close()


def test_max_steps_and_sim_ids(orc):
    w = wl.load_workload(1)
    Lo = orc_landscape(orc, w.landscape); L = gh.make_landscape(w.landscape)
    gh.upload(L, w.betas)
    for ms in (1, 2, 7):
        g = gh.simulate(L, w.ignitions, w.sim_param, w.seeds, max_steps=ms)
        o = orc.simulate_batch(Lo, w.betas, w.ignitions, w.sim_param, w.seeds, max_steps=ms)
        assert (g["burned"] == o["burned"]).all() and (g["steps"] == o["steps"]).all()
    # a shard of the batch with explicit sim ids reproduces the same fires (multi-GPU sharding)
    full = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    sl = wl.shard_sims(w.S, 1, 3)
    part = gh.simulate(L, w.ignitions[sl], w.sim_param[sl], w.seeds[sl], sim_ids=np.arange(w.S, dtype=np.int32)[sl])
    assert (part["burned"] == full["burned"][sl]).all() and (part["trials"] == full["trials"][sl]).all()
    L.close()


def test_param_shards_through_libfire_reproduce_the_full_batch():
    """two ranks' work done one after the other on this GPU, each with ITS OWN table of P / 2 vectors: burnt maps,
    steps, trials and scores of the merged shards equal the full batch bit for bit."""
    w = wl.load_workload(2)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, np.vstack([w.betas, w.ref_beta[None, :]]))
    ref = gh.simulate(L, [w.ref_ignition], [w.P], [w.ref_seed], sim_ids=[0])["burned"][0]
    gh.upload(L, w.betas)
    full = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    _, full_score, _ = gh.fitness(L, ref, full["burned"], w.metric)
    for world in (2, 3):
        shards = [wl.shard_by_param(w, r, world) for r in range(world)]
        res, scores = [], []
        for sh in shards:
            Lr = gh.make_landscape(w.landscape)                    # a rank's own handle: only its slice of the table exists
            gh.upload(Lr, sh.betas)
            assert sh.betas.shape[0] <= (w.P + world - 1) // world
            r = gh.simulate(Lr, sh.ignitions, sh.sim_param, sh.seeds, sim_ids=sh.sim_ids)
            res.append(r); scores.append(gh.fitness(Lr, ref, r["burned"], w.metric)[1])
            Lr.close()
        for key in ("burned", "steps", "trials"):
            assert (wl.merge_param_shards(shards, [r[key] for r in res], w.S) == full[key]).all(), (world, key)
        merged = wl.merge_param_shards(shards, scores, w.S)
        assert np.array_equal(merged.view(np.uint32), full_score.view(np.uint32))
    L.close()


def test_results_do_not_depend_on_launch_geometry_or_list_capacity(request):
    """Pin P-9: same bytes for every CTA size, residency, shared/global list split, and through the rescue kernel."""
    w = wl.load_workload(2)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, w.betas)
    base = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    again = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    assert (base["burned"] == again["burned"]).all()
    # (threads per CTA, CTAs per SM, shared list entries, total list entries, launch order, kernel family)
    # family 0 = automatic, 1 = two-phase kernel, 2 = asynchronous-warp kernel, 3 / 4 = the latter as clusters of 2 / 4 CTAs
    for threads, per_sm, shared, total, order, family in [
            (32, 1, 0, 0, 0, 0), (64, 8, 0, 0, 1, 0), (128, 2, 0, 0, 0, 0), (512, 1, 0, 0, 0, 1), (1024, 1, 0, 0, 1, 1),
            (256, 4, 16, 0, 0, 0), (256, 4, 5, 4096, 1, 0), (96, 3, 1, 0, 0, 0), (256, 4, 8, 8, 0, 0),
            (128, 4, 64, 100, 1, 0), (256, 2, 0, 1, 0, 0), (256, 5, 0, 0, 0, 0), (256, 6, 0, 0, 1, 0),
            (256, 8, 768, 0, 0, 0), (128, 1, 0, 0, 1, 0), (128, 16, 0, 0, 0, 1), (0, 0, 0, 0, 0, 1),
            (256, 4, 0, 0, 0, 2), (32, 2, 0, 0, 1, 2), (1024, 1, 0, 0, 0, 2), (512, 2, 16, 0, 0, 2),
            (256, 5, 5, 4096, 1, 2), (256, 6, 8, 8, 0, 2), (128, 4, 1, 1, 0, 2), (0, 0, 0, 0, 0, 2),
            (1024, 1, 0, 0, 0, 3), (1024, 1, 0, 0, 1, 4), (256, 2, 0, 0, 0, 4), (512, 1, 16, 0, 1, 3), (128, 4, 1, 4096, 0, 4),
            (64, 3, 5, 4096, 1, 3), (256, 4, 8, 8, 0, 3), (32, 1, 0, 0, 0, 4), (0, 0, 0, 0, 0, 3), (0, 0, 0, 0, 1, 4),
            (896, 1, 0, 0, 0, 3), (896, 1, 16, 0, 1, 4), (768, 1, 0, 0, 0, 2)]:
        mode = (threads, per_sm, shared, total, order, family)
        lf.fire_set_launch_geometry(L, threads, per_sm)
        lf.fire_set_list_capacity(L, shared, total)
        lf.fire_set_schedule(L, order)
        lf.fire_set_kernel(L, family)
        g = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
        ok = (g["burned"] == base["burned"]).all(axis=(1, 2))
        assert ok.all(), f"geometry {mode}: sims {np.flatnonzero(~ok)[:10]} differ"
        assert (g["steps"] == base["steps"]).all() and (g["trials"] == base["trials"]).all(), mode
    L.close()


# ---------------------------------------------------------------------------------- fitness
def test_fitness_counts_and_scores_bit_exact(orc):
    rng = np.random.default_rng(3)
    for H, W, S in [(64, 64, 7), (50, 77, 5), (1, 1, 2), (1024, 1024, 3), (33, 4100, 4)]:
        ls = small_landscape(rng, H, W)
        L = gh.make_landscape(ls)
        Ww = (W + 31) // 32
        mask = np.zeros((Ww * 32,), bool); mask[:W] = True
        tail = np.packbits(mask, bitorder="little").view("<u4")
        ref = rng.integers(0, 2 ** 32, (H, Ww), dtype=np.uint32) & tail
        burned = rng.integers(0, 2 ** 32, (S, H, Ww), dtype=np.uint32) & tail
        burned[0] = ref; burned[1] = 0
        if S > 2:
            burned[2] = ~ref & tail
        for metric in (0, 1):
            counts, score, N = gh.fitness(L, ref, burned, metric)
            oc, os_, oN = orc.fitness(ref, burned, W, metric)
            assert N == oN and (counts == oc).all()
            assert np.array_equal(score.view(np.uint32), os_.view(np.uint32))                    # bit-exact floats
        # empty reference: N = 0 gives inf / NaN, not an error
        counts, score, N = gh.fitness(L, np.zeros_like(ref), burned, 0)
        oc, os_, oN = orc.fitness(np.zeros_like(ref), burned, W, 0)
        assert N == 0 and np.array_equal(score, os_, equal_nan=True)
        L.close()


def test_group_stats_bit_exact(orc):
    rng = np.random.default_rng(4)
    for G, R, N in [(1, 2, 10), (1024, 16, 35785), (33, 50, 2 ** 24), (7, 3, 1)]:
        Ns = rng.integers(0, 2 ** 24, G * R).astype(np.uint32)
        I = (rng.random(G * R) * np.minimum(Ns, N)).astype(np.uint32)
        counts = np.stack([I, Ns], 1)
        sums, mv = gh.group_stats(counts, N, G, R)
        osums, omv = orc.group_stats(counts, N, G, R)
        assert (sums == osums).all() and np.array_equal(mv.view(np.uint64), omv.view(np.uint64))


def test_group_stats_beyond_64_bit_numerators():
    """R sum x^2 - (sum x)^2 beyond 2^64 (x up to 2 W H on an 8192 x 8192 lattice, many replicates): exact Python integers decide."""
    rng = np.random.default_rng(41)
    N = 8192 * 8192 // 2
    for G, R in [(5, 64), (3, 500), (2, 33)]:
        Ns = rng.integers(2 ** 25, 2 ** 26, G * R).astype(np.uint32)
        I = rng.integers(0, 2 ** 10, G * R).astype(np.uint32)
        counts = np.stack([I, Ns], 1)
        sums, mv = gh.group_stats(counts, N, G, R)
        for g in range(G):
            xs = [int(N) + int(Ns[g * R + r]) - 2 * int(I[g * R + r]) for r in range(R)]
            sx, sxx = sum(xs), sum(v * v for v in xs)
            assert int(sums[g, 0]) == sx and int(sums[g, 1]) == sxx
            num = R * sxx - sx * sx
            assert R * sxx >= 2 ** 64 or R == 33              # the 64-bit expression of the terms wraps
            var = num / (R * (R - 1)) / (N * N)
            assert abs(mv[g, 0] - sx / (R * N)) <= 1e-15 * abs(mv[g, 0])
            assert abs(mv[g, 1] - var) <= 1e-14 * var, (g, mv[g, 1], var)


def test_batches_larger_than_a_grid_dimension(orc):
    """S > 65,535 simulations in one call (the paper's Monte Carlo runs 10^6): init / finish kernels must not put S in gridDim.y."""
    rng = np.random.default_rng(17)
    ls = small_landscape(rng, 9, 11)
    S = 70000
    betas = np.array([[-0.4, -0.3, 0.2, 0.8, 0.4]], np.float32)
    ign = np.stack([rng.integers(0, 11, S), rng.integers(0, 9, S)], 1).astype(np.int32)
    seeds = rng.integers(0, 2 ** 63, S).astype(np.uint64)
    L = gh.make_landscape(ls); Lo = orc_landscape(orc, ls)
    gh.upload(L, betas)
    g = gh.simulate(L, ign, np.zeros(S, np.int32), seeds)
    o = orc.simulate_batch(Lo, betas, ign, np.zeros(S, np.int32), seeds, tables=[gh.thresholds(L, 0)])
    assert (g["burned"] == o["burned"]).all() and (g["steps"] == o["steps"]).all() and (g["trials"] == o["trials"]).all()
    # the handle is still usable (no sticky error)
    g2 = gh.simulate(L, ign[:5], np.zeros(5, np.int32), seeds[:5])
    assert (g2["burned"] == o["burned"][:5]).all()
    L.close()


def test_plain_c_program_through_the_abi(tmp_path, request):
    """Config 1 driven by a compiled C program (tests/c/drive_cfg.c: no Python, no ctypes between the caller and the library),
    compared with the oracle's stored digests, steps, trial counts and Eq. 2 counts."""
    import subprocess
    from paper_1701_03549_b200 import build as fire_build
    lib = fire_build.build()
    exe = tmp_path / "drive_cfg"
    cuda = "/usr/local/cuda"
    res = subprocess.run(["gcc", "-std=c99", "-O1", "-I", str(ROOT / "include"), "-I", f"{cuda}/include", str(ROOT / "tests" / "c" / "drive_cfg.c"),
                          str(lib), f"-L{cuda}/lib64", "-lcudart", f"-Wl,-rpath,{lib.parent}", f"-Wl,-rpath,{cuda}/lib64", "-o", str(exe)],
                         capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    w = wl.load_workload(1)
    ls = w.landscape
    H, W = ls["veg"].shape
    Ww = (W + 31) // 32
    with open(tmp_path / "in.bin", "wb") as f:
        f.write(np.array([W, H, w.P, w.S, w.metric], np.int32).tobytes())
        f.write(ls["veg"].astype(np.uint8).tobytes())
        for k in ("slope", "aspect", "wind"):
            f.write(ls[k].astype(np.float32).tobytes())
        f.write(np.vstack([w.betas, w.ref_beta[None, :]]).astype(np.float32).tobytes())
        f.write(w.ignitions.astype(np.int32).tobytes()); f.write(w.sim_param.astype(np.int32).tobytes())
        f.write(w.seeds.astype(np.uint64).tobytes())
        f.write(np.asarray(w.ref_ignition, np.int32).tobytes()); f.write(np.array([w.ref_seed], np.uint64).tobytes())
    res = subprocess.run([str(exe), str(tmp_path / "in.bin"), str(tmp_path / "out.bin")], capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stdout + res.stderr
    raw = (tmp_path / "out.bin").read_bytes()
    S, off = w.S, 0
    def take(dtype, count):
        nonlocal off
        a = np.frombuffer(raw, dtype, count, off); off += a.nbytes
        return a
    burned = take(np.uint32, S * H * Ww).reshape(S, H, Ww); steps = take(np.uint32, S); trials = take(np.uint64, S)
    counts = take(np.uint32, S * 2).reshape(S, 2); score = take(np.float32, S); area = int(take(np.uint32, 1)[0])
    gold = json.loads((GOLDEN / "cfg1_expected.json").read_text())
    assert area == gold["ref_area"]
    assert [gh.digest(burned[s]) for s in range(S)] == gold["digest"]
    assert (steps == np.array(gold["steps"], np.uint32)).all() and (trials == np.array(gold["trials"], np.uint64)).all()
    assert (counts[:, 0] == np.array(gold["intersection"], np.uint32)).all() and (counts[:, 1] == np.array(gold["area"], np.uint32)).all()
    x = area + counts[:, 1].astype(np.int64) - 2 * counts[:, 0].astype(np.int64)
    expect = (x.astype(np.float32) / np.float32(area)) if w.metric == 0 else None
    if expect is not None:
        assert np.array_equal(score.view(np.uint32), expect.view(np.uint32))
    report(request, sims=S, launches=res.stdout.strip())


def test_generation_host_matches_device_path():
    w = wl.load_workload(2)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, np.vstack([w.betas, w.ref_beta[None, :]]))
    ref = gh.simulate(L, [w.ref_ignition], [w.P], [w.ref_seed], sim_ids=[0])["burned"][0]
    gh.upload(L, w.betas)
    g = gh.simulate(L, w.ignitions, w.sim_param, w.seeds, keep_device=True)
    counts, score, N = gh.fitness(L, ref, g["burned"], w.metric)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_score = torch.empty(w.S, dtype=torch.float32).pin_memory()
    h_counts = torch.empty((w.S, 2), dtype=torch.int32).pin_memory()
    h_steps = torch.empty(w.S, dtype=torch.int32).pin_memory()
    ptr = lf.fire_generation_host(L, pin(w.betas), pin(w.ignitions), pin(w.sim_param), pin(w.seeds.view(np.int64)),
                                  pin(ref.view(np.int32)), w.metric, h_score, h_counts, h_steps)
    assert ptr != 0
    assert np.array_equal(h_score.numpy().view(np.uint32), score.view(np.uint32))
    assert (h_counts.numpy().view(np.uint32) == counts).all() and (h_steps.numpy().view(np.uint32) == g["steps"]).all()
    L.close()


def test_errors_are_codes_not_crashes():
    w = wl.load_workload(1)
    L = gh.make_landscape(w.landscape)
    with pytest.raises(lf.FireError) as ei:                                          # simulate before params
        gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    assert ei.value.code == lf.FIRE_ESTATE
    gh.upload(L, w.betas)
    with pytest.raises(lf.FireError) as ei:
        lf.fire_thresholds_download(L, 99, torch.empty((L.H, L.W, 8), dtype=torch.int32, device="cuda"))
    assert ei.value.code == lf.FIRE_ESTATE
    with pytest.raises(lf.FireError) as ei:
        lf.fire_set_launch_geometry(L, 100, 1)
    assert ei.value.code == lf.FIRE_EINVAL
    with pytest.raises(TypeError):
        lf.fire_params_upload(L, torch.zeros((2, 5)))                                # host tensor: there is no CPU path
    assert lf.load().fire_landscape_destroy(None) == lf.FIRE_EINVAL
    L.close()


# ---------------------------------------------------------------------------------- distribution (P-8)
@pytest.mark.parametrize("cfg", [1, 2])
def test_burned_area_distribution_ks(orc, request, cfg):
    """GPU seeds 0..999 vs oracle seeds 1000..1999 at the reference (near-transition) vector: KS p > 0.01."""
    from scipy.stats import ks_2samp
    w = wl.load_workload(cfg)
    Lo = orc_landscape(orc, w.landscape); L = gh.make_landscape(w.landscape)
    gh.upload(L, w.ref_beta[None, :])
    n = 1000
    ign = np.tile(np.array([w.ref_ignition], np.int32), (n, 1)); par = np.zeros(n, np.int32)
    g = gh.simulate(L, ign, par, np.arange(n, dtype=np.uint64))
    o = orc.simulate_batch(Lo, w.ref_beta[None, :], ign, par, np.arange(n, 2 * n, dtype=np.uint64))
    ga, oa = gh.popcount(g["burned"]), gh.popcount(o["burned"])
    ks = ks_2samp(ga, oa)
    report(request, gpu_mean_area=f"{ga.mean():.1f}", oracle_mean_area=f"{oa.mean():.1f}", ks_p=f"{ks.pvalue:.3f}")
    assert ks.pvalue > 0.01
    L.close()


# ---------------------------------------------------------------------------------- search loop on top of the batch API (f1)
def test_evaluator_scores_equal_the_oracle(orc):
    """search.Evaluator is 15 lines of seed / parameter-index / replicate layout on top of the batch API: one population through it
    and through the oracle fed the same (beta, ignition, seeds, sim ids) must give the same mean Eq. 2 fitness per individual."""
    from paper_1701_03549_b200 import search
    w = wl.load_workload(1)
    Lo = orc_landscape(orc, w.landscape)
    L = gh.make_landscape(w.landscape)
    ref_np = orc.simulate(Lo, w.ref_beta, w.ref_ignition, w.ref_seed, sim=0)["burned"]
    ev = search.Evaluator(L, gh.dev(ref_np), tuple(int(v) for v in w.ref_ignition), replicates=3, metric=0, seed=5)
    pop = np.vstack([w.betas[:7], w.ref_beta[None, :]]).astype(np.float64)
    for call in range(2):                                              # the seed carries the call number: check two calls
        got = ev(pop)
        P, R = pop.shape[0], 3
        S = P * R
        seeds = (np.uint64(5) << np.uint64(40)) | (np.uint64(call) << np.uint64(20)) | np.arange(S, dtype=np.uint64)
        o = orc.simulate_batch(Lo, pop.astype(np.float32), np.tile(np.asarray(w.ref_ignition, np.int32), (S, 1)),
                               np.repeat(np.arange(P, dtype=np.int32), R), seeds)
        _, score, _ = orc.fitness(ref_np, o["burned"], Lo.W, 0)
        want = score.astype(np.float64).reshape(P, R).mean(axis=1)
        assert np.array_equal(got, want), (call, got, want)
    L.close()


def test_genetic_algorithm_recovers_a_known_vector(request):
    """SURVEY 8 f1 / PAPER.md App. B, C on config 2: a reference burn is simulated from a KNOWN vector; the stochastic floor of
    Eq. 2 is measured as the paper does (:137: the reference vector itself, other seeds); the GA must bring its best individual
    to within twice that floor, far below the best of the random first generation, and the recovered vector is reported gene by
    gene.  GA-driven and Monte-Carlo-driven simulations are timed (Table 4: the GA's ensemble stays close to
    the real fire, a uniform prior does not, so their per-simulation times differ)."""
    import time
    from paper_1701_03549_b200 import search
    w = wl.load_workload(2)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, w.ref_beta[None, :])
    ref = gh.simulate(L, [w.ref_ignition], [0], [w.ref_seed], sim_ids=np.zeros(1, np.int32), keep_device=True)["burned"][0]
    R = 8
    ev = search.Evaluator(L, ref, tuple(int(v) for v in w.ref_ignition), replicates=R, metric=0, seed=7)
    floor = float(ev(np.repeat(w.ref_beta[None, :].astype(np.float64), 16, axis=0)).mean())      # 128 replicates of the true vector
    lo = np.array([-6.0, -1.0, -0.5, 0.0, 0.0]); hi = np.array([2.0, 0.0, 0.5, 2.0, 1.5])
    assert ((w.ref_beta >= lo) & (w.ref_beta <= hi)).all()
    gens, pop_size = 40, 96
    torch.cuda.synchronize(); t0 = time.perf_counter()
    best, fit, hist = search.genetic_algorithm(ev, lo, hi, pop_size=pop_size, generations=gens, n_elite=2, seed=11)
    torch.cuda.synchronize(); t_ga = time.perf_counter() - t0
    # the best individual re-evaluated on fresh seeds (its GA fitness is the minimum of noisy means, biased low)
    again = float(ev(np.repeat(best[None, :], 16, axis=0)).mean())
    n_mc = gens * pop_size
    torch.cuda.synchronize(); t0 = time.perf_counter()
    samples, fits = search.monte_carlo(ev, lo, hi, n_samples=n_mc, batch=pop_size, seed=12)
    torch.cuda.synchronize(); t_mc = time.perf_counter() - t0
    err = best - w.ref_beta.astype(np.float64)
    report(request, stochastic_floor=f"{floor:.3f}", first_generation_best=f"{hist[0][1]:.3f}", ga_best=f"{fit:.3f}",
           ga_best_on_fresh_seeds=f"{again:.3f}", monte_carlo_best=f"{fits[0]:.3f}",
           beta_hat=np.array2string(best, precision=2), beta_ref=np.array2string(w.ref_beta, precision=2),
           abs_error_per_gene=np.array2string(np.abs(err), precision=2), range_per_gene=np.array2string(hi - lo, precision=1),
           ga_sims_per_s=f"{gens * pop_size * R / t_ga:.0f}", mc_sims_per_s=f"{n_mc * R / t_mc:.0f}",
           ga_over_mc_speed=f"{(gens * pop_size * R / t_ga) / (n_mc * R / t_mc):.2f}")
    assert np.isfinite(fit) and ev.calls == 1 + gens + 1 + n_mc // pop_size
    assert fit <= hist[0][1] and again <= 2.0 * floor, (again, floor)           # calibrated down to the stochastic floor (x2)
    assert again < 0.5 * hist[0][2]                                             # far below the mean of a random population
    assert (best >= lo).all() and (best <= hi).all()
    # the GA's answer is at least as good as brute force with the same number of simulations
    assert fit <= fits[0] + 0.5 * floor
    L.close()


def test_unknown_ignition_search_as_the_paper_runs_it(request):
    """SURVEY 8 f2 / PAPER.md:97, :177, :360: seven genes (beta_0..4, x, y), candidates for (x, y) drawn inside the reference
    scar; the estimate and its spread come from the ensemble below a fitness cutoff and, for the final
    population, from the per-candidate statistics of fire_fitness_group_stats (a8)."""
    from paper_1701_03549_b200 import search
    w = wl.load_workload(2)
    L = gh.make_landscape(w.landscape)
    gh.upload(L, w.ref_beta[None, :])
    ref_t = gh.simulate(L, [w.ref_ignition], [0], [w.ref_seed], sim_ids=np.zeros(1, np.int32), keep_device=True)["burned"][0]
    ref_np = ref_t.cpu().numpy().view(np.uint32)
    scar = search.scar_cells(ref_np, L.W)
    R = 8
    ev = search.IgnitionEvaluator(L, ref_t, replicates=R, metric=0, seed=9)
    lo = np.array([-6.0, -1.0, -0.5, 0.0, 0.0, 0.0, 0.0]); hi = np.array([2.0, 0.0, 0.5, 2.0, 1.5, L.W - 1.0, L.H - 1.0])
    rng = np.random.default_rng(21)
    init = search.initial_population_with_ignition(rng, lo, hi, scar, 128)
    arch = []
    best, fit, hist = search.genetic_algorithm(ev, lo, hi, generations=40, n_elite=2, seed=22, init=init, archive=arch)
    inds = np.concatenate([a for a, _ in arch]); fits = np.concatenate([f for _, f in arch])
    floor = float(ev(np.repeat(np.concatenate([w.ref_beta.astype(np.float64), np.asarray(w.ref_ignition, np.float64)])[None, :], 16, axis=0)).mean())
    cutoff = max(1.25 * fit, min(1.0, 1.1 * floor))
    b, mean, sd, n = search.ensemble_estimate(inds, fits, cutoff)
    true_xy = np.asarray(w.ref_ignition, np.float64)
    d_best = float(np.hypot(*(np.rint(best[5:7]) - true_xy)))
    d_rand = float(np.hypot(*(scar - true_xy).T).mean())                # what a random scar cell would give
    # per-candidate mean and variance of delta for the final population, on the device (a8)
    final = arch[-1][0]
    _ = ev(final)
    N = int(gh.popcount(ref_np[None])[0])
    sums, mv = gh.group_stats(ev.last_counts.cpu().numpy().view(np.uint32), N, final.shape[0], R)
    k = int(np.argmin(mv[:, 0]))
    report(request, floor=f"{floor:.3f}", best_fitness=f"{fit:.3f}", best_ignition=np.rint(best[5:7]).astype(int).tolist(),
           true_ignition=list(w.ref_ignition), distance_cells=f"{d_best:.1f}", random_scar_cell_distance=f"{d_rand:.1f}",
           ensemble=n, cutoff=f"{cutoff:.3f}", ignition_mean=np.array2string(mean[5:7], precision=1),
           ignition_sd=np.array2string(sd[5:7], precision=1), beta_mean=np.array2string(mean[:5], precision=2),
           beta_sd=np.array2string(sd[:5], precision=2), beta_ref=np.array2string(w.ref_beta, precision=2),
           best_candidate_mean_delta=f"{mv[k, 0]:.3f}", best_candidate_sd_delta=f"{np.sqrt(mv[k, 1]):.3f}")
    assert np.isfinite(fit) and fit <= hist[0][1] and fit < 1.0 and n >= 2
    assert d_best < d_rand, (d_best, d_rand)                          # the search locates the ignition better than chance inside the scar
    assert (mv[:, 1] >= 0).all() and np.isfinite(mv).all()
    L.close()


def test_burn_out_time_variant_matches_the_oracle(orc, request):
    """fuel-dependent burn-out times 1..8 per vegetation class.  Random lattices, burn-time
    tables, step limits, CTA sizes, list capacities (down to the global spill and the rescue kernel of this variant); the oracle
    is fed the GPU's own threshold tables, so burnt maps, steps and trial counts must be bit-exact.  Setting all ones afterwards
    is the base model again."""
    rng = np.random.default_rng(20261105)
    n = 0
    for it in range(40):
        H, W = int(rng.integers(1, 120)), int(rng.integers(1, 160))
        ls = small_landscape(rng, H, W, nonburn=0.15)
        P, S = int(rng.integers(1, 4)), int(rng.integers(1, 30))
        betas = np.stack([[rng.uniform(-3.0, 0.0), rng.uniform(-1, 0), rng.uniform(-.5, .5), rng.uniform(0, 2), rng.uniform(0, 1.5)]
                          for _ in range(P)]).astype(np.float32)
        ign = np.stack([rng.integers(-1, W + 1, S), rng.integers(-1, H + 1, S)], 1).astype(np.int32)
        par = rng.integers(0, P, S).astype(np.int32)
        seeds = rng.integers(0, 2 ** 63, S).astype(np.uint64)
        max_steps = int(rng.choice([0, 0, 0, 4, 23]))
        bt = [1] + [int(v) for v in rng.integers(1, 9, 3)]
        if it % 7 == 0:
            bt = [1, 8, 1, 2]
        geom = (int(rng.choice([32, 64, 128, 256, 512, 1024])), int(rng.integers(1, 5)))
        caps = (int(rng.choice([0, 0, 1, 4, 16])), int(rng.choice([0, 0, 0, 2, 64])))
        Lo = orc_landscape(orc, ls)
        L = gh.make_landscape(ls)
        gh.upload(L, betas)
        tables = [gh.thresholds(L, p) for p in range(P)]
        lf.fire_set_launch_geometry(L, *geom)
        lf.fire_set_list_capacity(L, *caps)
        lf.fire_set_kernel(L, int(rng.choice([0, 1, 2])))             # the variant runs on the two-phase kernel whatever is asked
        lf.fire_set_burn_time(L, bt)
        g = gh.simulate(L, ign, par, seeds, max_steps=max_steps)
        what = (it, H, W, P, S, max_steps, bt, geom, caps)
        for s_ in range(S):
            if 0 <= par[s_] < P:
                o = orc.simulate_burn_time(Lo, betas[par[s_]], bt, ign[s_], int(seeds[s_]), sim=s_, max_steps=max_steps, table=tables[par[s_]])
                assert (g["burned"][s_] == o["burned"]).all(), (what, s_)
                assert g["steps"][s_] == o["steps"] and int(g["trials"][s_]) == o["trials"], (what, s_, g["steps"][s_], o["steps"])
        if it % 5 == 0:                                               # back to one step everywhere: the base model, bit for bit
            lf.fire_set_burn_time(L, [1, 1, 1, 1])
            g1 = gh.simulate(L, ign, par, seeds, max_steps=max_steps)
            o1 = orc.simulate_batch(Lo, betas, ign, par, seeds, max_steps=max_steps, tables=tables)
            assert (g1["burned"] == o1["burned"]).all() and (g1["steps"] == o1["steps"]).all() and (g1["trials"] == o1["trials"]).all(), what
        n += 1
        L.close()
    # config 2 at full size with burn times (forest 3 steps, the other classes 1-2): every sim against the oracle's own thresholds
    w = wl.load_workload(2)
    Lo = orc_landscape(orc, w.landscape); L = gh.make_landscape(w.landscape)
    gh.upload(L, w.betas)
    bt = [1, 3, 2, 1]
    lf.fire_set_burn_time(L, bt)
    g = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    idx = np.arange(0, w.S, 8)
    for s_ in idx:
        o = orc.simulate_burn_time(Lo, w.betas[w.sim_param[s_]], bt, w.ignitions[s_], int(w.seeds[s_]), sim=int(s_))
        assert (g["burned"][s_] == o["burned"]).all() and g["steps"][s_] == o["steps"] and int(g["trials"][s_]) == o["trials"], s_
    report(request, cases=n, cfg2_sims_checked=len(idx), cfg2_trials=int(g["trials"].sum()))
    L.close()


def test_dem_uphill_variant_and_hazard_map(orc, request):
    """(i) the literal DEM uphill test of PAPER.md:87 (fire_landscape_set_elevation) -- thresholds within one count of
    the oracle's table, propagation bit-exact on the GPU's table; (ii) the hazard map of PAPER.md:54 (fire_burn_count) equals the
    per-cell sum over the burnt maps, including a ragged width and more maps than one slab."""
    rng = np.random.default_rng(77)
    n_diff = 0
    for H, W in [(40, 50), (33, 77), (64, 64)]:
        ls = small_landscape(rng, H, W)
        z = (np.cumsum(rng.standard_normal((H, W)), axis=1) * 5 + 200).astype(np.float32)
        betas = np.array([[-0.8, -0.4, 0.3, 0.9, 1.2], [-1.5, 0.2, -0.1, 1.4, 0.4]], np.float32)
        Lo = orc_landscape(orc, ls); L = gh.make_landscape(ls)
        lf.fire_landscape_set_elevation(L, gh.dev(z))
        gh.upload(L, betas)
        tabs = []
        for p in range(2):
            g = gh.thresholds(L, p); o = orc.threshold_table_dem(Lo, betas[p], z)
            # entries whose source lies outside the lattice are never tried: the test hook evaluates them with sigma = 0 as well
            d = np.abs(g.astype(np.int64) - o.astype(np.int64))
            assert d.max() <= 1, (H, W, p, d.max())
            n_diff += int((d != 0).sum()); tabs.append(g)
        base = orc.threshold_table(Lo, betas[0])
        assert (tabs[0] != base).any()                                # the variant really changes the table
        S = 150
        ign = np.stack([rng.integers(0, W, S), rng.integers(0, H, S)], 1).astype(np.int32)
        par = rng.integers(0, 2, S).astype(np.int32); seeds = rng.integers(0, 2 ** 63, S).astype(np.uint64)
        g = gh.simulate(L, ign, par, seeds, keep_device=True)
        o = orc.simulate_batch(Lo, betas, ign, par, seeds, tables=tabs)
        gb = g["burned"].cpu().numpy().view(np.uint32)
        assert (gb == o["burned"]).all() and (g["steps"] == o["steps"]).all() and (g["trials"] == o["trials"]).all()
        count = torch.full((H, W), -1, dtype=torch.int32, device="cuda")
        lf.fire_burn_count(L, g["burned"], count)
        torch.cuda.synchronize()
        assert (count.cpu().numpy().view(np.uint32) == orc.burn_count(o["burned"], W)).all()
        L.close()
    report(request, one_count_differences=n_diff)


def test_time_of_burn_output(orc, request):
    """the step at which every cell ignites (fire_set_time_output) against the oracle's out_time (pinned on the CPU by
    BFS depth), with and without burn-out times, through the list spill and the rescue kernel; switching it off restores the
    default path."""
    rng = np.random.default_rng(91)
    n = 0
    for it in range(16):
        H, W = int(rng.integers(2, 90)), int(rng.integers(2, 120))
        ls = small_landscape(rng, H, W, nonburn=0.15)
        S = int(rng.integers(1, 12))
        betas = np.array([[rng.uniform(-2.0, 0.5), -0.4, 0.2, 0.9, 0.6]], np.float32)
        ign = np.stack([rng.integers(0, W, S), rng.integers(0, H, S)], 1).astype(np.int32)
        seeds = rng.integers(0, 2 ** 63, S).astype(np.uint64)
        bt = [1, 1, 1, 1] if it % 2 == 0 else [1] + [int(v) for v in rng.integers(1, 5, 3)]
        max_steps = int(rng.choice([0, 0, 9]))
        Lo = orc_landscape(orc, ls); L = gh.make_landscape(ls)
        gh.upload(L, betas)
        tab = gh.thresholds(L, 0)
        lf.fire_set_launch_geometry(L, int(rng.choice([64, 256, 1024])), 1)
        lf.fire_set_list_capacity(L, int(rng.choice([0, 2, 16])), int(rng.choice([0, 0, 3])))
        lf.fire_set_burn_time(L, bt)
        times = torch.full((S, H, W), 12345, dtype=torch.int32, device="cuda")
        lf.fire_set_time_output(L, times)
        g = gh.simulate(L, ign, np.zeros(S, np.int32), seeds, max_steps=max_steps)
        tg = times.cpu().numpy()
        for s_ in range(S):
            o = orc.simulate_burn_time(Lo, betas[0], bt, ign[s_], int(seeds[s_]), sim=s_, max_steps=max_steps, table=tab, want_time=True)
            assert (g["burned"][s_] == o["burned"]).all() and g["steps"][s_] == o["steps"], (it, s_)
            assert (tg[s_] == o["time"]).all(), (it, s_, np.argwhere(tg[s_] != o["time"])[:5])
        lf.fire_set_time_output(L, None)
        lf.fire_set_burn_time(L, None)
        g0 = gh.simulate(L, ign, np.zeros(S, np.int32), seeds, max_steps=max_steps)
        o0 = orc.simulate_batch(Lo, betas, ign, np.zeros(S, np.int32), seeds, max_steps=max_steps, tables=[tab])
        assert (g0["burned"] == o0["burned"]).all() and (g0["steps"] == o0["steps"]).all()
        n += 1
        L.close()
    report(request, cases=n)


def test_fused_fitness_counts(orc, request):
    """Eq. 2's counts (I, N*) written by fire_simulate_batch itself (fire_set_fused_counts) equal the oracle's counts
    of the same maps -- on every kernel family, through the list spill, the rescue kernel (which overwrites the counts of the
    simulations it redoes) and the burn-out variant; the maps themselves are unchanged and switching it off stops the writes."""
    w = wl.load_workload(2)
    ls = w.landscape
    L = gh.make_landscape(ls)
    gh.upload(L, w.betas)
    Lo = orc_landscape(orc, ls)
    ref = orc.simulate(Lo, w.ref_beta, w.ref_ignition, w.ref_seed, sim=0)["burned"]
    base = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    oc, _, _ = orc.fitness(ref, base["burned"], Lo.W, 0)
    ref_d = torch.from_numpy(ref.view(np.int32)).cuda()
    n = 0
    for threads, per_sm, shared, total, family, bt in [(0, 0, 0, 0, 0, None), (256, 4, 8, 8, 1, None), (128, 4, 1, 1, 2, None),
                                                       (1024, 1, 0, 0, 3, None), (256, 2, 5, 4096, 4, None), (64, 3, 2, 3, 0, None),
                                                       (0, 0, 0, 0, 0, [1, 1, 1, 1]), (256, 4, 2, 3, 0, [1, 3, 2, 4])]:
        counts = torch.full((w.S + 3, 2), 77, dtype=torch.int32, device="cuda")
        lf.fire_set_launch_geometry(L, threads, per_sm)
        lf.fire_set_list_capacity(L, shared, total)
        lf.fire_set_kernel(L, family)
        lf.fire_set_burn_time(L, bt)
        lf.fire_set_fused_counts(L, ref_d, counts)
        g = gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
        got = counts.cpu().numpy().view(np.uint32)
        if bt is None or max(bt) == 1:
            assert (g["burned"] == base["burned"]).all()
            want = oc
        else:
            want, _, _ = orc.fitness(ref, g["burned"], Lo.W, 0)
        assert (got[: w.S] == want).all(), (threads, per_sm, shared, total, family, bt, np.flatnonzero((got[: w.S] != want).any(axis=1))[:8])
        assert (got[w.S:] == 77).all()                                   # nothing past the batch is touched
        c2, _, _ = gh.fitness(L, ref, g["burned"], 0)
        assert (c2 == want).all()
        n += 1
    lf.fire_set_fused_counts(L, None, None)
    lf.fire_set_burn_time(L, None)
    counts.fill_(55)
    gh.simulate(L, w.ignitions, w.sim_param, w.seeds)
    assert (counts.cpu().numpy() == 55).all()
    with pytest.raises(TypeError):
        lf.fire_set_fused_counts(L, ref_d, None)
    L.close()
    report(request, cases=n)


# ---------------------------------------------------------------------------------- randomised parity
def test_random_lattices_geometries_and_kernels_match_the_oracle(orc, request):
    """Seeded fuzz: random lattice sizes (1 x 1 .. 140 x 200, ragged), vegetation, parameters, ignitions (some off the lattice
    or on non-burnable cells), step limits, CTA sizes, residencies, list capacities, launch orders, both kernel families and cluster sizes.
    The oracle is fed the GPU's own threshold tables, so burned maps, steps and trial counts must be bit-exact."""
    rng = np.random.default_rng(20260604)
    n = 0
    for it in range(60):
        H, W = int(rng.integers(1, 140)), int(rng.integers(1, 200))
        ls = {"veg": rng.choice(4, (H, W), p=[.15, .3, .3, .25]).astype(np.uint8),
              "slope": (rng.random((H, W)) * 0.6).astype(np.float32),
              "aspect": (rng.random((H, W)) * 2 * np.pi).astype(np.float32),
              "wind": (rng.random((H, W)) * 2 * np.pi).astype(np.float32)}
        P, S = int(rng.integers(1, 5)), int(rng.integers(1, 40))
        betas = np.stack([[rng.uniform(-2, 1.5), rng.uniform(-1, 0), rng.uniform(-.5, .5), rng.uniform(0, 2), rng.uniform(0, 1.5)]
                          for _ in range(P)]).astype(np.float32)
        ign = np.stack([rng.integers(-1, W + 1, S), rng.integers(-1, H + 1, S)], 1).astype(np.int32)
        par = rng.integers(0, P, S).astype(np.int32)
        seeds = rng.integers(0, 2 ** 63, S).astype(np.uint64)
        max_steps = int(rng.choice([0, 0, 0, 3, 17]))
        geom = (int(rng.choice([32, 64, 96, 128, 256, 512, 1024])), int(rng.integers(1, 9)))
        caps = (int(rng.choice([0, 0, 1, 4, 16])), int(rng.choice([0, 0, 0, 2, 64])))
        order, family = int(rng.integers(0, 2)), int(rng.choice([0, 1, 2, 3, 4]))
        mode = (order, family)
        Lo = orc_landscape(orc, ls)
        L = gh.make_landscape(ls)
        gh.upload(L, betas)
        tables = [gh.thresholds(L, p) for p in range(P)]
        o = orc.simulate_batch(Lo, betas, ign, par, seeds, max_steps=max_steps, tables=tables)
        lf.fire_set_launch_geometry(L, *geom)
        lf.fire_set_list_capacity(L, *caps)
        lf.fire_set_schedule(L, order)
        lf.fire_set_kernel(L, family)
        g = gh.simulate(L, ign, par, seeds, max_steps=max_steps)
        what = (it, H, W, P, S, max_steps, geom, caps, mode)
        assert (g["burned"] == o["burned"]).all(), what
        assert (g["steps"] == o["steps"]).all() and (g["trials"] == o["trials"]).all(), what
        n += 1
        L.close()
    report(request, cases=n)
