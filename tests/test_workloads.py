"""Host logic: synthetic generators, stored recipes, sim layout, sharding (no method arithmetic here)."""
import json

import numpy as np
import pytest

from conftest import GOLDEN
from paper_1701_03549_b200 import workloads as wl


@pytest.mark.parametrize("cfg", [1, 2, 4])
def test_landscape_is_deterministic_and_well_formed(cfg):
    a = wl.make_landscape(cfg); b = wl.make_landscape(cfg)
    c = wl.CONFIGS[cfg]
    for k in ("veg", "slope", "aspect", "wind"):
        assert a[k].shape == (c["H"], c["W"]) and (a[k] == b[k]).all()
    assert a["veg"].dtype == np.uint8 and a["slope"].dtype == np.float32
    wl.validate_landscape(a)
    assert ((a["aspect"] >= 0) & (a["aspect"] < 2 * np.pi + 1e-6)).all()
    frac0 = (a["veg"] == 0).mean()
    assert 0.07 < frac0 < 0.13 and a["veg"].max() == 3                 # iid 4 classes, 10 % non-burnable
    assert a["veg"][c["H"] // 2, c["W"] // 2] != 0
    if c["wind"] == "const":
        assert (a["wind"] == np.float32(np.pi / 4)).all()              # uniform 45 deg
    else:
        assert abs(a["wind"].mean() - 1.5 * np.pi) < 0.2 and np.ptp(a["wind"]) <= np.pi / 3 + 1e-5


def test_clustered_landscape_small_instance():
    a = wl.make_landscape(3, size=256)
    assert a["veg"].max() == 5 and 0.03 < (a["veg"] == 0).mean() < 0.07
    from scipy import ndimage
    _, n = ndimage.label(a["veg"] == 0)
    assert n < 0.02 * (a["veg"] == 0).sum()                            # patches, not salt-and-pepper


def test_aspect_points_downslope():
    a = wl.make_landscape(2)
    # rebuild elevation the same way and check that walking along the aspect bearing descends
    n = wl._noise((256, 256), 8.0, 1002); z = (n - n.min()) / (n.max() - n.min()) * 1500.0
    ys, xs = np.mgrid[8:248:16, 8:248:16]
    asp = a["aspect"][ys, xs]
    step_e, step_n = np.sin(asp), np.cos(asp)
    from scipy.ndimage import map_coordinates
    z1 = map_coordinates(z, [ys - 0.5 * step_n, xs + 0.5 * step_e], order=1)    # north = decreasing row
    steep = a["slope"][ys, xs] > 0.05
    assert (z1[steep] < z[ys, xs][steep]).mean() > 0.98


def test_validate_rejects_bad_rasters():
    a = wl.make_landscape(1)
    bad = dict(a); bad["slope"] = a["slope"].copy(); bad["slope"][0, 0] = np.nan
    with pytest.raises(ValueError):
        wl.validate_landscape(bad)
    bad["slope"][0, 0] = 1.6
    with pytest.raises(ValueError):
        wl.validate_landscape(bad)


@pytest.mark.parametrize("cfg,S,P", [(1, 64, 16), (2, 256, 64), (3, 2048, 256), (4, 16384, 1), (5, 64, 16)])
def test_sim_layout(cfg, S, P):
    r = wl.load_recipe(cfg)
    betas = wl.f32_from_bits(r["betas_f32_bits"]).reshape(-1, 5)
    assert betas.shape == (P, 5)
    assert np.allclose(betas, np.array(r["betas_readable"], np.float32))
    ign, sp, seeds, groups = wl.sim_layout(cfg, P, r)
    assert ign.shape == (S, 2) and sp.shape == (S,) and seeds.shape == (S,)
    assert (np.diff(sp) >= 0).all() and sp.min() == 0 and sp.max() == P - 1      # param-major
    assert (seeds == ((cfg << 32) | np.arange(S))).all() and seeds.dtype == np.uint64
    c = wl.CONFIGS[cfg]
    assert ((ign >= 0) & (ign < [c["W"], c["H"]])).all()
    if cfg == 4:
        assert groups == (1024, 16) and len({tuple(i) for i in ign}) == 1024
        x0, y0, x1, y1 = r["meta"]["ref_bbox"]
        assert ((ign[:, 0] >= x0) & (ign[:, 0] <= x1) & (ign[:, 1] >= y0) & (ign[:, 1] <= y1)).all()
    if cfg == 5:
        assert len({tuple(i) for i in ign}) == 4 and (ign >= 512).all() and (ign < 4096 - 512).all()


def test_golden_expected_files_are_consistent():
    for cfg in (1, 2, 3, 4, 5):
        e = json.loads((GOLDEN / f"cfg{cfg}_expected.json").read_text())
        S = e["S"]
        for k in ("steps", "area", "trials", "cand_steps", "distinct", "intersection", "digest"):
            assert len(e[k]) == S
        assert e["totals"]["trials"] == sum(e["trials"])
        a = np.array(e["area"]); t = np.array(e["trials"]); st = np.array(e["steps"])
        assert (st <= np.maximum(a, 1)).all() and (np.array(e["intersection"]) <= a).all()
        assert (np.array(e["distinct"]) <= np.array(e["cand_steps"])).all() and (np.array(e["cand_steps"]) <= t).all()


def test_shard_sims_partitions_the_batch():
    for S in (1, 7, 64, 2048, 16384):
        for world in (1, 2, 3, 8):
            parts = [wl.shard_sims(S, r, world) for r in range(world)]
            idx = np.concatenate([np.arange(S)[p] for p in parts])
            assert (idx == np.arange(S)).all()
            sizes = [p.stop - p.start for p in parts]
            assert max(sizes) - min(sizes) <= 1
