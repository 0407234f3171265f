"""`-m "not gpu"`: pins of the oracle's f4 variants: the literal DEM uphill test of PAPER.md:87 and the hazard map."""
import numpy as np

from conftest import OFFSETS, pack_bitmap


def test_dem_uphill_on_a_plane_equals_the_aspect_rule(orc):
    """On a planar DEM the slope faces one bearing everywhere: "target higher than source" <=> travelling against that bearing,
    which is R-7's test cos(phi_d - aspect) < 0 -- except along contour lines, where the plane gives a tie (not uphill) and the
    cosine an exact or rounded zero.  Entries whose source lies outside the lattice get sigma = 0."""
    H, W = 12, 14
    rng = np.random.default_rng(3)
    for gx, gy in [(0.7, 0.0), (0.0, -0.5), (0.4, 0.9), (-0.8, 0.3)]:            # dz/dx (east), dz/dy (south), per cell
        ys, xs = np.mgrid[0:H, 0:W]
        z = (gx * xs + gy * ys).astype(np.float32) * 30.0
        aspect = np.float32(np.mod(np.arctan2(-gx, gy), 2 * np.pi))              # downslope bearing (R-4, R-5)
        slope = np.float32(np.arctan(np.hypot(gx, gy)))
        ls = {"veg": rng.integers(1, 4, (H, W)).astype(np.uint8), "slope": np.full((H, W), slope, np.float32),
              "aspect": np.full((H, W), aspect, np.float32), "wind": rng.uniform(0, 6.28, (H, W)).astype(np.float32)}
        L = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
        beta = np.array([-0.7, -0.3, 0.2, 0.6, 1.3], np.float32)
        a = orc.threshold_table(L, beta)
        b = orc.threshold_table_dem(L, beta, z)
        for d, (dx, dy) in enumerate(OFFSETS):
            rise = gx * dx + gy * dy                                              # elevation gained travelling in direction d
            inside = np.zeros((H, W), bool)
            inside[max(dy, 0):H + min(dy, 0), max(dx, 0):W + min(dx, 0)] = True   # source = target - offset inside the lattice
            if abs(rise) > 1e-6:
                assert (a[..., d][inside] == b[..., d][inside]).all(), (gx, gy, d)
            flat = orc.threshold_table(L, np.array([-0.7, -0.3, 0.2, 0.6, 0.0], np.float32))
            assert (b[..., d][~inside] == flat[..., d][~inside]).all()            # no source, no slope term
            if rise <= 0:
                assert (b[..., d] == flat[..., d]).all()                          # level or downhill: sigma ignored
            else:
                assert (b[..., d][inside] > flat[..., d][inside]).all()           # uphill with beta_4 > 0: more likely


def test_dem_uphill_flat_or_zero_slope_ignores_sigma(orc):
    rng = np.random.default_rng(4)
    H, W = 9, 10
    ls = {"veg": rng.integers(0, 4, (H, W)).astype(np.uint8), "slope": rng.uniform(0, 0.5, (H, W)).astype(np.float32),
          "aspect": rng.uniform(0, 6.28, (H, W)).astype(np.float32), "wind": rng.uniform(0, 6.28, (H, W)).astype(np.float32)}
    L = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    beta = np.array([-0.5, -0.3, 0.2, 0.6, 1.1], np.float32); beta0 = beta.copy(); beta0[4] = 0
    assert (orc.threshold_table_dem(L, beta, np.full((H, W), 123.0, np.float32)) == orc.threshold_table(L, beta0)).all()
    ls["slope"][:] = 0
    L0 = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    z = rng.uniform(0, 100, (H, W)).astype(np.float32)
    assert (orc.threshold_table_dem(L0, beta, z) == orc.threshold_table(L0, beta0)).all()
    assert (orc.threshold_table_dem(L, beta, z)[ls["veg"] == 0] == 0).all()


def test_burn_count_is_the_per_cell_sum(orc):
    rng = np.random.default_rng(5)
    S, H, W = 37, 6, 45
    masks = rng.random((S, H, W)) < 0.3
    packed = np.stack([pack_bitmap(m) for m in masks])
    got = orc.burn_count(packed, W)
    want = np.zeros((H, W), np.uint32)
    for s in range(S):
        for y in range(H):
            for x in range(W):
                want[y, x] += int(masks[s, y, x])
    assert (got == want).all() and got.dtype == np.uint32


def test_class_indicator_table(orc):
    """Per-class vegetation term: the paper's indicator is the table (0, 1, 0, 0, ...); a zero table is beta_1 = 0; a table that is c
    on every burnable class shifts beta_0 by c beta_1 (when that sum is exact in double)."""
    rng = np.random.default_rng(6)
    H, W = 11, 13
    ls = {"veg": rng.integers(0, 5, (H, W)).astype(np.uint8), "slope": rng.uniform(0, 0.5, (H, W)).astype(np.float32),
          "aspect": rng.uniform(0, 6.28, (H, W)).astype(np.float32), "wind": rng.uniform(0, 6.28, (H, W)).astype(np.float32)}
    L = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    beta = np.array([-0.75, -0.5, 0.2, 0.6, 0.4], np.float32)
    assert (orc.threshold_table_classes(L, beta, [0, 1, 0, 0, 0]) == orc.threshold_table(L, beta)).all()
    b_no = beta.copy(); b_no[1] = 0
    assert (orc.threshold_table_classes(L, beta, [0, 0, 0, 0, 0]) == orc.threshold_table(L, b_no)).all()
    b_shift = b_no.copy(); b_shift[0] = np.float32(-0.75 + 2.0 * -0.5)             # exact: -1.75
    assert (orc.threshold_table_classes(L, beta, [0, 2, 2, 2, 2]) == orc.threshold_table(L, b_shift)).all()
    t = orc.threshold_table_classes(L, beta, [0, 1, 0.5, 0.25, 0])
    base = orc.threshold_table(L, b_no)
    for v, sign in [(1, -1), (2, -1), (3, -1), (4, 0)]:                          # beta_1 < 0: a positive I_f lowers the probability
        sel = ls["veg"] == v
        if sel.any():
            assert ((t[sel] < base[sel]).all() if sign < 0 else (t[sel] == base[sel]).all()), v
    assert (t[ls["veg"] == 0] == 0).all()
