"""Pins for the oracle's random stream (C-1) and contagion thresholds (C-2, C-3, Eq. 1)."""
import math

import numpy as np
import pytest
from scipy.special import expit

from conftest import GOLDEN, OFFSETS

REF_BETA = (-5.0, -10.0, 5.0, 18.1, -5.0)      # PAPER.md:184-188, Table 2


# ------------------------------------------------------------------ Philox4x32-10
def test_philox_known_answers(orc):
    rows = [l.split() for l in (GOLDEN / "philox4x32_10_kat.txt").read_text().splitlines()
            if l and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(h, 16) for h in r]
        out = orc.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_rnd_keying_uses_all_five_fields(orc):
    """north_star: keyed by (seed, sim, step, cell, direction) -- changing any field changes the word,
    and the 8 directions of one cell come from two Philox blocks (d>>2) x four words (d&3)."""
    base = dict(seed=(7 << 32) | 5, sim=3, step=11, cell=1234)
    words = [orc.rnd(d=d, **base) for d in range(8)]
    assert len(set(words)) == 8
    lo = orc.philox4x32_10([1234, 11, 3, 0], [5, 7])
    hi = orc.philox4x32_10([1234, 11, 3, 1], [5, 7])
    assert words == [int(x) for x in lo] + [int(x) for x in hi]
    for k, v in (("seed", base["seed"] + 1), ("seed", base["seed"] + (1 << 32)), ("sim", 4), ("step", 12),
                 ("cell", 1235)):
        other = dict(base); other[k] = v
        assert [orc.rnd(d=d, **other) for d in range(8)] != words


def test_rnd_uniform_and_uncorrelated(orc):
    """PAPER.md:141 'uncorrelated and uniform': chi^2 on the top byte; neighbouring cells/steps/dirs uncorrelated."""
    from scipy.stats import chisquare
    n = 40000
    w = np.array([orc.rnd(99, 1, s, c, d) for s in range(10) for c in range(n // 80) for d in range(8)], np.uint64)
    _, p = chisquare(np.bincount((w >> np.uint64(24)).astype(int), minlength=256))
    assert p > 1e-3
    u = w.astype(np.float64) / 2.0**32
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 0.02
    assert abs(u.mean() - 0.5) < 0.01


# ------------------------------------------------------------------ geometry (R-4 .. R-8)
def test_direction_offsets_are_compass_bearings(orc):
    for d in range(8):
        dx, dy = orc.direction_offset(d)
        assert (dx, dy) == OFFSETS[d]
        bearing = math.atan2(dx, -dy) % (2 * math.pi)          # row 0 = north, x = east (R-5)
        assert bearing == pytest.approx(d * math.pi / 4)


def test_omega_is_one_downwind_minus_one_upwind(orc):
    """omega = 1 if the target is downwind from the ignited cell, -1 if upwind."""
    for d in range(8):
        c = orc.covariates(2, 0.0, 0.0, d * math.pi / 4)       # wind blows toward bearing d*45 deg
        assert c["omega"][d] == pytest.approx(1.0, abs=1e-6)
        assert c["omega"][(d + 4) % 8] == pytest.approx(-1.0, abs=1e-6)
        assert c["omega"][(d + 2) % 8] == pytest.approx(0.0, abs=1e-6)


def test_psi_is_one_facing_nw_minus_one_facing_se(orc):
    """relative aspect 1 for NW-facing sites, -1 for SE-facing, only above 5 degrees."""
    steep, flat = math.radians(10), math.radians(4.9)
    assert orc.covariates(2, steep, math.radians(315), 0)["psi"] == pytest.approx(1.0, abs=1e-6)
    assert orc.covariates(2, steep, math.radians(135), 0)["psi"] == pytest.approx(-1.0, abs=1e-6)
    assert orc.covariates(2, steep, math.radians(45), 0)["psi"] == pytest.approx(0.0, abs=1e-6)
    assert orc.covariates(2, flat, math.radians(315), 0)["psi"] == 0.0
    assert orc.covariates(2, math.radians(5.1), math.radians(315), 0)["psi"] > 0.99


def test_sigma_only_when_target_is_higher_on_a_plane(orc):
    """slope used only when the target is higher than the burning cell.  Independent check
    against an explicit planar DEM whose downslope bearing is the aspect (R-7)."""
    rng = np.random.default_rng(1)
    for _ in range(200):
        a = rng.uniform(0, 2 * math.pi); s = rng.uniform(0.01, 1.2)
        c = orc.covariates(2, s, a, 0.0)
        for d, (dx, dy) in enumerate(OFFSETS):
            east, north = dx, -dy
            # plane falling toward bearing a: z = -tan(s) * (east*sin a + north*cos a)
            dz = -math.tan(s) * (east * math.sin(a) + north * math.cos(a))
            if abs(dz) < 1e-9:
                continue
            if dz > 0:
                assert c["sigma"][d] == pytest.approx(math.tan(np.float32(s)), rel=1e-12)   # = slope% / 100
            else:
                assert c["sigma"][d] == 0.0
    assert (orc.covariates(2, 0.0, 1.0, 0.0)["sigma"] == 0).all()       # slope zero -> ignored


def test_vegetation_classes(orc):
    """0 non burnable, 1 forest, 2 shrubland; R-9: classes >= 2 burn with I_f = 0."""
    assert not orc.covariates(0, 0, 0, 0)["burnable"]
    assert orc.covariates(1, 0, 0, 0)["I_f"] == 1.0
    for v in (2, 3, 4, 5, 255):
        c = orc.covariates(v, 0, 0, 0)
        assert c["burnable"] and c["I_f"] == 0.0
    b = (0.3, -1.5, 0, 0, 0)
    assert orc.probability(b, 1, 0, 0, 0, 0) == pytest.approx(expit(0.3 - 1.5))
    assert orc.probability(b, 3, 0, 0, 0, 0) == pytest.approx(expit(np.float32(0.3)))
    assert orc.threshold(b, 0, 0, 0, 0, 0) == 0


# ------------------------------------------------------------------ thresholds: closed forms
def test_threshold_closed_forms(orc):
    assert orc.threshold((0, 0, 0, 0, 0), 2, 0.3, 1.0, 2.0, 3) == 2**31            # p = 1/2 exactly
    prev = -1
    for x in np.linspace(-30, 30, 241):
        b = (np.float32(x), 0, 0, 0, 0)
        T = orc.threshold(b, 2, 0, 0, 0, 0)
        Tm = orc.threshold((-np.float32(x), 0, 0, 0, 0), 2, 0, 0, 0, 0)
        assert T >= prev; prev = T                                                  # monotone in x
        if 0 < T < 0xFFFFFFFF or 0 < Tm < 0xFFFFFFFF:
            assert abs(T + Tm - 2**32) <= 1                                         # p(x) + p(-x) = 1
        assert abs(T - min(round(float(expit(np.float64(np.float32(x)))) * 2**32), 0xFFFFFFFF)) <= 1
    assert orc.threshold((23, 0, 0, 0, 0), 2, 0, 0, 0, 0) == 0xFFFFFFFF             # certain
    assert orc.threshold((50, 0, 0, 0, 0), 2, 0, 0, 0, 0) == 0xFFFFFFFF
    assert orc.threshold((-23, 0, 0, 0, 0), 2, 0, 0, 0, 0) == 0                     # never
    assert orc.threshold((-50, 0, 0, 0, 0), 2, 0, 0, 0, 0) == 0
    assert orc.trial_succeeds(0xFFFFFFFF, 0xFFFFFFFF) and orc.trial_succeeds(5, 6)
    assert not orc.trial_succeeds(6, 6) and not orc.trial_succeeds(0, 0)


def test_worked_values_of_eq1_with_table2_vector(orc):
    """tests/golden/eq1_worked_values.txt: 60-digit decimal evaluation of Eq. 1 (no libm)."""
    rows = [l for l in (GOLDEN / "eq1_worked_values.txt").read_text().splitlines() if l and not l.startswith("#")]
    assert len(rows) >= 10
    for l in rows:
        f = l.split("|")
        veg, s, a, w, d = f[0].split()
        T = orc.threshold(REF_BETA, int(veg), float(s), float(a), float(w), int(d))
        assert T == int(f[3]), l
        if int(veg) != 0:
            p = orc.probability(REF_BETA, int(veg), float(s), float(a), float(w), int(d))
            assert p == pytest.approx(float(f[2]), rel=1e-12), l


def test_probability_matches_independent_numpy_formula(orc):
    """Full Eq. 1 with all five terms vs a numpy restatement on random cells (tolerance, not bits)."""
    rng = np.random.default_rng(3)
    for _ in range(300):
        beta = rng.normal(0, 2, 5).astype(np.float32)
        veg = int(rng.integers(0, 6)); s = np.float32(rng.uniform(0, 1.0))
        a = np.float32(rng.uniform(0, 2 * np.pi)); w = np.float32(rng.uniform(0, 2 * np.pi))
        for d in range(8):
            b = beta.astype(np.float64)
            psi = np.cos(float(a) - np.deg2rad(315)) if float(s) > np.deg2rad(5) else 0.0
            omega = np.cos(float(w) - d * np.pi / 4)
            sigma = np.tan(float(s)) if np.cos(d * np.pi / 4 - float(a)) < 0 and s > 0 else 0.0
            x = b[0] + b[1] * (veg == 1) + b[2] * psi + b[3] * omega + b[4] * sigma
            assert orc.probability(beta, veg, s, a, w, d) == pytest.approx(expit(x), rel=1e-9, abs=1e-15)


def test_threshold_table_layout(orc):
    rng = np.random.default_rng(5)
    H, W = 5, 7
    L = orc.Landscape(rng.integers(0, 4, (H, W)), rng.uniform(0, 0.6, (H, W)), rng.uniform(0, 6.28, (H, W)),
                      rng.uniform(0, 6.28, (H, W)))
    beta = (-1.0, -0.5, 0.3, 1.0, 0.5)
    tab = orc.threshold_table(L, beta)
    assert tab.shape == (H, W, 8)
    for y in range(H):
        for x in range(W):
            for d in range(8):
                assert tab[y, x, d] == orc.threshold(beta, L.veg[y, x], L.slope[y, x], L.aspect[y, x], L.wind[y, x], d)
