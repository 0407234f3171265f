"""Writes tests/golden/eq1_worked_values.txt: worked values of Eq. 1 and of the
32-bit threshold T = round_half_even(2^32 p) for the paper's reference parameter vector
(-5, -10, 5, 18.1, -5) (Table 2) on hand-picked cells.

Independent route: Python's arbitrary-precision ``decimal`` (60 digits) with Taylor series
for sin/cos and Decimal.exp().  It imports neither the oracle nor the CUDA package and does
not use libm.  Inputs are the exact binary values a C program would hold (f32 parameters
and rasters widened to double, phi_d = d * (double)(pi/4)); the arithmetic is exact real
arithmetic, rounded once at the end.  Each row records the margin to the nearest rounding
boundary so that an IEEE-double implementation (error ~1e-16 relative) must reproduce T exactly.

    python tests/golden/make_eq1_worked.py
"""
from __future__ import annotations

import math
import struct
from decimal import Decimal, getcontext, ROUND_HALF_EVEN
from pathlib import Path

getcontext().prec = 60
PI = Decimal("3.14159265358979323846264338327950288419716939937510582097494")


def f32(x: float) -> float:
    return struct.unpack("<f", struct.pack("<f", x))[0]


def dsin(x: Decimal) -> Decimal:
    x = x - (x / (2 * PI)).to_integral_value() * 2 * PI
    term, total, n = x, x, 1
    while abs(term) > Decimal(10) ** -58:
        term = -term * x * x / ((2 * n) * (2 * n + 1))
        total += term
        n += 1
    return total


def dcos(x: Decimal) -> Decimal:
    return dsin(x + PI / 2)


def phi(d: int) -> Decimal:
    return Decimal(d * (math.pi / 4.0))          # the double a C program computes, taken exactly


def worked(beta, veg, slope, aspect, wind, d):
    b = [Decimal(f32(v)) for v in beta]
    s, a, w = Decimal(f32(slope)), Decimal(f32(aspect)), Decimal(f32(wind))
    I_f = Decimal(1 if veg == 1 else 0)
    psi = dcos(a - phi(7)) if s > Decimal(5.0 * math.pi / 180.0) else Decimal(0)
    omega = dcos(w - phi(d))
    uphill = (s > 0) and (dcos(phi(d) - a) < 0)
    sigma = dsin(s) / dcos(s) if uphill else Decimal(0)
    x = b[0] + b[1] * I_f + b[2] * psi + b[3] * omega + b[4] * sigma
    p = 1 / (1 + (-x).exp())
    scaled = p * (1 << 32)
    T = int(scaled.to_integral_value(rounding=ROUND_HALF_EVEN))
    T = min(T, 0xFFFFFFFF) if veg != 0 else 0
    frac = scaled - int(scaled)
    margin = abs(frac - Decimal("0.5"))
    return x, p, T, margin


CASES = [
    # name, veg, slope, aspect, wind, d
    ("shrub flat downwind (wind toward N, travel N)", 2, 0.0, 0.0, 0.0, 0),
    ("forest flat downwind", 1, 0.0, 0.0, 0.0, 0),
    ("shrub flat upwind (travel S against wind toward N)", 2, 0.0, 0.0, 0.0, 4),
    ("forest flat upwind", 1, 0.0, 0.0, 0.0, 4),
    ("shrub flat crosswind (travel E)", 2, 0.0, 0.0, 0.0, 2),
    ("shrub flat quartering wind (travel NE)", 2, 0.0, 0.0, 0.0, 1),
    ("shrub NW-facing 0.2 rad slope, travel SE = uphill", 2, 0.2, 7 * math.pi / 4, 0.0, 3),
    ("shrub NW-facing 0.2 rad slope, travel NW = downhill", 2, 0.2, 7 * math.pi / 4, 0.0, 7),
    ("forest SE-facing 0.3 rad slope, wind toward E, travel E", 1, 0.3, 3 * math.pi / 4, math.pi / 2, 2),
    ("shrub S-facing 0.05 rad slope (< 5 deg: no aspect term), travel N = uphill", 2, 0.05, math.pi, 0.0, 0),
    ("other fuel class 3 (I_f = 0) W-facing 0.4 rad, wind toward SE, travel E = uphill", 3, 0.4, 3 * math.pi / 2, 3 * math.pi / 4, 2),
    ("non-burnable", 0, 0.1, 1.0, 2.0, 5),
]
BETA = (-5.0, -10.0, 5.0, 18.1, -5.0)


def main():
    out = Path(__file__).with_name("eq1_worked_values.txt")
    lines = ["# Worked values of Eq. 1 (PAPER.md:76) with the reference vector of Table 2 (PAPER.md:184-188)",
             "# beta = (-5, -10, 5, 18.1, -5) held as f32.  Written by tests/golden/make_eq1_worked.py",
             "# (60-digit decimal arithmetic; no libm, no oracle, no CUDA).",
             "# columns: veg slope_f32 aspect_f32 wind_f32 d | x | p | T | margin_to_rounding_boundary | name"]
    for name, veg, s, a, w, d in CASES:
        x, p, T, margin = worked(BETA, veg, s, a, w, d)
        assert veg == 0 or T in (0, 0xFFFFFFFF) or margin > Decimal("1e-3"), (name, margin)
        lines.append(f"{veg} {f32(s)!r} {f32(a)!r} {f32(w)!r} {d} | {x:.30f} | {p:.30e} | {T} | {margin:.3e} | {name}")
    out.write_text("\n".join(lines) + "\n")
    print(out.read_text())


if __name__ == "__main__":
    main()
