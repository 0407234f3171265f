"""Writes the stored inputs and expected values of the five BASELINE.json configs.

    python -m oracle.make_workloads [cfg ...] [--no-expected]

Calls ONLY the CPU oracle (oracle/fire_oracle.c) and the raster generators
(paper_1701_03549_b200/workloads.py, which holds none of the method's arithmetic).
Nothing here ever comes from the CUDA path.

Outputs
  paper_1701_03549_b200/workloads/cfgN.json   inputs: parameter vectors (beta_0 solved by
        bisection for a target mean spread probability), reference vector / ignition / seed,
        candidate ignitions (cfg 4), ignitions (cfg 5).  Recipe: DESIGN.md "Input recipe".
  tests/golden/cfgN_expected.json             oracle results for every simulation of the
        config: steps, burned area, trials, candidate cell-steps, distinct targets, and an
        8-byte BLAKE2b digest of the canonical burned bitmap; fitness counts vs the reference.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

from oracle import fire_oracle as orc                      # noqa: E402
from paper_1701_03549_b200 import workloads as wl          # noqa: E402

P_OF_CFG = {1: 16, 2: 64, 3: 256, 4: 1, 5: 16}
PBAR_RANGE = {1: (0.15, 0.45), 2: (0.15, 0.45), 3: (0.22, 0.32), 5: (0.40, 0.55)}
REF_TAIL = (-0.5, 0.3, 1.0, 0.5)           # (beta_1..beta_4) of the reference / fixed vector
REF_PBAR = {1: 0.30, 2: 0.30, 3: 0.30, 4: 0.30, 5: 0.475}
METRIC = {1: 0, 2: 1, 3: 0, 4: 0, 5: 0}


def bits(a) -> list:
    return [int(v) for v in np.asarray(a, np.float32).ravel().view(np.uint32)]


def digest(bitmap: np.ndarray) -> str:
    return hashlib.blake2b(np.ascontiguousarray(bitmap, "<u4").tobytes(), digest_size=8).hexdigest()


def solve_beta0(tail, pbar, sample) -> np.float32:
    """beta_0 such that the mean of Eq. 1 over the sample cells x 8 directions equals pbar."""
    lo, hi = -40.0, 40.0
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        m = orc.mean_probability([mid, *tail], *sample)
        if m < pbar:
            lo = mid
        else:
            hi = mid
    return np.float32(0.5 * (lo + hi))


def make(cfg: int, want_expected: bool = True) -> None:
    t0 = time.time()
    ls = wl.make_landscape(cfg)
    wl.validate_landscape(ls)
    W, H = ls["W"], ls["H"]
    L = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    burnable = np.flatnonzero(ls["veg"].ravel() != 0)
    rng = np.random.Generator(np.random.PCG64(6000 + cfg))
    idx = rng.choice(burnable, size=min(4096, burnable.size), replace=False)
    sample = tuple(ls[k].ravel()[idx] for k in ("veg", "slope", "aspect", "wind"))

    # ---- parameter vectors
    P = P_OF_CFG[cfg]
    rng = np.random.Generator(np.random.PCG64(4000 + cfg))
    ref_beta = np.array([solve_beta0(REF_TAIL, REF_PBAR[cfg], sample), *REF_TAIL], np.float32)
    if cfg == 4:
        betas = ref_beta[None, :].copy()               # fixed parameters, unknown ignition
        pbars = [REF_PBAR[cfg]]
    else:
        betas = np.zeros((P, 5), np.float32)
        pbars = []
        for p in range(P):
            tail = (rng.uniform(-1, 0), rng.uniform(-0.5, 0.5), rng.uniform(0, 2), rng.uniform(0, 1.5))
            pbar = rng.uniform(*PBAR_RANGE[cfg])
            betas[p, 1:] = tail
            betas[p, 0] = solve_beta0([float(np.float32(v)) for v in tail], pbar, sample)
            pbars.append(float(pbar))

    # ---- reference fire: first seed whose burn is large enough
    cx, cy = W // 2, H // 2
    rng5 = np.random.Generator(np.random.PCG64(5000 + cfg))
    if cfg == 5:
        ys, xs = np.nonzero(ls["veg"] != 0)
        ok = (xs >= W // 8) & (xs < W - W // 8) & (ys >= H // 8) & (ys < H - H // 8)
        pick = rng5.choice(np.flatnonzero(ok), size=4, replace=False)
        ignitions5 = [[int(xs[i]), int(ys[i])] for i in pick]
        ref_ign = tuple(ignitions5[0])
    else:
        ref_ign = (cx, cy)
    need = max(200, int(0.005 * W * H))
    ref_table = orc.threshold_table(L, ref_beta)
    k = 0
    while True:
        ref_seed = (0xF1 << 40) | (cfg << 32) | k
        ref = orc.simulate(L, ref_beta, ref_ign, ref_seed, sim=0, table=ref_table)
        area = int(sum(bin(int(w)).count("1") for w in ref["burned"].ravel() if w))
        if area >= need:
            break
        k += 1
        assert k < 1000, "no reference fire large enough"
    print(f"cfg{cfg}: reference seed k={k} area={area} steps={ref['steps']} trials={ref['trials']}", flush=True)

    recipe = {"cfg": cfg, "W": W, "H": H, "metric": METRIC[cfg],
              "betas_f32_bits": bits(betas), "betas_readable": [[float(v) for v in r] for r in betas],
              "ref_beta_f32_bits": bits(ref_beta), "ref_beta_readable": [float(v) for v in ref_beta],
              "ref_ignition": [int(ref_ign[0]), int(ref_ign[1])], "ref_seed": int(ref_seed),
              "meta": {"pbar_targets": pbars, "ref_pbar": REF_PBAR[cfg], "ref_area": area,
                       "ref_steps": ref["steps"], "written_by": "oracle/make_workloads.py"}}
    if cfg == 4:
        b = np.array([[(int(w) >> i) & 1 for w in row for i in range(32)] for row in ref["burned"]], bool)[:, :W]
        ys, xs = np.nonzero(b)
        x0, x1, y0, y1 = xs.min(), xs.max(), ys.min(), ys.max()
        yy, xx = np.nonzero(ls["veg"][y0:y1 + 1, x0:x1 + 1] != 0)
        assert yy.size >= 1024, "reference bounding box too small for 1024 candidates"
        pick = rng5.choice(yy.size, size=1024, replace=False)
        recipe["candidates"] = [[int(xx[i] + x0), int(yy[i] + y0)] for i in pick]
        recipe["meta"]["ref_bbox"] = [int(x0), int(y0), int(x1), int(y1)]
    if cfg == 5:
        recipe["ignitions"] = ignitions5
    out = ROOT / "paper_1701_03549_b200" / "workloads" / f"cfg{cfg}.json"
    out.parent.mkdir(parents=True, exist_ok=True)
    out.write_text(json.dumps(recipe, separators=(",", ":")) + "\n")
    print(f"cfg{cfg}: wrote {out.relative_to(ROOT)} ({time.time() - t0:.1f}s)", flush=True)
    if not want_expected:
        return

    # ---- expected values of the whole batch (oracle, table per parameter vector)
    w = wl.load_workload(cfg, landscape=ls)
    S = w.S
    steps = np.zeros(S, np.int64); areas = np.zeros(S, np.int64); trials = np.zeros(S, np.int64)
    cands = np.zeros(S, np.int64); distinct = np.zeros(S, np.int64)
    I_cnt = np.zeros(S, np.int64); digs = [""] * S
    refw = ref["burned"]
    N_ref = int(np.unpackbits(refw.view(np.uint8)).sum())
    for p in range(w.P):
        sel = np.flatnonzero(w.sim_param == p)
        table = ref_table if (cfg == 4) else orc.threshold_table(L, w.betas[p])
        tabs = [None] * w.P
        tabs[p] = table
        CH = 256 if cfg != 5 else 4                       # bound the [S][H][Ww] output buffer
        for c0 in range(0, sel.size, CH):
            ss = sel[c0:c0 + CH]
            r = orc.simulate_batch(L, w.betas, w.ignitions[ss], w.sim_param[ss], w.seeds[ss],
                                   sim_index=ss.astype(np.int32), tables=tabs)
            for j, s in enumerate(ss):
                bm = r["burned"][j]
                steps[s] = r["steps"][j]; trials[s] = r["trials"][j]
                cands[s] = r["cand_steps"][j]; distinct[s] = r["distinct"][j]
                areas[s] = int(np.unpackbits(bm.view(np.uint8)).sum())
                I_cnt[s] = int(np.unpackbits((bm & refw).view(np.uint8)).sum())
                digs[s] = digest(bm)
        print(f"cfg{cfg}: param {p + 1}/{w.P} done ({time.time() - t0:.0f}s)", flush=True)
    exp = {"cfg": cfg, "S": S, "ref_area": N_ref, "ref_digest": digest(refw), "ref_steps": ref["steps"],
           "steps": steps.tolist(), "area": areas.tolist(), "trials": trials.tolist(),
           "cand_steps": cands.tolist(), "distinct": distinct.tolist(), "intersection": I_cnt.tolist(),
           "digest": digs,
           "totals": {"trials": int(trials.sum()), "cand_steps": int(cands.sum()),
                      "distinct": int(distinct.sum()), "area": int(areas.sum()), "steps_max": int(steps.max())},
           "written_by": "oracle/make_workloads.py (CPU oracle only)"}
    out = ROOT / "tests" / "golden" / f"cfg{cfg}_expected.json"
    out.parent.mkdir(parents=True, exist_ok=True)
    out.write_text(json.dumps(exp, separators=(",", ":")) + "\n")
    frac = areas / float(W * H)
    print(f"cfg{cfg}: S={S} trials={trials.sum():.3e} cand={cands.sum():.3e} distinct={distinct.sum():.3e} "
          f"area mean={areas.mean():.0f} med={np.median(areas):.0f} max={areas.max()} "
          f"steps mean={steps.mean():.0f} max={steps.max()} "
          f"frac<100 cells={np.mean(areas < 100):.2f} frac>1%={np.mean(frac > 0.01):.2f} "
          f"({time.time() - t0:.0f}s)", flush=True)
    # acceptance checks of the recipe
    if cfg == 3:
        assert np.mean(frac > 0.01) >= 0.25, "cfg3: fewer than 25 % of sims burn > 1 % of the lattice"
    if cfg == 5:
        nburnable = int((ls["veg"] != 0).sum())
        # a fire can still die in its first steps by chance (1 of 64 does, 206 cells): DESIGN.md
        assert np.mean(areas > 0.5 * nburnable) >= 0.95, "cfg5: > 5 % of sims burned <= 50 % of burnable cells"


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("cfgs", nargs="*", type=int, default=[1, 2, 3, 4, 5])
    ap.add_argument("--no-expected", action="store_true")
    a = ap.parse_args()
    for c in a.cfgs:
        make(c, want_expected=not a.no_expected)
