"""Seeded synthetic inputs for the five BASELINE.json configs ("Input recipe").

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no Eq. 1, no thresholds, no Philox, no CA step, no fitness.  It only
(1) generates the raster layers with numpy/scipy and (2) reads the stored parameter
vectors / ignition lists in ``workloads/cfgN.json``.  Those JSON files were written by
``oracle/make_workloads.py`` (which calls only ``oracle/``) because choosing beta_0 for a
target mean spread probability, and picking a reference fire, needs the model itself.

The synthetic landscapes stand in for the paper's Northern-Patagonia rasters
(801x801 cells of 30 m, vegetation {0,1,2}, slope, aspect, WindNinja wind
direction), which are not available.  Shapes, sizes and distributions follow BASELINE.json.
"""
from __future__ import annotations

import json
from dataclasses import dataclass, field
from pathlib import Path

import numpy as np

_DIR = Path(__file__).resolve().parent / "workloads"

CELL_M = 30.0  # PAPER.md:109, 30 m x 30 m cells

# cfg -> (W, H, sigma_e [cells], z_max [m], veg kind, wind kind)
CONFIGS = {
    1: dict(W=64, H=64, sigma_e=4.0, z_max=500.0, veg="iid4", wind="const"),
    2: dict(W=256, H=256, sigma_e=8.0, z_max=1500.0, veg="iid4", wind="field"),
    3: dict(W=1024, H=1024, sigma_e=32.0, z_max=2000.0, veg="clustered6", wind="field"),
    4: dict(W=512, H=512, sigma_e=4.0, z_max=500.0, veg="iid4", wind="const"),
    5: dict(W=4096, H=4096, sigma_e=64.0, z_max=3000.0, veg="clustered6", wind="field"),
}

WORKLOAD_NAMES = {
    1: "cfg1 64x64, 16 vectors x 4 replicates = 64 sims",
    2: "cfg2 256x256, GA population 64 x 4 replicates = 256 sims, Jaccard",
    3: "cfg3 1024x1024 GA population 256 x 8 replicates = 2048 sims, near-transition",
    4: "cfg4 512x512 ignition search, 1024 candidates x 16 replicates = 16384 sims",
    5: "cfg5 4096x4096, 16 high-spread vectors x 4 ignitions = 64 sims",
}


def _noise(shape, sigma, seed):
    from scipy.ndimage import gaussian_filter
    rng = np.random.Generator(np.random.PCG64(seed))
    return gaussian_filter(rng.standard_normal(shape), sigma, mode="reflect", truncate=4.0)


def make_landscape(cfg: int, size: int | None = None) -> dict:
    """Rasters of config ``cfg``: veg u8, slope/aspect/wind f32 radians, row-major [H][W].

    ``size`` overrides W = H (used by small parity cases with the same generators)."""
    c = CONFIGS[cfg]
    W = H = size if size is not None else c["W"]
    n = _noise((H, W), c["sigma_e"], 1000 + cfg)
    z = (n - n.min()) / (n.max() - n.min()) * c["z_max"]
    dz_drow, dz_dcol = np.gradient(z, CELL_M)
    slope = np.arctan(np.hypot(dz_drow, dz_dcol))
    # aspect = compass bearing (clockwise from north, row 0 = north) the slope faces, i.e. downslope
    aspect = np.mod(np.arctan2(-dz_dcol, dz_drow), 2.0 * np.pi)
    if c["veg"] == "iid4":
        rng = np.random.Generator(np.random.PCG64(2000 + cfg))
        veg = rng.choice(4, size=(H, W), p=[0.1, 0.3, 0.3, 0.3]).astype(np.uint8)
    else:
        f = _noise((H, W), c["sigma_e"] / 4.0, 2000 + cfg)
        q = np.quantile(f, [0.05, 0.24, 0.43, 0.62, 0.81])
        veg = np.digitize(f, q).astype(np.uint8)          # 0 on 5 % of cells, in patches
    if c["wind"] == "const":
        wind = np.full((H, W), np.pi / 4.0)
    else:
        g = _noise((H, W), c["sigma_e"], 3000 + cfg)
        wind = 1.5 * np.pi + (np.pi / 6.0) * g / np.abs(g).max()
    # the centre cell is the known ignition of configs 1-4: make sure it can burn
    if veg[H // 2, W // 2] == 0:
        veg[H // 2, W // 2] = 2
    return {"veg": np.ascontiguousarray(veg), "slope": slope.astype(np.float32),
            "aspect": aspect.astype(np.float32), "wind": wind.astype(np.float32), "W": W, "H": H}


def validate_landscape(ls: dict) -> None:
    """R-20: finite inputs, 0 <= slope < pi/2 (host-side precondition check)."""
    for k in ("slope", "aspect", "wind"):
        if not np.isfinite(ls[k]).all():
            raise ValueError(f"raster {k} holds non-finite values")
    if (ls["slope"] < 0).any() or (ls["slope"] >= np.pi / 2).any():
        raise ValueError("slope must lie in [0, pi/2)")


@dataclass
class Workload:
    cfg: int
    name: str
    landscape: dict
    betas: np.ndarray          # f32 [P][5]
    ignitions: np.ndarray      # i32 [S][2] (x, y)
    sim_param: np.ndarray      # i32 [S]
    seeds: np.ndarray          # u64 [S]
    metric: int                # 0 = Eq. 2 delta, 1 = Jaccard
    ref_beta: np.ndarray       # f32 [5]
    ref_ignition: tuple
    ref_seed: int
    groups: tuple | None = None  # (G, R) for config 4
    meta: dict = field(default_factory=dict)

    @property
    def S(self) -> int:
        return int(self.sim_param.shape[0])

    @property
    def P(self) -> int:
        return int(self.betas.shape[0])


def f32_from_bits(bits) -> np.ndarray:
    return np.asarray(bits, dtype=np.uint32).view(np.float32)


def load_recipe(cfg: int) -> dict:
    with open(_DIR / f"cfg{cfg}.json") as f:
        return json.load(f)


def sim_layout(cfg: int, P: int, recipe: dict):
    """(ignitions, sim_param, seeds, groups) of config cfg: param-major then replicate."""
    c = CONFIGS[cfg]
    cx, cy = c["W"] // 2, c["H"] // 2
    if cfg in (1, 2, 3):
        R = {1: 4, 2: 4, 3: 8}[cfg]
        S = P * R
        sim_param = np.repeat(np.arange(P, dtype=np.int32), R)
        ign = np.tile(np.array([[cx, cy]], np.int32), (S, 1))
        groups = None
    elif cfg == 4:
        cand = np.asarray(recipe["candidates"], np.int32).reshape(-1, 2)
        R = 16
        S = cand.shape[0] * R
        sim_param = np.zeros(S, np.int32)
        ign = np.repeat(cand, R, axis=0)
        groups = (cand.shape[0], R)
    else:
        ig = np.asarray(recipe["ignitions"], np.int32).reshape(-1, 2)
        S = P * ig.shape[0]
        sim_param = np.repeat(np.arange(P, dtype=np.int32), ig.shape[0])
        ign = np.tile(ig, (P, 1))
        groups = None
    seeds = (np.uint64(cfg) << np.uint64(32)) | np.arange(S, dtype=np.uint64)
    return np.ascontiguousarray(ign), sim_param, seeds, groups


def load_workload(cfg: int, landscape: dict | None = None) -> Workload:
    r = load_recipe(cfg)
    betas = f32_from_bits(r["betas_f32_bits"]).reshape(-1, 5).copy()
    ign, sim_param, seeds, groups = sim_layout(cfg, betas.shape[0], r)
    ls = landscape if landscape is not None else make_landscape(cfg)
    return Workload(cfg=cfg, name=WORKLOAD_NAMES[cfg], landscape=ls, betas=betas, ignitions=ign,
                    sim_param=sim_param, seeds=seeds, metric=int(r["metric"]),
                    ref_beta=f32_from_bits(r["ref_beta_f32_bits"]).copy(),
                    ref_ignition=tuple(r["ref_ignition"]), ref_seed=int(r["ref_seed"]),
                    groups=groups, meta=r.get("meta", {}))


def shard_sims(S: int, rank: int, world: int) -> slice:
    """Contiguous, near-equal shard of the sim axis for rank ``rank`` of ``world`` (multi-GPU)."""
    base, rem = divmod(S, world)
    lo = rank * base + min(rank, rem)
    return slice(lo, lo + base + (1 if rank < rem else 0))


@dataclass
class ParamShard:
    """What rank ``rank`` of ``world`` runs when a generation is partitioned BY PARAMETER VECTOR (PAPER.md:117:
    individuals are independent): the rank uploads only `betas` (so it builds P_local / P of the threshold table), simulates
    the sims at positions `index` of the batch with `sim_param` re-based to its slice and `sim_ids` = their global batch
    positions (the `sim` field of the random-number key, so every fire is the one the full batch would produce)."""
    p_lo: int
    p_hi: int
    betas: np.ndarray          # f32 [P_local][5]
    index: np.ndarray          # i64 [S_local]  positions in the full batch, ascending
    sim_param: np.ndarray      # i32 [S_local]  in [0, P_local)
    sim_ids: np.ndarray        # i32 [S_local]  = index
    ignitions: np.ndarray      # i32 [S_local][2]
    seeds: np.ndarray          # u64 [S_local]


def shard_by_param(w: Workload, rank: int, world: int) -> ParamShard:
    """Contiguous, near-equal slices of the parameter-vector axis; a sim goes where its vector goes.  Sims whose `sim_param`
    is outside [0, P) (R-12: they burn nothing) go to rank 0, which keeps them invalid (index P_local)."""
    sl = shard_sims(w.P, rank, world)
    sp = np.asarray(w.sim_param, np.int64)
    mine = (sp >= sl.start) & (sp < sl.stop)
    if rank == 0:
        mine |= (sp < 0) | (sp >= w.P)
    index = np.flatnonzero(mine)
    local = sp[index] - sl.start
    local[(sp[index] < 0) | (sp[index] >= w.P)] = sl.stop - sl.start          # stays out of range
    return ParamShard(p_lo=sl.start, p_hi=sl.stop, betas=np.ascontiguousarray(w.betas[sl]), index=index,
                      sim_param=local.astype(np.int32), sim_ids=index.astype(np.int32),
                      ignitions=np.ascontiguousarray(w.ignitions[index]), seeds=np.ascontiguousarray(w.seeds[index]))


def merge_param_shards(parts: list, values: list, S: int) -> np.ndarray:
    """Per-shard result vectors (one entry per local sim) back into batch order."""
    out = np.empty((S,) + tuple(np.asarray(values[0]).shape[1:]), dtype=np.asarray(values[0]).dtype)
    seen = np.zeros(S, bool)
    for sh, v in zip(parts, values):
        out[sh.index] = np.asarray(v)[: len(sh.index)]
        seen[sh.index] = True
    if not seen.all():
        raise ValueError("shards do not cover the batch")
    return out
