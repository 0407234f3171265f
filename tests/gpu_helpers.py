"""Marshalling helpers for the `-m gpu` parity tests: numpy <-> CUDA tensors around the C-ABI binding.

No arithmetic of the method lives here; every result comes out of libfire's kernels."""
from __future__ import annotations

import hashlib

import numpy as np
import torch

from paper_1701_03549_b200 import libfire as lf


_SIGNED = {np.dtype(np.uint32): np.int32, np.dtype(np.uint64): np.int64}


def dev(a: np.ndarray) -> torch.Tensor:
    """numpy -> CUDA tensor; unsigned 32/64-bit arrays travel as the signed type of the same bit pattern."""
    a = np.ascontiguousarray(a)
    if a.dtype in _SIGNED:
        a = a.view(_SIGNED[a.dtype])
    return torch.from_numpy(a).cuda()


def make_landscape(ls: dict) -> lf.Landscape:
    """ls: dict(veg u8, slope/aspect/wind f32) of numpy rasters -> handle."""
    L = lf.fire_landscape_create(dev(ls["veg"].astype(np.uint8)), dev(ls["slope"].astype(np.float32)),
                                 dev(ls["aspect"].astype(np.float32)), dev(ls["wind"].astype(np.float32)))
    torch.cuda.synchronize()
    return L


def upload(L: lf.Landscape, betas) -> None:
    b = np.ascontiguousarray(np.asarray(betas, np.float32).reshape(-1, 5))
    lf.fire_params_upload(L, dev(b))


def thresholds(L: lf.Landscape, p: int) -> np.ndarray:
    out = torch.empty((L.H, L.W, 8), dtype=torch.int32, device="cuda")
    lf.fire_thresholds_download(L, p, out)
    torch.cuda.synchronize()
    return out.cpu().numpy().view(np.uint32)


def simulate(L: lf.Landscape, ignitions, sim_param, seeds, sim_ids=None, max_steps: int = 0, keep_device: bool = False):
    """Returns dict(burned u32[S][H][Ww], steps u32[S], trials u64[S]) as numpy (burned stays a tensor if keep_device)."""
    ign = np.ascontiguousarray(np.asarray(ignitions, np.int32).reshape(-1, 2))
    S = ign.shape[0]
    sp = np.ascontiguousarray(np.asarray(sim_param, np.int32))
    sd = np.ascontiguousarray(np.asarray(seeds, np.uint64))
    burned = torch.full((S, L.H, L.Ww), -1, dtype=torch.int32, device="cuda")     # poison: every word must be written
    steps = torch.full((S,), -1, dtype=torch.int32, device="cuda")
    trials = torch.full((S,), -1, dtype=torch.int64, device="cuda")
    ids = dev(np.asarray(sim_ids, np.int32)) if sim_ids is not None else None
    lf.fire_simulate_batch(L, dev(ign), dev(sp), dev(sd), burned, steps, trials, sim_ids=ids, max_steps=max_steps)
    torch.cuda.synchronize()
    return {"burned": burned if keep_device else burned.cpu().numpy().view(np.uint32),
            "steps": steps.cpu().numpy().view(np.uint32), "trials": trials.cpu().numpy().view(np.uint64)}


def fitness(L: lf.Landscape, reference: np.ndarray, burned, metric: int):
    """counts u32[S][2], scores f32[S], N."""
    b = burned if isinstance(burned, torch.Tensor) else dev(np.asarray(burned, np.uint32))
    S = b.shape[0]
    score = torch.empty((S,), dtype=torch.float32, device="cuda")
    counts = torch.full((S, 2), -1, dtype=torch.int32, device="cuda")
    area = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    lf.fire_fitness(L, dev(np.asarray(reference, np.uint32)), b, metric, score, counts, area)
    torch.cuda.synchronize()
    return counts.cpu().numpy().view(np.uint32), score.cpu().numpy(), int(area.cpu().numpy().view(np.uint32)[0])


def group_stats(counts: np.ndarray, N: int, G: int, R: int):
    sums = torch.empty((G, 2), dtype=torch.int64, device="cuda")
    mv = torch.empty((G, 2), dtype=torch.float64, device="cuda")
    lf.fire_fitness_group_stats(dev(np.asarray(counts, np.uint32)), N, G, R, sums, mv)
    torch.cuda.synchronize()
    return sums.cpu().numpy().view(np.uint64), mv.cpu().numpy()


def digest(bitmap: np.ndarray) -> str:
    """Same 8-byte BLAKE2b of the canonical little-endian words as oracle/make_workloads.py uses."""
    return hashlib.blake2b(np.ascontiguousarray(bitmap, "<u4").tobytes(), digest_size=8).hexdigest()


def popcount(a: np.ndarray) -> np.ndarray:
    """Per-sim popcount of u32[S][...]."""
    a = np.ascontiguousarray(a)
    return np.unpackbits(a.view(np.uint8).reshape(a.shape[0], -1), axis=1).sum(axis=1, dtype=np.int64)
