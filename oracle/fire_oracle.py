"""ctypes front-end of the CPU oracle (oracle/fire_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, bench.py's cpu_baseline /
``--impl reference`` legs and ``__graft_entry__.smoke()`` may import this module.
It never imports the CUDA package and the CUDA package never imports it.

Argument marshalling only: every number comes out of fire_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "fire_oracle.c"
_LIB = _HERE / "libfire_oracle.so"
CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> Path:
    """Compile fire_oracle.c with gcc (building the checker is not using it)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(["gcc", *CFLAGS, "-o", str(tmp), str(_SRC), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _declare(_lib)
    return _lib


_u8p = C.POINTER(C.c_uint8)
_u32p = C.POINTER(C.c_uint32)
_i32p = C.POINTER(C.c_int32)
_u64p = C.POINTER(C.c_uint64)
_f32p = C.POINTER(C.c_float)
_f64p = C.POINTER(C.c_double)


class OrcCov(C.Structure):
    _fields_ = [("burnable", C.c_int), ("I_f", C.c_double), ("psi", C.c_double),
                ("omega", C.c_double * 8), ("sigma", C.c_double * 8)]


def _declare(l):
    l.orc_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
    l.orc_philox4x32_10.restype = None
    l.orc_rnd.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_int]
    l.orc_rnd.restype = C.c_uint32
    l.orc_direction_offset.argtypes = [C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    l.orc_direction_offset.restype = None
    l.orc_covariates.argtypes = [C.c_uint8, C.c_float, C.c_float, C.c_float, C.POINTER(OrcCov)]
    l.orc_covariates.restype = None
    l.orc_probability.argtypes = [_f32p, C.c_uint8, C.c_float, C.c_float, C.c_float, C.c_int]
    l.orc_probability.restype = C.c_double
    l.orc_mean_probability.argtypes = [_f32p, _u8p, _f32p, _f32p, _f32p, C.c_int]
    l.orc_mean_probability.restype = C.c_double
    l.orc_threshold.argtypes = [_f32p, C.c_uint8, C.c_float, C.c_float, C.c_float, C.c_int]
    l.orc_threshold.restype = C.c_uint32
    l.orc_trial_succeeds.argtypes = [C.c_uint32, C.c_uint32]
    l.orc_trial_succeeds.restype = C.c_int
    l.orc_threshold_table.argtypes = [_f32p, _u8p, _f32p, _f32p, _f32p, C.c_int, C.c_int, _u32p]
    l.orc_threshold_table.restype = None
    l.orc_threshold_table_dem.argtypes = [_f32p, _u8p, _f32p, _f32p, _f32p, _f32p, C.c_int, C.c_int, _u32p]
    l.orc_threshold_table_dem.restype = None
    l.orc_threshold_table_classes.argtypes = [_f32p, _u8p, _f32p, _f32p, _f32p, _f32p, C.c_int, C.c_int, _u32p]
    l.orc_threshold_table_classes.restype = None
    l.orc_simulate.argtypes = [_u8p, _f32p, _f32p, _f32p, C.c_int, C.c_int, _f32p, _u32p,
                               C.c_int, C.c_int, C.c_uint64, C.c_uint32, C.c_uint32,
                               _u32p, _i32p, _u32p, _u64p]
    l.orc_simulate.restype = C.c_int
    l.orc_simulate_burn_time.argtypes = [_u8p, _f32p, _f32p, _f32p, C.c_int, C.c_int, _f32p, _u32p, _u8p,
                                         C.c_int, C.c_int, C.c_uint64, C.c_uint32, C.c_uint32,
                                         _u32p, _i32p, _u32p, _u64p]
    l.orc_simulate_burn_time.restype = C.c_int
    l.orc_simulate_batch.argtypes = [_u8p, _f32p, _f32p, _f32p, C.c_int, C.c_int, _f32p, C.c_int,
                                     C.POINTER(_u32p), _i32p, _i32p, _u64p, _i32p, C.c_int,
                                     C.c_uint32, _u32p, _u32p, _u64p, C.c_int]
    l.orc_simulate_batch.restype = C.c_int
    l.orc_fitness_counts.argtypes = [_u32p, _u32p, C.c_int, C.c_int, _u32p]
    l.orc_fitness_counts.restype = None
    l.orc_fitness_score.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, C.c_int]
    l.orc_fitness_score.restype = C.c_float
    l.orc_group_stats.argtypes = [_u32p, C.c_uint32, C.c_int, C.c_int, _u64p, _f64p]
    l.orc_group_stats.restype = None
    l.orc_max_threads.argtypes = []
    l.orc_max_threads.restype = C.c_int


def _p(a: np.ndarray, t):
    return a.ctypes.data_as(t)


def _c(a, dtype) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=dtype)


# --------------------------------------------------------------------------- RNG
def philox4x32_10(ctr, key) -> np.ndarray:
    ctr = _c(ctr, np.uint32); key = _c(key, np.uint32); out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(ctr, _u32p), _p(key, _u32p), _p(out, _u32p))
    return out


def rnd(seed: int, sim: int, step: int, cell: int, d: int) -> int:
    return int(lib().orc_rnd(seed, sim, step, cell, d))


def direction_offset(d: int):
    dx, dy = C.c_int(), C.c_int()
    lib().orc_direction_offset(d, C.byref(dx), C.byref(dy))
    return dx.value, dy.value


# --------------------------------------------------------------------- Eq. 1 / C-2 / C-3
def covariates(veg: int, slope: float, aspect: float, wind: float) -> dict:
    c = OrcCov()
    lib().orc_covariates(int(veg), float(slope), float(aspect), float(wind), C.byref(c))
    return {"burnable": bool(c.burnable), "I_f": c.I_f, "psi": c.psi,
            "omega": np.array(c.omega[:]), "sigma": np.array(c.sigma[:])}


def probability(beta, veg, slope, aspect, wind, d) -> float:
    b = _c(beta, np.float32)
    return float(lib().orc_probability(_p(b, _f32p), int(veg), float(slope), float(aspect), float(wind), int(d)))


def mean_probability(beta, veg, slope, aspect, wind) -> float:
    b = _c(beta, np.float32)
    v = _c(veg, np.uint8).ravel(); s = _c(slope, np.float32).ravel()
    a = _c(aspect, np.float32).ravel(); w = _c(wind, np.float32).ravel()
    return float(lib().orc_mean_probability(_p(b, _f32p), _p(v, _u8p), _p(s, _f32p), _p(a, _f32p),
                                            _p(w, _f32p), int(v.size)))


def threshold(beta, veg, slope, aspect, wind, d) -> int:
    b = _c(beta, np.float32)
    return int(lib().orc_threshold(_p(b, _f32p), int(veg), float(slope), float(aspect), float(wind), int(d)))


def trial_succeeds(r: int, T: int) -> bool:
    return bool(lib().orc_trial_succeeds(r, T))


class Landscape:
    """The four rasters, row-major [H][W], radians."""

    def __init__(self, veg, slope, aspect, wind):
        self.veg = _c(veg, np.uint8)
        self.slope = _c(slope, np.float32)
        self.aspect = _c(aspect, np.float32)
        self.wind = _c(wind, np.float32)
        self.H, self.W = self.veg.shape
        assert self.slope.shape == self.aspect.shape == self.wind.shape == (self.H, self.W)
        self.Ww = (self.W + 31) // 32

    def _ptrs(self):
        return (_p(self.veg, _u8p), _p(self.slope, _f32p), _p(self.aspect, _f32p), _p(self.wind, _f32p))


def threshold_table(L: Landscape, beta) -> np.ndarray:
    b = _c(beta, np.float32)
    out = np.zeros((L.H, L.W, 8), np.uint32)
    lib().orc_threshold_table(_p(b, _f32p), *L._ptrs(), L.W, L.H, _p(out, _u32p))
    return out


def threshold_table_dem(L: Landscape, beta, elevation) -> np.ndarray:
    """Table with the literal DEM uphill test of PAPER.md:87 (variant f4): elevation f32[H][W]."""
    b = _c(beta, np.float32)
    z = _c(elevation, np.float32)
    assert z.shape == (L.H, L.W)
    out = np.zeros((L.H, L.W, 8), np.uint32)
    lib().orc_threshold_table_dem(_p(b, _f32p), *L._ptrs(), _p(z, _f32p), L.W, L.H, _p(out, _u32p))
    return out


def threshold_table_classes(L: Landscape, beta, class_if) -> np.ndarray:
    """Table with a per-class vegetation term (variant f4): class_if[v] = I_f of vegetation class v."""
    b = _c(beta, np.float32)
    w = np.zeros(256, np.float32)
    w[: len(class_if)] = np.asarray(class_if, np.float32)
    out = np.zeros((L.H, L.W, 8), np.uint32)
    lib().orc_threshold_table_classes(_p(b, _f32p), *L._ptrs(), _p(w, _f32p), L.W, L.H, _p(out, _u32p))
    return out


def burn_count(burned_batch, W: int) -> np.ndarray:
    """Hazard map (the use of [12]): for every cell, in how many of the maps it is burnt.  u32[H][W]."""
    b = np.ascontiguousarray(burned_batch, dtype="<u4")
    bits = np.unpackbits(b.view(np.uint8), axis=-1, bitorder="little")[..., :W]
    return bits.sum(axis=0, dtype=np.uint32)


# --------------------------------------------------------------------------- C-4
def simulate(L: Landscape, beta, ignition, seed: int, sim: int = 0, max_steps: int = 0,
             table: np.ndarray | None = None, want_time: bool = False):
    """One simulation.  Returns dict(burned u32[H][Ww], steps, trials, cand_steps, distinct, time)."""
    b = _c(beta, np.float32)
    burned = np.zeros((L.H, L.Ww), np.uint32)
    steps = C.c_uint32(0)
    counters = np.zeros(3, np.uint64)
    time = np.zeros((L.H, L.W), np.int32) if want_time else None
    tab = None
    if table is not None:
        tab = _c(table, np.uint32)
        assert tab.shape == (L.H, L.W, 8)
    rc = lib().orc_simulate(*L._ptrs(), L.W, L.H, _p(b, _f32p),
                            _p(tab, _u32p) if tab is not None else None,
                            int(ignition[0]), int(ignition[1]), int(seed), int(sim), int(max_steps),
                            _p(burned, _u32p), _p(time, _i32p) if want_time else None,
                            C.byref(steps), _p(counters, _u64p))
    if rc != 0:
        raise MemoryError("orc_simulate failed")
    return {"burned": burned, "steps": int(steps.value), "trials": int(counters[0]),
            "cand_steps": int(counters[1]), "distinct": int(counters[2]), "time": time}


def simulate_burn_time(L: Landscape, beta, burn_time, ignition, seed: int, sim: int = 0, max_steps: int = 0,
                       table: np.ndarray | None = None, want_time: bool = False):
    """One simulation with fuel-dependent burn-out times (C-4', R-21): burn_time[v] = steps a cell of class v stays active."""
    b = _c(beta, np.float32)
    bt = np.zeros(256, np.uint8)
    bt[: len(burn_time)] = np.asarray(burn_time, np.uint8)
    burned = np.zeros((L.H, L.Ww), np.uint32)
    steps = C.c_uint32(0)
    counters = np.zeros(3, np.uint64)
    time = np.zeros((L.H, L.W), np.int32) if want_time else None
    tab = None
    if table is not None:
        tab = _c(table, np.uint32)
        assert tab.shape == (L.H, L.W, 8)
    rc = lib().orc_simulate_burn_time(*L._ptrs(), L.W, L.H, _p(b, _f32p), _p(tab, _u32p) if tab is not None else None,
                                      _p(bt, _u8p), int(ignition[0]), int(ignition[1]), int(seed), int(sim),
                                      int(max_steps), _p(burned, _u32p), _p(time, _i32p) if want_time else None,
                                      C.byref(steps), _p(counters, _u64p))
    if rc != 0:
        raise MemoryError("orc_simulate_burn_time failed")
    return {"burned": burned, "steps": int(steps.value), "trials": int(counters[0]),
            "cand_steps": int(counters[1]), "distinct": int(counters[2]), "time": time}


def simulate_batch(L: Landscape, betas, ignitions, sim_param, seeds, sim_index=None, max_steps: int = 0,
                   tables=None, nthreads: int = 0):
    """Independent simulations, OpenMP over sims.  tables: None or list of P (None | u32[H][W][8])."""
    betas = _c(betas, np.float32).reshape(-1, 5)
    P = betas.shape[0]
    ign = _c(ignitions, np.int32).reshape(-1, 2)
    S = ign.shape[0]
    sp = _c(sim_param, np.int32); sd = _c(seeds, np.uint64)
    assert sp.shape == (S,) and sd.shape == (S,)
    si = _c(sim_index, np.int32) if sim_index is not None else None
    burned = np.zeros((S, L.H, L.Ww), np.uint32)
    steps = np.zeros(S, np.uint32)
    counters = np.zeros((S, 3), np.uint64)
    tabs_keep, tabp = [], None
    if tables is not None:
        arr = (_u32p * P)()
        for p in range(P):
            if tables[p] is None:
                arr[p] = None
            else:
                t = _c(tables[p], np.uint32); tabs_keep.append(t)
                assert t.shape == (L.H, L.W, 8)
                arr[p] = _p(t, _u32p)
        tabp = arr
    rc = lib().orc_simulate_batch(*L._ptrs(), L.W, L.H, _p(betas, _f32p), P, tabp,
                                  _p(ign, _i32p), _p(sp, _i32p), _p(sd, _u64p),
                                  _p(si, _i32p) if si is not None else None, S, int(max_steps),
                                  _p(burned, _u32p), _p(steps, _u32p), _p(counters, _u64p), int(nthreads))
    if rc < 0:
        raise MemoryError("orc_simulate_batch failed")
    return {"burned": burned, "steps": steps, "trials": counters[:, 0].copy(),
            "cand_steps": counters[:, 1].copy(), "distinct": counters[:, 2].copy(), "threads": rc}


# --------------------------------------------------------------------------- C-5
def fitness_counts(reference, burned, W: int) -> tuple[int, int, int]:
    ref = _c(reference, np.uint32); b = _c(burned, np.uint32)
    H = ref.shape[0]
    out = np.zeros(3, np.uint32)
    lib().orc_fitness_counts(_p(ref, _u32p), _p(b, _u32p), int(W), int(H), _p(out, _u32p))
    return int(out[0]), int(out[1]), int(out[2])


def fitness_score(I: int, Nstar: int, N: int, metric: int) -> np.float32:
    return np.float32(lib().orc_fitness_score(I, Nstar, N, metric))


def fitness(reference, burned_batch, W: int, metric: int):
    """counts u32[S][2] = (I, Nstar), scores f32[S], N."""
    burned_batch = _c(burned_batch, np.uint32)
    S = burned_batch.shape[0]
    counts = np.zeros((S, 2), np.uint32); scores = np.zeros(S, np.float32); N = 0
    with np.errstate(all="ignore"):
        for s in range(S):
            I, Ns, N = fitness_counts(reference, burned_batch[s], W)
            counts[s] = (I, Ns)
            scores[s] = fitness_score(I, Ns, N, metric)
    return counts, scores, N


def group_stats(counts, N: int, G: int, R: int):
    cnt = _c(counts, np.uint32).reshape(G * R, 2)
    sums = np.zeros((G, 2), np.uint64); mv = np.zeros((G, 2), np.float64)
    lib().orc_group_stats(_p(cnt, _u32p), int(N), G, R, _p(sums, _u64p), _p(mv, _f64p))
    return sums, mv


def max_threads() -> int:
    return int(lib().orc_max_threads())
