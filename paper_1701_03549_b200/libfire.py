"""Thin Python binding of the C ABI in include/fire.h: same names, argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libfire.so; PyTorch is used for device
memory and streams.  There is NO CPU fallback: if libfire_sm100a.so cannot be loaded, or there is no
CUDA device, every call raises.  This module never imports anything under ``oracle/``.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import torch

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libfire_sm100a.so"

FIRE_OK, FIRE_EINVAL, FIRE_ENOMEM, FIRE_ESTATE, FIRE_ECUDA, FIRE_ELIMIT = 0, -1, -2, -3, -4, -5
FIRE_FITNESS_STATIC_MAX_SIMS = 16384
FIRE_METRIC_DELTA, FIRE_METRIC_JACCARD = 0, 1

# every symbol include/fire.h declares (tests check the library exports exactly these)
SYMBOLS = [
    "fire_landscape_create", "fire_landscape_destroy", "fire_params_upload", "fire_simulate_batch",
    "fire_fitness", "fire_fitness_static", "fire_fitness_group_stats", "fire_thresholds_download", "fire_generation_host",
    "fire_launch_count", "fire_set_launch_geometry", "fire_set_list_capacity", "fire_set_schedule", "fire_set_kernel", "fire_set_burn_time", "fire_set_time_output", "fire_set_fused_counts", "fire_landscape_set_elevation", "fire_landscape_set_class_indicator", "fire_burn_count", "fire_error_string",
    "fire_set_profiling", "fire_profile_read",
]


class FireError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {error_string(code)} ({code})")


_lib = None
_vp = C.c_void_p


def load() -> C.CDLL:
    """dlopen libfire_sm100a.so (built in-tree by paper_1701_03549_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise FileNotFoundError(f"{LIB_PATH} is missing: run `python -m paper_1701_03549_b200.build` "
                                "(needs nvcc; there is no CPU fallback)")
    lib = C.CDLL(str(LIB_PATH))
    lib.fire_landscape_create.argtypes = [C.POINTER(_vp), _vp, _vp, _vp, _vp, C.c_int32, C.c_int32, _vp]
    lib.fire_landscape_destroy.argtypes = [_vp]
    lib.fire_params_upload.argtypes = [_vp, _vp, C.c_int32, _vp]
    lib.fire_simulate_batch.argtypes = [_vp, _vp, _vp, _vp, _vp, C.c_int32, C.c_uint32, _vp, _vp, _vp, _vp]
    lib.fire_fitness.argtypes = [_vp, _vp, _vp, C.c_int32, C.c_int32, _vp, _vp, _vp, _vp]
    lib.fire_fitness_static.argtypes = [_vp, _vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, _vp, _vp, _vp]
    lib.fire_fitness_group_stats.argtypes = [_vp, C.c_uint32, C.c_int32, C.c_int32, _vp, _vp, _vp]
    lib.fire_thresholds_download.argtypes = [_vp, C.c_int32, _vp, _vp]
    lib.fire_generation_host.argtypes = [_vp, _vp, C.c_int32, _vp, _vp, _vp, _vp, C.c_int32, C.c_uint32, _vp,
                                         C.c_int32, _vp, _vp, _vp, C.POINTER(_vp), _vp]
    lib.fire_launch_count.argtypes = [_vp]
    lib.fire_launch_count.restype = C.c_int64
    lib.fire_set_launch_geometry.argtypes = [_vp, C.c_int32, C.c_int32]
    lib.fire_set_list_capacity.argtypes = [_vp, C.c_int32, C.c_int32]
    lib.fire_set_schedule.argtypes = [_vp, C.c_int32]
    lib.fire_set_kernel.argtypes = [_vp, C.c_int32]
    lib.fire_set_burn_time.argtypes = [_vp, _vp, C.c_int32, _vp]
    lib.fire_set_time_output.argtypes = [_vp, _vp]
    lib.fire_set_fused_counts.argtypes = [_vp, _vp, _vp]
    lib.fire_landscape_set_elevation.argtypes = [_vp, _vp, _vp]
    lib.fire_landscape_set_class_indicator.argtypes = [_vp, _vp, C.c_int32, _vp]
    lib.fire_burn_count.argtypes = [_vp, _vp, C.c_int32, _vp, _vp]
    lib.fire_set_profiling.argtypes = [_vp, C.c_int32]
    lib.fire_profile_read.argtypes = [_vp, C.POINTER(C.c_float), C.c_int32, C.POINTER(C.c_int32)]
    lib.fire_error_string.argtypes = [C.c_int]
    lib.fire_error_string.restype = C.c_char_p
    for name in SYMBOLS:
        if name not in ("fire_launch_count", "fire_error_string"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def error_string(code: int) -> str:
    return load().fire_error_string(int(code)).decode()


def _check(rc: int, where: str) -> None:
    if rc != FIRE_OK:
        raise FireError(rc, where)


def _dev(t: torch.Tensor | None, dtype: torch.dtype, name: str, shape=None) -> int | None:
    """Device pointer of a contiguous CUDA tensor of the given dtype (None passes through as NULL)."""
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA tensor (there is no CPU path)")
    if t.dtype != dtype:
        raise TypeError(f"{name}: expected dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{name}: tensor must be contiguous")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


def _host(t: torch.Tensor | None, dtype: torch.dtype, name: str, shape=None) -> int | None:
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or t.is_cuda:
        raise TypeError(f"{name}: expected a host tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected contiguous {dtype}")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


class Landscape:
    """Owner of a ``fire_landscape*`` handle; remembers W, H for shape checks."""

    def __init__(self, handle: int, W: int, H: int, device: torch.device):
        self.handle, self.W, self.H, self.device = handle, W, H, device
        self.Ww = (W + 31) // 32
        self.P = 0

    def close(self) -> None:
        if self.handle:
            fire_landscape_destroy(self)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fire_landscape_create(veg: torch.Tensor, slope: torch.Tensor, aspect: torch.Tensor, wind: torch.Tensor,
                          stream=None) -> Landscape:
    """veg u8[H][W], slope/aspect/wind f32[H][W] (radians) on the GPU -> handle (include/fire.h, a1)."""
    if not torch.cuda.is_available():
        raise FireError(FIRE_ECUDA, "fire_landscape_create (no CUDA device; there is no CPU fallback)")
    H, W = veg.shape
    args = [_dev(veg, torch.uint8, "veg"), _dev(slope, torch.float32, "slope", (H, W)),
            _dev(aspect, torch.float32, "aspect", (H, W)), _dev(wind, torch.float32, "wind", (H, W))]
    out = _vp()
    with torch.cuda.device(veg.device):
        _check(load().fire_landscape_create(C.byref(out), *args, W, H, _stream(stream)), "fire_landscape_create")
    return Landscape(out.value, W, H, veg.device)


def fire_landscape_destroy(L: Landscape) -> None:
    h, L.handle = L.handle, 0
    if h:
        _check(load().fire_landscape_destroy(h), "fire_landscape_destroy")


def fire_params_upload(L: Landscape, beta: torch.Tensor, stream=None) -> None:
    """beta f32[P][5] on the GPU -> thresholds u32[P][H][W][8] inside the handle (a2, Eq. 1)."""
    if beta.dim() != 2 or beta.shape[1] != 5:
        raise ValueError("beta: expected shape [P][5]")
    P = int(beta.shape[0])
    _check(load().fire_params_upload(L.handle, _dev(beta, torch.float32, "beta"), P, _stream(stream)),
           "fire_params_upload")
    L.P = P


def fire_simulate_batch(L: Landscape, ignitions: torch.Tensor, sim_param: torch.Tensor, seeds: torch.Tensor,
                        out_burned: torch.Tensor, out_steps: torch.Tensor | None = None,
                        out_trials: torch.Tensor | None = None, sim_ids: torch.Tensor | None = None,
                        max_steps: int = 0, stream=None) -> None:
    """ignitions i32[S][2], sim_param i32[S], seeds i64[S] (bit pattern of the u64 seed) ->
    out_burned i32[S][H][ceil(W/32)] (bit pattern of u32 words), out_steps i32[S], out_trials i64[S] (a3-a6)."""
    S = int(sim_param.shape[0])
    _check(load().fire_simulate_batch(
        L.handle, _dev(ignitions, torch.int32, "ignitions", (S, 2)), _dev(sim_param, torch.int32, "sim_param", (S,)),
        _dev(seeds, torch.int64, "seeds", (S,)), _dev(sim_ids, torch.int32, "sim_ids", (S,)), S, int(max_steps),
        _dev(out_burned, torch.int32, "out_burned", (S, L.H, L.Ww)), _dev(out_steps, torch.int32, "out_steps", (S,)),
        _dev(out_trials, torch.int64, "out_trials", (S,)), _stream(stream)), "fire_simulate_batch")


def fire_fitness(L: Landscape, reference: torch.Tensor, burned: torch.Tensor, metric: int, out_score: torch.Tensor,
                 out_counts: torch.Tensor | None = None, out_ref_area: torch.Tensor | None = None, stream=None) -> None:
    """reference i32[H][Ww], burned i32[S][H][Ww] -> out_score f32[S], out_counts i32[S][2] = (I, N*),
    out_ref_area i32[1] = N (a7, Eq. 2)."""
    S = int(burned.shape[0])
    _check(load().fire_fitness(
        L.handle, _dev(reference, torch.int32, "reference", (L.H, L.Ww)),
        _dev(burned, torch.int32, "burned", (S, L.H, L.Ww)), S, int(metric),
        _dev(out_score, torch.float32, "out_score", (S,)), _dev(out_counts, torch.int32, "out_counts", (S, 2)),
        _dev(out_ref_area, torch.int32, "out_ref_area", (1,)), _stream(stream)), "fire_fitness")


def fire_fitness_static(reference: torch.Tensor, burned: torch.Tensor, W: int, metric: int, out_score: torch.Tensor,
                        out_ref_area: torch.Tensor | None = None, stream=None) -> None:
    """fire_fitness without a handle and without any device allocation (scratch in a static device array of the library):
    reference i32[H][Ww], burned i32[S][H][Ww] -> out_score f32[S], out_ref_area i32[1]; S <= FIRE_FITNESS_STATIC_MAX_SIMS."""
    S, H, Ww = (int(v) for v in burned.shape)
    if Ww != (int(W) + 31) // 32:
        raise ValueError("burned: last dimension must be ceil(W / 32)")
    with torch.cuda.device(burned.device):
        _check(load().fire_fitness_static(
            _dev(reference, torch.int32, "reference", (H, Ww)), _dev(burned, torch.int32, "burned", (S, H, Ww)),
            int(W), H, S, int(metric), _dev(out_score, torch.float32, "out_score", (S,)),
            _dev(out_ref_area, torch.int32, "out_ref_area", (1,)), _stream(stream)), "fire_fitness_static")


def fire_fitness_group_stats(counts: torch.Tensor, ref_area: int, G: int, R: int, out_sums: torch.Tensor,
                             out_mean_var: torch.Tensor, stream=None) -> None:
    """counts i32[G*R][2] -> out_sums i64[G][2] = (sum x, sum x^2), out_mean_var f64[G][2] (a8)."""
    with torch.cuda.device(counts.device):
        _check(load().fire_fitness_group_stats(
            _dev(counts, torch.int32, "counts", (G * R, 2)), int(ref_area), G, R,
            _dev(out_sums, torch.int64, "out_sums", (G, 2)), _dev(out_mean_var, torch.float64, "out_mean_var", (G, 2)),
            _stream(stream)), "fire_fitness_group_stats")


def fire_thresholds_download(L: Landscape, p: int, out: torch.Tensor, stream=None) -> None:
    """Test hook: thresholds of parameter vector p -> out i32[H][W][8] (bit pattern of u32)."""
    _check(load().fire_thresholds_download(L.handle, int(p), _dev(out, torch.int32, "out", (L.H, L.W, 8)),
                                           _stream(stream)), "fire_thresholds_download")


def fire_generation_host(L: Landscape, beta: torch.Tensor, ignitions: torch.Tensor, sim_param: torch.Tensor,
                         seeds: torch.Tensor, reference: torch.Tensor, metric: int, out_score: torch.Tensor,
                         out_counts: torch.Tensor | None = None, out_steps: torch.Tensor | None = None,
                         sim_ids: torch.Tensor | None = None, max_steps: int = 0, stream=None) -> int:
    """One GA generation with HOST (ideally pinned) tensors; synchronises.  Returns the device pointer of the
    burnt maps u32[S][H][Ww], owned by the handle and valid until the next call on it."""
    P, S = int(beta.shape[0]), int(sim_param.shape[0])
    burned_dev = _vp()
    with torch.cuda.device(L.device):
        _check(load().fire_generation_host(
            L.handle, _host(beta, torch.float32, "beta", (P, 5)), P, _host(ignitions, torch.int32, "ignitions", (S, 2)),
            _host(sim_param, torch.int32, "sim_param", (S,)), _host(seeds, torch.int64, "seeds", (S,)),
            _host(sim_ids, torch.int32, "sim_ids", (S,)), S, int(max_steps),
            _host(reference, torch.int32, "reference", (L.H, L.Ww)), int(metric),
            _host(out_score, torch.float32, "out_score", (S,)), _host(out_counts, torch.int32, "out_counts", (S, 2)),
            _host(out_steps, torch.int32, "out_steps", (S,)), C.byref(burned_dev), _stream(stream)),
            "fire_generation_host")
    L.P = P
    return int(burned_dev.value)


def fire_launch_count(L: Landscape) -> int:
    return int(load().fire_launch_count(L.handle))


def fire_set_launch_geometry(L: Landscape, threads_per_cta: int = 0, ctas_per_sm: int = 0) -> None:
    _check(load().fire_set_launch_geometry(L.handle, int(threads_per_cta), int(ctas_per_sm)), "fire_set_launch_geometry")


def fire_set_schedule(L: Landscape, mode: int = 0) -> None:
    _check(load().fire_set_schedule(L.handle, int(mode)), "fire_set_schedule")


def fire_landscape_set_elevation(L: Landscape, elevation: torch.Tensor, stream=None) -> None:
    _check(load().fire_landscape_set_elevation(L.handle, _dev(elevation, torch.float32, "elevation", (L.H, L.W)), _stream(stream)),
           "fire_landscape_set_elevation")


def fire_landscape_set_class_indicator(L: Landscape, class_if, stream=None) -> None:
    """class_if: sequence of I_f values per vegetation class, or None / empty for the paper's forest indicator."""
    import numpy as np
    w = np.ascontiguousarray(np.asarray(class_if if class_if is not None else [], dtype=np.float32))
    _check(load().fire_landscape_set_class_indicator(L.handle, w.ctypes.data if w.size else None, int(w.size), _stream(stream)),
           "fire_landscape_set_class_indicator")


def fire_burn_count(L: Landscape, burned: torch.Tensor, out_count: torch.Tensor, stream=None) -> None:
    S = int(burned.shape[0])
    _check(load().fire_burn_count(L.handle, _dev(burned, torch.int32, "burned", (S, L.H, L.Ww)), S,
                                  _dev(out_count, torch.int32, "out_count", (L.H, L.W)), _stream(stream)), "fire_burn_count")


def fire_set_burn_time(L: Landscape, burn_time, stream=None) -> None:
    """burn_time: sequence of steps per vegetation class (1..8), or None / empty for the base model."""
    import numpy as np
    bt = np.ascontiguousarray(np.asarray(burn_time if burn_time is not None else [], dtype=np.uint8))
    _check(load().fire_set_burn_time(L.handle, bt.ctypes.data if bt.size else None, int(bt.size), _stream(stream)), "fire_set_burn_time")


def fire_set_time_output(L: Landscape, out_time: torch.Tensor | None) -> None:
    """out_time: int32 CUDA tensor [S_max][H][W] kept alive by the caller, or None to switch the output off."""
    ptr = None
    if out_time is not None:
        if out_time.dtype != torch.int32 or not out_time.is_cuda or not out_time.is_contiguous() or tuple(out_time.shape[1:]) != (L.H, L.W):
            raise TypeError("out_time must be a contiguous int32 CUDA tensor of shape [S][H][W]")
        ptr = out_time.data_ptr()
    _check(load().fire_set_time_output(L.handle, ptr), "fire_set_time_output")


def fire_set_fused_counts(L: Landscape, reference: torch.Tensor | None, out_counts: torch.Tensor | None) -> None:
    """reference i32[H][Ww], out_counts i32[S_max][2]: CUDA tensors kept alive by the caller; both None switch the output off."""
    if (reference is None) != (out_counts is None):
        raise TypeError("reference and out_counts are set or cleared together")
    rp = cp = None
    if reference is not None:
        rp = _dev(reference, torch.int32, "reference", (L.H, L.Ww))
        if out_counts.dtype != torch.int32 or not out_counts.is_cuda or not out_counts.is_contiguous() or tuple(out_counts.shape[1:]) != (2,):
            raise TypeError("out_counts must be a contiguous int32 CUDA tensor of shape [S][2]")
        cp = out_counts.data_ptr()
    _check(load().fire_set_fused_counts(L.handle, rp, cp), "fire_set_fused_counts")


def fire_set_kernel(L: Landscape, family: int = 0) -> None:
    _check(load().fire_set_kernel(L.handle, int(family)), "fire_set_kernel")


def fire_set_list_capacity(L: Landscape, shared_entries: int = 0, total_entries: int = 0) -> None:
    _check(load().fire_set_list_capacity(L.handle, int(shared_entries), int(total_entries)), "fire_set_list_capacity")


def fire_set_profiling(L: Landscape, enabled: bool) -> None:
    with torch.cuda.device(L.device):
        _check(load().fire_set_profiling(L.handle, 1 if enabled else 0), "fire_set_profiling")


def fire_profile_read(L: Landscape, max_entries: int = 64) -> list[float]:
    """Elapsed milliseconds of the propagation kernels recorded since the last read, oldest first (synchronises)."""
    buf = (C.c_float * max_entries)()
    n = C.c_int32(0)
    with torch.cuda.device(L.device):
        _check(load().fire_profile_read(L.handle, buf, max_entries, C.byref(n)), "fire_profile_read")
    return [float(buf[i]) for i in range(n.value)]
