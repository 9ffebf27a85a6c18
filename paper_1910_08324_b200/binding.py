"""Thin ctypes binding of the C ABI in ``include/spd.h`` - argument marshalling only.

Every function has the name and the argument order of its C counterpart; device
buffers are ``torch`` CUDA tensors (PyTorch supplies device memory and streams,
nothing else), host buffers are numpy arrays or CPU tensors.  All arithmetic of
the method runs in the CUDA kernels of ``csrc/``; if the shared library is not
built or no sm_100 device is present the calls raise - there is no fallback.
"""
from __future__ import annotations

import ctypes
import os
from typing import List, Optional, Sequence, Tuple

import numpy as np

from . import _build

SPD_OK = 0
SPD_ERR_INVALID_ARG = -1
SPD_ERR_UNSUPPORTED_DEVICE = -2
SPD_ERR_ALLOC = -3
SPD_ERR_CUDA = -4

SPD_WIDTHS_ALL, SPD_WIDTHS_POW2, SPD_WIDTHS_BOXDIT, SPD_WIDTHS_IGRID, SPD_WIDTHS_GEOMETRIC = range(5)
WIDTH_KINDS = {"ALL": 0, "POW2": 1, "BOXDIT": 2, "IGRID": 3, "GEOMETRIC": 4}
SPD_FLAG_FORCE_GENERIC = 0x1
SPD_FLAG_BLOCK_TREE = 0x2
SPD_FLAG_GENERIC_WORKSPACE = 0x4
SPD_FLAG_WIDTH_U8 = 0x8
SPD_OPT_SEGMENTS_PER_ROW = 1
SPD_OPT_HOST_ROWS_PER_BLOCK = 2
SPD_PATH_DYADIC_TREE, SPD_PATH_GENERIC, SPD_PATH_IGRID_TREE, SPD_PATH_GRID = 1, 2, 3, 4
SPD_GRID_EVERY_SAMPLE, SPD_GRID_DIT, SPD_GRID_BOXDIT, SPD_GRID_IGRID = range(4)
GRID_KINDS = {"EVERY_SAMPLE": 0, "DIT": 1, "BOXDIT": 2, "IGRID": 3}

# every symbol include/spd.h declares
EXPORTS = (
    "spd_width_set_generate", "spd_plan_create", "spd_plan_create_ex", "spd_plan_destroy",
    "spd_plan_get_widths", "spd_plan_get_info", "spd_run", "spd_find_candidates",
    "spd_run_flagged", "spd_find_candidates_flagged", "spd_row_stats",
    "spd_run_host", "spd_last_error_string", "spd_version",
    "spd_separation_generate", "spd_plan_create_grid", "spd_width_sigma", "spd_run_sigma_w",
    "spd_destroy", "spd_plan_set_option", "spd_row_stats_converge", "spd_cluster_candidates",
    "spd_run_host_candidates", "spd_plan_create_grid_ex", "spd_row_stats_static",
    "spd_plan_get_iterations", "spd_run_iterations",
)


class SpdError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"spd status {status}: {message}")
        self.status = status


class spd_candidate(ctypes.Structure):
    _fields_ = [("dm", ctypes.c_int32), ("t", ctypes.c_int32), ("snr", ctypes.c_float),
                ("width_idx", ctypes.c_int32)]


CANDIDATE_DTYPE = np.dtype([("dm", "<i4"), ("t", "<i4"), ("snr", "<f4"), ("width_idx", "<i4")])


class spd_plan_info(ctypes.Structure):
    _fields_ = [("n_dm", ctypes.c_int64), ("n_t", ctypes.c_int64),
                ("n_widths", ctypes.c_int32), ("max_width", ctypes.c_int32),
                ("path", ctypes.c_int32), ("launches_per_run", ctypes.c_int32),
                ("threads_per_block", ctypes.c_int32), ("blocks", ctypes.c_int32),
                ("chunk", ctypes.c_int32), ("segments_per_row", ctypes.c_int32),
                ("smem_bytes", ctypes.c_int64), ("workspace_bytes", ctypes.c_int64),
                ("activity_bytes", ctypes.c_int64), ("activity_block", ctypes.c_int32),
                ("activity_per_row", ctypes.c_int32),
                ("tree_kernel", ctypes.c_int32),
                ("piece_chunks", ctypes.c_int32),
                ("width_bytes", ctypes.c_int32),
                ("flags", ctypes.c_uint32)]


_lib: Optional[ctypes.CDLL] = None
_vp, _i32, _i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64


def library_path() -> str:
    return _build.LIB_PATH


def load(build_if_missing: bool = True) -> ctypes.CDLL:
    """dlopen ``libspd_b200.so`` (building it first if needed) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        _build.build()
    if not os.path.exists(_build.LIB_PATH):
        raise SpdError(SPD_ERR_UNSUPPORTED_DEVICE,
                       f"{_build.LIB_PATH} is not built; run paper_1910_08324_b200.build() (no CPU fallback)")
    lib = ctypes.CDLL(_build.LIB_PATH)
    lib.spd_version.restype = ctypes.c_int
    lib.spd_last_error_string.restype = ctypes.c_char_p
    lib.spd_width_set_generate.restype = ctypes.c_int
    lib.spd_width_set_generate.argtypes = [_i32, _i32, _i32, _vp, _i32, ctypes.POINTER(_i32)]
    lib.spd_plan_create.restype = ctypes.c_int
    lib.spd_plan_create.argtypes = [ctypes.POINTER(_vp), _i64, _i64, _vp, _i32, _i32]
    lib.spd_plan_create_ex.restype = ctypes.c_int
    lib.spd_plan_create_ex.argtypes = [ctypes.POINTER(_vp), _i64, _i64, _vp, _i32, _i32, ctypes.c_uint32]
    lib.spd_plan_create_grid.restype = ctypes.c_int
    lib.spd_plan_create_grid.argtypes = [ctypes.POINTER(_vp), _i64, _i64, _vp, _vp, _i32, _i32]
    lib.spd_plan_create_grid_ex.restype = ctypes.c_int
    lib.spd_plan_create_grid_ex.argtypes = [ctypes.POINTER(_vp), _i64, _i64, _vp, _vp, _i32, _i32, ctypes.c_uint32]
    lib.spd_separation_generate.restype = ctypes.c_int
    lib.spd_separation_generate.argtypes = [_i32, _i32, _vp, _i32, _vp]
    lib.spd_width_sigma.restype = ctypes.c_int
    lib.spd_width_sigma.argtypes = [_vp, _vp, _vp, _vp, _vp]
    lib.spd_run_sigma_w.restype = ctypes.c_int
    lib.spd_run_sigma_w.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.spd_plan_destroy.restype = None
    lib.spd_plan_destroy.argtypes = [_vp]
    lib.spd_plan_get_widths.restype = ctypes.c_int
    lib.spd_plan_get_widths.argtypes = [_vp, _vp, ctypes.POINTER(_i32)]
    lib.spd_plan_get_info.restype = ctypes.c_int
    lib.spd_plan_get_info.argtypes = [_vp, ctypes.POINTER(spd_plan_info)]
    lib.spd_run.restype = ctypes.c_int
    lib.spd_run.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.spd_find_candidates.restype = ctypes.c_int
    lib.spd_find_candidates.argtypes = [_vp, _vp, _vp, ctypes.c_float, _vp, _i64, _vp, _vp]
    lib.spd_run_flagged.restype = ctypes.c_int
    lib.spd_run_flagged.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_float, _vp, _vp]
    lib.spd_find_candidates_flagged.restype = ctypes.c_int
    lib.spd_find_candidates_flagged.argtypes = [_vp, _vp, _vp, _vp, ctypes.c_float, _vp, _i64, _vp, _vp]
    lib.spd_row_stats.restype = ctypes.c_int
    lib.spd_row_stats.argtypes = [_vp, _vp, ctypes.c_float, _i32, _vp, _vp, _vp]
    lib.spd_run_host.restype = ctypes.c_int
    lib.spd_run_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp]
    lib.spd_destroy.restype = None
    lib.spd_destroy.argtypes = [_vp]
    lib.spd_plan_set_option.restype = ctypes.c_int
    lib.spd_plan_set_option.argtypes = [_vp, _i32, _i64]
    lib.spd_plan_get_iterations.restype = ctypes.c_int
    lib.spd_plan_get_iterations.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp, _vp]
    lib.spd_run_iterations.restype = ctypes.c_int
    lib.spd_run_iterations.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.spd_row_stats_static.restype = ctypes.c_int
    lib.spd_row_stats_static.argtypes = [_vp, _i64, _i64, ctypes.c_float, _i32, _vp, _vp, _vp]
    lib.spd_row_stats_converge.restype = ctypes.c_int
    lib.spd_row_stats_converge.argtypes = [_vp, _vp, ctypes.c_float, _i32, ctypes.c_float, _vp, _vp, _vp, _vp]
    lib.spd_cluster_candidates.restype = ctypes.c_int
    lib.spd_cluster_candidates.argtypes = [_vp, _vp, _vp, _vp, _i64, _i32, _vp, _i64, _vp, _vp]
    lib.spd_run_host_candidates.restype = ctypes.c_int
    lib.spd_run_host_candidates.argtypes = [_vp, _vp, _vp, _vp, ctypes.c_float, _i32, _vp, _i64,
                                            ctypes.POINTER(_i64), ctypes.POINTER(_i64)]
    _lib = lib
    return lib


def spd_last_error_string() -> str:
    return load().spd_last_error_string().decode("utf-8", "replace")


def _check(status: int) -> None:
    if status != SPD_OK:
        raise SpdError(status, spd_last_error_string())


def spd_version() -> int:
    return int(load().spd_version())


def spd_width_set_generate(kind, param: int, max_width: int) -> np.ndarray:
    """Ascending int32 width set; ``kind`` is an SPD_WIDTHS_* value or its name."""
    lib = load()
    k = WIDTH_KINDS[kind.upper()] if isinstance(kind, str) else int(kind)
    n = _i32(0)
    _check(lib.spd_width_set_generate(k, int(param), int(max_width), None, 0, ctypes.byref(n)))
    out = np.empty(n.value, dtype=np.int32)
    _check(lib.spd_width_set_generate(k, int(param), int(max_width), out.ctypes.data, n.value, ctypes.byref(n)))
    return out


def spd_plan_create(n_dm: int, n_t: int, width_set: Sequence[int], max_width: int, flags: int = 0) -> int:
    """Returns the opaque plan handle (an integer address)."""
    lib = load()
    w = np.ascontiguousarray(np.asarray(width_set, dtype=np.int32).reshape(-1))
    handle = _vp(0)
    if flags:
        st = lib.spd_plan_create_ex(ctypes.byref(handle), int(n_dm), int(n_t), w.ctypes.data, int(w.size),
                                    int(max_width), int(flags))
    else:
        st = lib.spd_plan_create(ctypes.byref(handle), int(n_dm), int(n_t), w.ctypes.data, int(w.size),
                                 int(max_width))
    _check(st)
    return int(handle.value)


def spd_separation_generate(kind, param: int, widths: Sequence[int]) -> np.ndarray:
    """Boxcar separation of every width; ``kind`` is an SPD_GRID_* value or its name."""
    lib = load()
    k = GRID_KINDS[kind.upper()] if isinstance(kind, str) else int(kind)
    w = np.ascontiguousarray(np.asarray(widths, dtype=np.int32).reshape(-1))
    out = np.empty(w.size, dtype=np.int32)
    _check(lib.spd_separation_generate(k, int(param), w.ctypes.data, int(w.size), out.ctypes.data))
    return out


def spd_plan_create_grid(n_dm: int, n_t: int, width_set: Sequence[int], separations: Sequence[int],
                         max_width: int, flags: int = 0) -> int:
    """Plan with a boxcar separation per width; returns the opaque handle (flags: spd_plan_create_grid_ex)."""
    lib = load()
    w = np.ascontiguousarray(np.asarray(width_set, dtype=np.int32).reshape(-1))
    sp = np.ascontiguousarray(np.asarray(separations, dtype=np.int32).reshape(-1))
    if w.size != sp.size:
        raise ValueError("width_set and separations differ in length")
    handle = _vp(0)
    if flags:
        _check(lib.spd_plan_create_grid_ex(ctypes.byref(handle), int(n_dm), int(n_t), w.ctypes.data, sp.ctypes.data,
                                           int(w.size), int(max_width), int(flags)))
    else:
        _check(lib.spd_plan_create_grid(ctypes.byref(handle), int(n_dm), int(n_t), w.ctypes.data, sp.ctypes.data,
                                        int(w.size), int(max_width)))
    return int(handle.value)


def spd_plan_destroy(plan: int) -> None:
    if plan:
        load().spd_plan_destroy(_vp(plan))


def spd_destroy(plan: int) -> None:
    """north_star's name for spd_plan_destroy (the C symbol of the same name)."""
    if plan:
        load().spd_destroy(_vp(plan))


def spd_plan_set_option(plan: int, option: int, value: int) -> None:
    _check(load().spd_plan_set_option(_vp(plan), int(option), int(value)))


def spd_plan_get_widths(plan: int) -> np.ndarray:
    lib = load()
    n = _i32(0)
    _check(lib.spd_plan_get_widths(_vp(plan), None, ctypes.byref(n)))
    out = np.empty(n.value, dtype=np.int32)
    _check(lib.spd_plan_get_widths(_vp(plan), out.ctypes.data, ctypes.byref(n)))
    return out


def spd_plan_get_info(plan: int) -> dict:
    info = spd_plan_info()
    _check(load().spd_plan_get_info(_vp(plan), ctypes.byref(info)))
    return {name: int(getattr(info, name)) for name, _ in spd_plan_info._fields_}


def _dev_ptr(t, dtype, numel: Optional[int], name: str) -> int:
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous {dtype}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name} has {t.numel()} elements, expected {numel}")
    return t.data_ptr()


def _width_dtype(info):
    import torch
    return torch.uint8 if info["width_bytes"] == 1 else torch.int32


def _stream_handle(stream) -> int:
    import torch
    if stream is None:
        return int(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


def spd_run(plan: int, plane, mean, sigma, out_snr, out_width, stream=None) -> None:
    """Enqueue the hot path on device tensors (asynchronous on ``stream`` / torch's current stream)."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    _check(load().spd_run(
        _vp(plan),
        _dev_ptr(plane, torch.float32, n, "plane"),
        _dev_ptr(mean, torch.float32, info["n_dm"], "mean"),
        _dev_ptr(sigma, torch.float32, info["n_dm"], "sigma"),
        _dev_ptr(out_snr, torch.float32, n, "out_snr"),
        _dev_ptr(out_width, _width_dtype(info), n, "out_width"),
        _vp(_stream_handle(stream))))


def spd_find_candidates(plan: int, out_snr, out_width, threshold: float, capacity: int, stream=None):
    """Returns (list tensor uint8 [capacity*16] on the device, n_found int64 device tensor[1])."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    lst = torch.empty(max(int(capacity), 1) * ctypes.sizeof(spd_candidate), dtype=torch.uint8,
                      device=out_snr.device)
    n_found = torch.zeros(1, dtype=torch.int64, device=out_snr.device)
    _check(load().spd_find_candidates(
        _vp(plan), _dev_ptr(out_snr, torch.float32, n, "out_snr"),
        _dev_ptr(out_width, _width_dtype(info), n, "out_width"), ctypes.c_float(threshold),
        _vp(lst.data_ptr()), int(capacity), _vp(n_found.data_ptr()), _vp(_stream_handle(stream))))
    return lst, n_found


def spd_run_flagged(plan: int, plane, mean, sigma, out_snr, out_width, threshold: float, activity,
                    stream=None) -> None:
    """spd_run plus the fused threshold test: also fills the ``activity`` map (uint8 device tensor of
    ``spd_plan_get_info(plan)["activity_bytes"]`` bytes)."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    _check(load().spd_run_flagged(
        _vp(plan),
        _dev_ptr(plane, torch.float32, n, "plane"),
        _dev_ptr(mean, torch.float32, info["n_dm"], "mean"),
        _dev_ptr(sigma, torch.float32, info["n_dm"], "sigma"),
        _dev_ptr(out_snr, torch.float32, n, "out_snr"),
        _dev_ptr(out_width, _width_dtype(info), n, "out_width"),
        ctypes.c_float(threshold),
        _dev_ptr(activity, torch.uint8, info["activity_bytes"], "activity"),
        _vp(_stream_handle(stream))))


def spd_find_candidates_flagged(plan: int, out_snr, out_width, activity, threshold: float, capacity: int,
                                stream=None, lst=None, n_found=None):
    """Candidate stage over the blocks marked in ``activity``; returns (list, n_found) as spd_find_candidates."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    if lst is None:
        lst = torch.empty(max(int(capacity), 1) * ctypes.sizeof(spd_candidate), dtype=torch.uint8,
                          device=out_snr.device)
    if n_found is None:
        n_found = torch.zeros(1, dtype=torch.int64, device=out_snr.device)
    _check(load().spd_find_candidates_flagged(
        _vp(plan), _dev_ptr(out_snr, torch.float32, n, "out_snr"),
        _dev_ptr(out_width, _width_dtype(info), n, "out_width"),
        _dev_ptr(activity, torch.uint8, info["activity_bytes"], "activity"), ctypes.c_float(threshold),
        _vp(lst.data_ptr()), int(capacity), _vp(n_found.data_ptr()), _vp(_stream_handle(stream))))
    return lst, n_found


def spd_row_stats(plan: int, plane, clip_sigma: float = 0.0, n_reject_passes: int = 0, mean=None, sigma=None,
                  stream=None):
    """Per-DM mean and population sigma of ``plane`` (device tensors); returns (mean, sigma)."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    if mean is None:
        mean = torch.empty(info["n_dm"], dtype=torch.float32, device=plane.device)
    if sigma is None:
        sigma = torch.empty(info["n_dm"], dtype=torch.float32, device=plane.device)
    _check(load().spd_row_stats(
        _vp(plan), _dev_ptr(plane, torch.float32, n, "plane"), ctypes.c_float(clip_sigma), int(n_reject_passes),
        _dev_ptr(mean, torch.float32, info["n_dm"], "mean"), _dev_ptr(sigma, torch.float32, info["n_dm"], "sigma"),
        _vp(_stream_handle(stream))))
    return mean, sigma


def spd_plan_get_iterations(plan: int):
    """Iterations of a grid plan (eq. 12): list of dicts first_width, n_widths, separation, n_points."""
    n = _i32(0)
    _check(load().spd_plan_get_iterations(_vp(plan), 0, ctypes.byref(n), None, None, None, None))
    k = n.value
    fw, nw, sp = (np.zeros(k, dtype=np.int32) for _ in range(3))
    npts = np.zeros(k, dtype=np.int64)
    _check(load().spd_plan_get_iterations(_vp(plan), k, ctypes.byref(n), fw.ctypes.data, nw.ctypes.data,
                                          sp.ctypes.data, npts.ctypes.data))
    return [{"first_width": int(fw[i]), "n_widths": int(nw[i]), "separation": int(sp[i]), "n_points": int(npts[i])}
            for i in range(k)]


def spd_run_iterations(plan: int, plane, mean, sigma, out_snr=None, out_width=None, stream=None):
    """Output separated by iteration: returns (planes, out_snr, out_width) where planes[i] = (Y^i, W^i) are
    [n_dm, n_points[i]] views into the concatenated device buffers."""
    import torch
    info = spd_plan_get_info(plan)
    its = spd_plan_get_iterations(plan)
    n_dm = info["n_dm"]
    total = n_dm * sum(it["n_points"] for it in its)
    if out_snr is None:
        out_snr = torch.empty(total, dtype=torch.float32, device=plane.device)
    if out_width is None:
        out_width = torch.empty(total, dtype=torch.int32, device=plane.device)
    _check(load().spd_run_iterations(
        _vp(plan), _dev_ptr(plane, torch.float32, n_dm * info["n_t"], "plane"),
        _dev_ptr(mean, torch.float32, n_dm, "mean"), _dev_ptr(sigma, torch.float32, n_dm, "sigma"),
        _dev_ptr(out_snr, torch.float32, total, "out_snr"), _dev_ptr(out_width, torch.int32, total, "out_width"),
        _vp(_stream_handle(stream))))
    planes, off = [], 0
    for it in its:
        cnt = n_dm * it["n_points"]
        planes.append((out_snr[off:off + cnt].view(n_dm, it["n_points"]),
                       out_width[off:off + cnt].view(n_dm, it["n_points"])))
        off += cnt
    return planes, out_snr, out_width


SPD_STATIC_MAX_ROWS = 8192
SPD_STATIC_MAX_PARTIALS = 65536


def spd_row_stats_static(plane, mean, sigma, clip_sigma: float = 0.0, n_reject_passes: int = 0, stream=None):
    """spd_row_stats without a plan and without any allocation (static device scratch, n_dm <= 8192): the
    caller passes every buffer - ``plane`` [n_dm][n_t], ``mean`` and ``sigma`` [n_dm], float32 device tensors.
    Calls that overlap on the GPU race on the shared scratch (include/spd.h)."""
    import torch
    n_dm, n_t = int(plane.shape[0]), int(plane.shape[1])
    _check(load().spd_row_stats_static(
        _dev_ptr(plane, torch.float32, n_dm * n_t, "plane"), n_dm, n_t, ctypes.c_float(clip_sigma),
        int(n_reject_passes), _dev_ptr(mean, torch.float32, n_dm, "mean"),
        _dev_ptr(sigma, torch.float32, n_dm, "sigma"), _vp(_stream_handle(stream))))
    return mean, sigma


def spd_row_stats_converge(plan: int, plane, clip_sigma: float, max_reject_passes: int, rel_tol: float,
                           mean=None, sigma=None, n_passes=None, stream=None):
    """spd_row_stats repeated until convergence on the device; returns (mean, sigma, n_passes)."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    if mean is None:
        mean = torch.empty(info["n_dm"], dtype=torch.float32, device=plane.device)
    if sigma is None:
        sigma = torch.empty(info["n_dm"], dtype=torch.float32, device=plane.device)
    if n_passes is None:
        n_passes = torch.empty(info["n_dm"], dtype=torch.int32, device=plane.device)
    _check(load().spd_row_stats_converge(
        _vp(plan), _dev_ptr(plane, torch.float32, n, "plane"), ctypes.c_float(clip_sigma), int(max_reject_passes),
        ctypes.c_float(rel_tol), _dev_ptr(mean, torch.float32, info["n_dm"], "mean"),
        _dev_ptr(sigma, torch.float32, info["n_dm"], "sigma"), _dev_ptr(n_passes, torch.int32, info["n_dm"], "n_passes"),
        _vp(_stream_handle(stream))))
    return mean, sigma, n_passes


def spd_cluster_candidates(plan: int, out_snr, lst, n_found, capacity_in: int, dm_radius: int, capacity_out: int,
                           stream=None, lst_out=None, n_out=None):
    """2-D (DM x time) peak stage over a candidate list; returns (list_out, n_out) as spd_find_candidates."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    if lst_out is None:
        lst_out = torch.empty(max(int(capacity_out), 1) * ctypes.sizeof(spd_candidate), dtype=torch.uint8,
                              device=out_snr.device)
    if n_out is None:
        n_out = torch.zeros(1, dtype=torch.int64, device=out_snr.device)
    _check(load().spd_cluster_candidates(
        _vp(plan), _dev_ptr(out_snr, torch.float32, n, "out_snr"), _vp(lst.data_ptr()), _vp(n_found.data_ptr()),
        int(capacity_in), int(dm_radius), _vp(lst_out.data_ptr()), int(capacity_out), _vp(n_out.data_ptr()),
        _vp(_stream_handle(stream))))
    return lst_out, n_out


def spd_width_sigma(plan: int, plane, mean, sigma_w=None, stream=None):
    """Standard deviation per (DM row, width) from power-of-two decimations of ``plane``; returns the
    float32 [n_dm, n_widths] device tensor."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    if sigma_w is None:
        sigma_w = torch.empty((info["n_dm"], info["n_widths"]), dtype=torch.float32, device=plane.device)
    _check(load().spd_width_sigma(
        _vp(plan), _dev_ptr(plane, torch.float32, n, "plane"), _dev_ptr(mean, torch.float32, info["n_dm"], "mean"),
        _dev_ptr(sigma_w, torch.float32, info["n_dm"] * info["n_widths"], "sigma_w"), _vp(_stream_handle(stream))))
    return sigma_w


def spd_run_sigma_w(plan: int, plane, mean, sigma_w, out_snr, out_width, stream=None) -> None:
    """spd_run with a measured standard deviation per (row, width) instead of sqrt(width) * sigma."""
    import torch
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    _check(load().spd_run_sigma_w(
        _vp(plan), _dev_ptr(plane, torch.float32, n, "plane"), _dev_ptr(mean, torch.float32, info["n_dm"], "mean"),
        _dev_ptr(sigma_w, torch.float32, info["n_dm"] * info["n_widths"], "sigma_w"),
        _dev_ptr(out_snr, torch.float32, n, "out_snr"), _dev_ptr(out_width, torch.int32, n, "out_width"),
        _vp(_stream_handle(stream))))


def candidates_to_numpy(lst, n_found, capacity: int) -> Tuple[int, np.ndarray]:
    """Synchronising helper: (count, structured array of the stored candidates sorted by (dm, t))."""
    count = int(n_found.item())
    k = min(count, int(capacity))
    raw = lst[: k * ctypes.sizeof(spd_candidate)].cpu().numpy()
    arr = raw.view(CANDIDATE_DTYPE).copy()
    arr.sort(order=["dm", "t"])
    return count, arr


def _host_ptr(a, dtype, numel: int, name: str) -> Tuple[int, object]:
    try:
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or not a.is_contiguous():
                raise TypeError(f"{name} must be a contiguous CPU tensor or numpy array")
            if a.numel() != numel:
                raise ValueError(f"{name} has {a.numel()} elements, expected {numel}")
            return a.data_ptr(), a
    except ImportError:  # pragma: no cover
        pass
    arr = np.asarray(a)
    if arr.dtype != dtype or not arr.flags.c_contiguous or arr.size != numel:
        raise TypeError(f"{name} must be C-contiguous {dtype} with {numel} elements")
    return arr.ctypes.data, arr


def spd_run_host(plan: int, plane, mean, sigma, out_snr, out_width) -> None:
    """End-to-end call on HOST buffers (blocking): H2D, kernels, D2H inside the library."""
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    p0, _k0 = _host_ptr(plane, np.float32, n, "plane")
    p1, _k1 = _host_ptr(mean, np.float32, info["n_dm"], "mean")
    p2, _k2 = _host_ptr(sigma, np.float32, info["n_dm"], "sigma")
    p3, _k3 = _host_ptr(out_snr, np.float32, n, "out_snr")
    p4, _k4 = _host_ptr(out_width, np.uint8 if info["width_bytes"] == 1 else np.int32, n, "out_width")
    _check(load().spd_run_host(_vp(plan), _vp(p0), _vp(p1), _vp(p2), _vp(p3), _vp(p4)))


def spd_run_host_candidates(plan: int, plane, mean, sigma, threshold: float, dm_radius: int, capacity: int,
                            out_list=None):
    """End-to-end call on HOST buffers that returns the candidate list (blocking).  ``out_list`` may be a
    preallocated (pinned) uint8 buffer of capacity * 16 bytes.  Returns (n_found, n_1d, structured array of the
    stored candidates sorted by (dm, t))."""
    info = spd_plan_get_info(plan)
    n = info["n_dm"] * info["n_t"]
    p0, _k0 = _host_ptr(plane, np.float32, n, "plane")
    p1, _k1 = _host_ptr(mean, np.float32, info["n_dm"], "mean")
    p2, _k2 = _host_ptr(sigma, np.float32, info["n_dm"], "sigma")
    nbytes = max(int(capacity), 1) * ctypes.sizeof(spd_candidate)
    if out_list is None:
        out_list = np.empty(nbytes, dtype=np.uint8)
    p3, keep = _host_ptr(out_list, np.uint8, nbytes, "out_list")
    n_found, n_1d = _i64(0), _i64(0)
    _check(load().spd_run_host_candidates(_vp(plan), _vp(p0), _vp(p1), _vp(p2), ctypes.c_float(threshold),
                                          int(dm_radius), _vp(p3), int(capacity), ctypes.byref(n_found),
                                          ctypes.byref(n_1d)))
    k = min(int(n_found.value), int(capacity))
    raw = keep.numpy() if hasattr(keep, "numpy") else np.asarray(keep)
    arr = raw[: k * ctypes.sizeof(spd_candidate)].view(CANDIDATE_DTYPE).copy()
    arr.sort(order=["dm", "t"])
    return int(n_found.value), int(n_1d.value), arr


class Plan:
    """Owns one ``spd_plan``; convenience wrapper over the functions above."""

    def __init__(self, n_dm: int, n_t: int, width_set: Sequence[int], max_width: Optional[int] = None,
                 flags: int = 0, separations: Optional[Sequence[int]] = None):
        w = np.asarray(width_set, dtype=np.int32)
        mw = int(w.max()) if max_width is None else max_width
        if separations is None:
            self.handle = spd_plan_create(n_dm, n_t, w, mw, flags)
        else:
            self.handle = spd_plan_create_grid(n_dm, n_t, w, separations, mw, flags)
        self.info = spd_plan_get_info(self.handle)
        self.widths = spd_plan_get_widths(self.handle)
        self.n_dm, self.n_t = int(n_dm), int(n_t)

    def set_option(self, option: int, value: int):
        spd_plan_set_option(self.handle, option, value)
        self.info = spd_plan_get_info(self.handle)

    def _new_width(self, device):
        import torch
        return torch.empty((self.n_dm, self.n_t), dtype=_width_dtype(self.info), device=device)

    def run(self, plane, mean, sigma, out_snr=None, out_width=None, stream=None):
        import torch
        if out_snr is None:
            out_snr = torch.empty((self.n_dm, self.n_t), dtype=torch.float32, device=plane.device)
        if out_width is None:
            out_width = self._new_width(plane.device)
        spd_run(self.handle, plane, mean, sigma, out_snr, out_width, stream)
        return out_snr, out_width

    def find_candidates(self, out_snr, out_width, threshold: float, capacity: int, stream=None):
        return spd_find_candidates(self.handle, out_snr, out_width, threshold, capacity, stream)

    def run_flagged(self, plane, mean, sigma, threshold: float, out_snr=None, out_width=None, activity=None,
                    stream=None):
        import torch
        if out_snr is None:
            out_snr = torch.empty((self.n_dm, self.n_t), dtype=torch.float32, device=plane.device)
        if out_width is None:
            out_width = self._new_width(plane.device)
        if activity is None:
            activity = torch.empty(self.info["activity_bytes"], dtype=torch.uint8, device=plane.device)
        spd_run_flagged(self.handle, plane, mean, sigma, out_snr, out_width, threshold, activity, stream)
        return out_snr, out_width, activity

    def find_candidates_flagged(self, out_snr, out_width, activity, threshold: float, capacity: int, stream=None,
                                lst=None, n_found=None):
        return spd_find_candidates_flagged(self.handle, out_snr, out_width, activity, threshold, capacity, stream,
                                           lst, n_found)

    def row_stats(self, plane, clip_sigma: float = 0.0, n_reject_passes: int = 0, mean=None, sigma=None,
                  stream=None):
        return spd_row_stats(self.handle, plane, clip_sigma, n_reject_passes, mean, sigma, stream)

    def row_stats_converge(self, plane, clip_sigma: float, max_reject_passes: int, rel_tol: float, mean=None,
                           sigma=None, n_passes=None, stream=None):
        return spd_row_stats_converge(self.handle, plane, clip_sigma, max_reject_passes, rel_tol, mean, sigma,
                                      n_passes, stream)

    def cluster_candidates(self, out_snr, lst, n_found, capacity_in: int, dm_radius: int, capacity_out: int,
                           stream=None, lst_out=None, n_out=None):
        return spd_cluster_candidates(self.handle, out_snr, lst, n_found, capacity_in, dm_radius, capacity_out,
                                      stream, lst_out, n_out)

    def run_host_candidates(self, plane, mean, sigma, threshold: float, dm_radius: int, capacity: int,
                            out_list=None):
        return spd_run_host_candidates(self.handle, plane, mean, sigma, threshold, dm_radius, capacity, out_list)

    def iterations(self):
        return spd_plan_get_iterations(self.handle)

    def run_iterations(self, plane, mean, sigma, out_snr=None, out_width=None, stream=None):
        return spd_run_iterations(self.handle, plane, mean, sigma, out_snr, out_width, stream)

    def width_sigma(self, plane, mean, sigma_w=None, stream=None):
        return spd_width_sigma(self.handle, plane, mean, sigma_w, stream)

    def run_sigma_w(self, plane, mean, sigma_w, out_snr=None, out_width=None, stream=None):
        import torch
        if out_snr is None:
            out_snr = torch.empty((self.n_dm, self.n_t), dtype=torch.float32, device=plane.device)
        if out_width is None:
            out_width = torch.empty((self.n_dm, self.n_t), dtype=torch.int32, device=plane.device)
        spd_run_sigma_w(self.handle, plane, mean, sigma_w, out_snr, out_width, stream)
        return out_snr, out_width

    def run_host(self, plane, mean, sigma, out_snr, out_width):
        spd_run_host(self.handle, plane, mean, sigma, out_snr, out_width)

    def close(self):
        if getattr(self, "handle", 0):
            spd_plan_destroy(self.handle)
            self.handle = 0

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
