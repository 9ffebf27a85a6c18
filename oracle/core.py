"""ORACLE (test infrastructure only) - numpy front-end of ``spd_oracle.c``.

Builds ``oracle/libspd_oracle.so`` with gcc on first use (``build()``), loads it
with ctypes and exposes the oracle functions on numpy arrays.  Imports nothing
from the CUDA product.  See ``spd_oracle.c`` for the passages followed and the
pins; ``formulas.py`` for the paper's sensitivity formulae.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "spd_oracle.c")
_LIB = os.path.join(_HERE, "libspd_oracle.so")
_lib: Optional[ctypes.CDLL] = None

_i64 = ctypes.c_int64
_i32 = ctypes.c_int32
_f64 = ctypes.c_double
_vp = ctypes.c_void_p


def build(force: bool = False) -> str:
    """Compile the oracle shared library (plain C, -O2, OpenMP over rows)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_spd_direct.restype = None
        lib.oracle_spd_direct.argtypes = [_vp, _i64, _i64, _vp, _vp, _vp, _i32, _i64, _i64, _vp, _vp, _vp]
        lib.oracle_spd_grid_iter.restype = None
        lib.oracle_spd_grid_iter.argtypes = [_vp, _i64, _i64, _vp, _vp, _vp, _vp, _i32, _i32, _vp, _vp, _vp]
        lib.oracle_spd_grid.restype = None
        lib.oracle_spd_grid.argtypes = [_vp, _i64, _i64, _vp, _vp, _vp, _vp, _i32, _i64, _i64, _vp, _vp, _vp]
        lib.oracle_width_sigma.restype = None
        lib.oracle_width_sigma.argtypes = [_vp, _i64, _i64, _vp, _i32, _vp]
        lib.oracle_spd_direct_sw.restype = None
        lib.oracle_spd_direct_sw.argtypes = [_vp, _i64, _i64, _vp, _vp, _vp, _i32, _i64, _i64, _vp, _vp, _vp]
        lib.oracle_spd_prefix.restype = None
        lib.oracle_spd_prefix.argtypes = [_vp, _i64, _i64, _vp, _vp, _vp, _i32, _vp, _vp, _vp]
        lib.oracle_snr_of_width.restype = None
        lib.oracle_snr_of_width.argtypes = [_vp, _i64, _f64, _f64, _i64, _vp, _i64, _vp]
        lib.oracle_row_stats.restype = None
        lib.oracle_row_stats.argtypes = [_vp, _i64, _i64, _vp, _vp]
        lib.oracle_row_stats_clipped.restype = None
        lib.oracle_row_stats_clipped.argtypes = [_vp, _i64, _i64, _f64, _i32, _f64, _f64, _vp, _vp, _vp, _vp]
        lib.oracle_spd_grid_sw.restype = None
        lib.oracle_spd_grid_sw.argtypes = [_vp, _i64, _i64, _vp, _vp, _vp, _vp, _i32, _i64, _i64, _vp, _vp, _vp]
        lib.oracle_cluster_candidates.restype = _i64
        lib.oracle_cluster_candidates.argtypes = [_vp, _i64, _i64, _vp, _i32, _vp, _vp, _vp, _i64, _i32, _vp]
        lib.oracle_find_candidates.restype = _i64
        lib.oracle_find_candidates.argtypes = [_vp, _vp, _i64, _i64, ctypes.c_float, _i64, _vp, _vp, _vp, _vp]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _plane(x) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    if x.ndim == 1:
        x = x[None, :]
    assert x.ndim == 2
    return x


def _stats(v, n_dm: int) -> np.ndarray:
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(v, dtype=np.float64), (n_dm,)))
    return a


def _widths(widths: Sequence[int]) -> np.ndarray:
    w = np.ascontiguousarray(sorted(set(int(v) for v in widths)), dtype=np.int32)
    assert w.size > 0 and w[0] >= 1
    return w


def spd_direct(x, mean, sigma, widths, t0: int = 0, t1: Optional[int] = None
               ) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Oracle A: direct summation.  Returns (snr f64, width_idx i32, second f64),
    each [n_dm, t1 - t0]; samples are row positions t0 <= n < t1."""
    x = _plane(x)
    n_dm, n_t = x.shape
    t1 = n_t if t1 is None else int(t1)
    t0 = int(t0)
    assert 0 <= t0 <= t1 <= n_t
    w = _widths(widths)
    mu, sg = _stats(mean, n_dm), _stats(sigma, n_dm)
    snr = np.empty((n_dm, t1 - t0), dtype=np.float64)
    idx = np.empty((n_dm, t1 - t0), dtype=np.int32)
    sec = np.empty((n_dm, t1 - t0), dtype=np.float64)
    _load().oracle_spd_direct(x.ctypes.data, n_dm, n_t, mu.ctypes.data, sg.ctypes.data,
                              w.ctypes.data, int(w.size), t0, t1,
                              snr.ctypes.data, idx.ctypes.data, sec.ctypes.data)
    return snr, idx, sec


def spd_grid(x, mean, sigma, widths, seps, t0: int = 0, t1: Optional[int] = None
             ) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Direct summation with a boxcar separation per width (ascending widths, seps[k] >= 1):
    width k is evaluated only where n % seps[k] == 0.  Returns (snr, width_idx, second)."""
    x = _plane(x)
    n_dm, n_t = x.shape
    t1 = n_t if t1 is None else int(t1)
    t0 = int(t0)
    assert 0 <= t0 <= t1 <= n_t
    w = np.ascontiguousarray([int(v) for v in widths], dtype=np.int32)
    sp = np.ascontiguousarray([int(v) for v in seps], dtype=np.int32)
    assert w.size > 0 and w.size == sp.size and w[0] >= 1 and np.all(np.diff(w) > 0) and np.all(sp >= 1)
    mu, sg = _stats(mean, n_dm), _stats(sigma, n_dm)
    snr = np.empty((n_dm, t1 - t0), dtype=np.float64)
    idx = np.empty((n_dm, t1 - t0), dtype=np.int32)
    sec = np.empty((n_dm, t1 - t0), dtype=np.float64)
    _load().oracle_spd_grid(x.ctypes.data, n_dm, n_t, mu.ctypes.data, sg.ctypes.data,
                            w.ctypes.data, sp.ctypes.data, int(w.size), t0, t1,
                            snr.ctypes.data, idx.ctypes.data, sec.ctypes.data)
    return snr, idx, sec


def grid_iterations(seps):
    """The iterations of a grid: runs [kb, ke) of consecutive widths that share a separation."""
    sp = [int(v) for v in seps]
    out, kb = [], 0
    for k in range(1, len(sp) + 1):
        if k == len(sp) or sp[k] != sp[kb]:
            out.append((kb, k))
            kb = k
    return out


def spd_grid_iter(x, mean, sigma, widths, seps, kb: int, ke: int
                  ) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """The output of one iteration (eq. 12): widths[kb:ke] share the separation s = seps[kb];
    point m is sample s * m.  Returns (snr, width_idx, second), each [n_dm, ceil(n_t / s)]; width_idx is the
    index in ``widths``."""
    x = _plane(x)
    n_dm, n_t = x.shape
    w = np.ascontiguousarray([int(v) for v in widths], dtype=np.int32)
    sp = np.ascontiguousarray([int(v) for v in seps], dtype=np.int32)
    kb, ke = int(kb), int(ke)
    assert w.size == sp.size and 0 <= kb < ke <= w.size and np.all(np.diff(w) > 0) and np.all(sp[kb:ke] == sp[kb])
    s = int(sp[kb])
    n_pts = (n_t + s - 1) // s
    mu, sg = _stats(mean, n_dm), _stats(sigma, n_dm)
    snr = np.empty((n_dm, n_pts), dtype=np.float64)
    idx = np.empty((n_dm, n_pts), dtype=np.int32)
    sec = np.empty((n_dm, n_pts), dtype=np.float64)
    _load().oracle_spd_grid_iter(x.ctypes.data, n_dm, n_t, mu.ctypes.data, sg.ctypes.data,
                                 w.ctypes.data, sp.ctypes.data, kb, ke,
                                 snr.ctypes.data, idx.ctypes.data, sec.ctypes.data)
    return snr, idx, sec


def width_sigma(x, widths) -> np.ndarray:
    """Standard deviation per width from power-of-two decimations, interpolated (reading A17):
    float64 [n_dm, n_widths] for the ascending, de-duplicated width set."""
    x = _plane(x)
    n_dm, n_t = x.shape
    w = _widths(widths)
    out = np.empty((n_dm, w.size), dtype=np.float64)
    _load().oracle_width_sigma(x.ctypes.data, n_dm, n_t, w.ctypes.data, int(w.size), out.ctypes.data)
    return out


def spd_direct_sw(x, mean, sigma_w, widths, t0: int = 0, t1: Optional[int] = None
                  ) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Direct summation with a standard deviation per (row, width): sigma_w is [n_dm, n_widths]."""
    x = _plane(x)
    n_dm, n_t = x.shape
    t1 = n_t if t1 is None else int(t1)
    t0 = int(t0)
    w = _widths(widths)
    mu = _stats(mean, n_dm)
    sw = np.ascontiguousarray(sigma_w, dtype=np.float64).reshape(n_dm, w.size)
    snr = np.empty((n_dm, t1 - t0), dtype=np.float64)
    idx = np.empty((n_dm, t1 - t0), dtype=np.int32)
    sec = np.empty((n_dm, t1 - t0), dtype=np.float64)
    _load().oracle_spd_direct_sw(x.ctypes.data, n_dm, n_t, mu.ctypes.data, sw.ctypes.data,
                                 w.ctypes.data, int(w.size), t0, t1,
                                 snr.ctypes.data, idx.ctypes.data, sec.ctypes.data)
    return snr, idx, sec


def spd_prefix(x, mean, sigma, widths) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Oracle B: double-precision running-sum difference on full rows."""
    x = _plane(x)
    n_dm, n_t = x.shape
    w = _widths(widths)
    mu, sg = _stats(mean, n_dm), _stats(sigma, n_dm)
    snr = np.empty((n_dm, n_t), dtype=np.float64)
    idx = np.empty((n_dm, n_t), dtype=np.int32)
    sec = np.empty((n_dm, n_t), dtype=np.float64)
    _load().oracle_spd_prefix(x.ctypes.data, n_dm, n_t, mu.ctypes.data, sg.ctypes.data,
                              w.ctypes.data, int(w.size),
                              snr.ctypes.data, idx.ctypes.data, sec.ctypes.data)
    return snr, idx, sec


def snr_of_width(row, mean: float, sigma: float, L: int, samples) -> np.ndarray:
    """SNR_L[n] by direct summation at the listed samples of one row."""
    row = np.ascontiguousarray(row, dtype=np.float32).reshape(-1)
    s = np.ascontiguousarray(samples, dtype=np.int64)
    out = np.empty(s.shape, dtype=np.float64)
    _load().oracle_snr_of_width(row.ctypes.data, row.size, float(mean), float(sigma), int(L),
                                s.ctypes.data, int(s.size), out.ctypes.data)
    return out


def row_stats(x) -> Tuple[np.ndarray, np.ndarray]:
    """Per-row mean and population standard deviation (reading A6)."""
    x = _plane(x)
    n_dm, n_t = x.shape
    mu = np.empty(n_dm, dtype=np.float64)
    sg = np.empty(n_dm, dtype=np.float64)
    _load().oracle_row_stats(x.ctypes.data, n_dm, n_t, mu.ctypes.data, sg.ctypes.data)
    return mu, sg


def row_stats_clipped(x, clip: float, n_reject_passes: int, rel_tol: float = -1.0, border_eps: float = 0.0,
                      details: bool = False):
    """Per-row mean and population sigma with point-wise outlier rejection at ``clip`` sigmas
    (reading A14), all in double: at most ``n_reject_passes`` rejection passes,
    stopping early once a pass changes neither estimate by more than ``rel_tol`` * sigma
    (``rel_tol`` < 0: never).  Returns (mean, sigma), or with ``details`` also the passes done per
    row and the number of samples within ``border_eps`` * sigma of a rejection limit."""
    x = _plane(x)
    n_dm, n_t = x.shape
    mu = np.empty(n_dm, dtype=np.float64)
    sg = np.empty(n_dm, dtype=np.float64)
    n_pass = np.empty(n_dm, dtype=np.int32)
    n_border = np.empty(n_dm, dtype=np.int64)
    _load().oracle_row_stats_clipped(x.ctypes.data, n_dm, n_t, float(clip), int(n_reject_passes),
                                     float(rel_tol), float(border_eps), mu.ctypes.data, sg.ctypes.data,
                                     n_pass.ctypes.data, n_border.ctypes.data)
    if details:
        return mu, sg, n_pass, n_border
    return mu, sg


def spd_grid_sw(x, mean, sigma_w, widths, seps, t0: int = 0, t1: Optional[int] = None
                ) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """``spd_grid`` with a standard deviation per (row, width): sigma_w is [n_dm, n_widths]."""
    x = _plane(x)
    n_dm, n_t = x.shape
    t1 = n_t if t1 is None else int(t1)
    t0 = int(t0)
    assert 0 <= t0 <= t1 <= n_t
    w = np.ascontiguousarray([int(v) for v in widths], dtype=np.int32)
    sp = np.ascontiguousarray([int(v) for v in seps], dtype=np.int32)
    assert w.size > 0 and w.size == sp.size and w[0] >= 1 and np.all(np.diff(w) > 0) and np.all(sp >= 1)
    mu = _stats(mean, n_dm)
    sw = np.ascontiguousarray(sigma_w, dtype=np.float64).reshape(n_dm, w.size)
    snr = np.empty((n_dm, t1 - t0), dtype=np.float64)
    idx = np.empty((n_dm, t1 - t0), dtype=np.int32)
    sec = np.empty((n_dm, t1 - t0), dtype=np.float64)
    _load().oracle_spd_grid_sw(x.ctypes.data, n_dm, n_t, mu.ctypes.data, sw.ctypes.data,
                               w.ctypes.data, sp.ctypes.data, int(w.size), t0, t1,
                               snr.ctypes.data, idx.ctypes.data, sec.ctypes.data)
    return snr, idx, sec


def find_candidates(snr, width_idx, threshold: float, capacity: Optional[int] = None):
    """Reading A9 candidate rule on a float32 SNR plane.  Returns
    (count, dm i32[], t i32[], snr f32[], width_idx i32[]) in (dm, t) order."""
    snr = _plane(snr)
    n_dm, n_t = snr.shape
    wid = np.ascontiguousarray(width_idx, dtype=np.int32).reshape(n_dm, n_t)
    cap = int(snr.size if capacity is None else capacity)
    c_dm = np.empty(cap, dtype=np.int32)
    c_t = np.empty(cap, dtype=np.int32)
    c_snr = np.empty(cap, dtype=np.float32)
    c_w = np.empty(cap, dtype=np.int32)
    count = int(_load().oracle_find_candidates(snr.ctypes.data, wid.ctypes.data, n_dm, n_t,
                                               ctypes.c_float(threshold), cap,
                                               c_dm.ctypes.data, c_t.ctypes.data,
                                               c_snr.ctypes.data, c_w.ctypes.data))
    k = min(count, cap)
    return count, c_dm[:k], c_t[:k], c_snr[:k], c_w[:k]


def cluster_candidates(snr, widths, c_dm, c_t, c_width, dm_radius: int) -> np.ndarray:
    """Reading A18: 2-D (DM x time) peak rule over 1-D candidates of a float32 SNR plane.
    ``c_width`` are indices into the ascending width set.  Returns the boolean keep mask."""
    snr = _plane(snr)
    n_dm, n_t = snr.shape
    w = _widths(widths)
    cd = np.ascontiguousarray(c_dm, dtype=np.int32)
    ct = np.ascontiguousarray(c_t, dtype=np.int32)
    cw = np.ascontiguousarray(c_width, dtype=np.int32)
    assert cd.size == ct.size == cw.size
    keep = np.zeros(cd.size, dtype=np.uint8)
    _load().oracle_cluster_candidates(snr.ctypes.data, n_dm, n_t, w.ctypes.data, int(w.size),
                                      cd.ctypes.data, ct.ctypes.data, cw.ctypes.data, int(cd.size),
                                      int(dm_radius), keep.ctypes.data)
    return keep.astype(bool)
