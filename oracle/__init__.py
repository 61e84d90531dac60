"""ORACLE -- TEST INFRASTRUCTURE ONLY (see the header of ``gridder_oracle.c``).

ctypes front end of the plain double-precision CPU direct-scatter gridder of PAPER.md section 5
(Eq. 1, :174-183).  It imports nothing from ``paper_1003_5575_b200`` and the CUDA library imports
nothing from here.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may use it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gridder_oracle.c"
_LIB = _HERE / "libgridder_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """gcc -O2 -ffp-contract=off -fopenmp -> oracle/libgridder_oracle.so (rebuilt when stale)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-o", str(tmp), str(_SRC), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("grid_size", C.c_int32), ("cell_size", C.c_double), ("oversample", C.c_int32),
                ("n_wplanes", C.c_int32), ("support", C.POINTER(C.c_int32)), ("w_max", C.c_double),
                ("kernel_is_complex", C.c_int32), ("kernel", C.POINTER(C.c_float)),
                ("table_index", C.POINTER(C.c_int32))]


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.oracle_map.restype = C.c_int
        _lib.oracle_grid_windows.restype = C.c_int
        _lib.oracle_max_threads.restype = C.c_int
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def _ptr(a, ctype):
    return a.ctypes.data_as(C.POINTER(ctype))


class _Args:
    """Keeps the numpy buffers alive next to the C struct that points at them."""

    def __init__(self, grid_size, cell_size, oversample, support, kernel, w_max=1.0,
                 kernel_is_complex=False, table_index=None):
        self.support = np.ascontiguousarray(support, dtype=np.int32).ravel()
        self.kernel = np.ascontiguousarray(kernel, dtype=np.float32).ravel()
        need = int(sum((int(s) * oversample) ** 2 for s in self.support)) * (2 if kernel_is_complex else 1)
        if self.kernel.size != need:
            raise ValueError(f"kernel table has {self.kernel.size} floats, expected {need}")
        if grid_size % 2 or any((int(s) * oversample) % 2 for s in self.support):
            raise ValueError("grid_size and every S*O must be even")
        self.table_index = None if table_index is None else np.ascontiguousarray(table_index, dtype=np.int32).ravel()
        self.p = _Params(int(grid_size), float(cell_size), int(oversample), int(self.support.size),
                         _ptr(self.support, C.c_int32), float(w_max), int(bool(kernel_is_complex)),
                         _ptr(self.kernel, C.c_float),
                         None if self.table_index is None else _ptr(self.table_index, C.c_int32))


def _inputs(uvw_m, freq_hz, vis=None, weight=None):
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float64)
    if uvw.ndim == 2:
        uvw = uvw[None]
    n_time, n_bl, _ = uvw.shape
    freq = np.ascontiguousarray(freq_hz, dtype=np.float64).ravel()
    n = n_time * n_bl * freq.size
    v = w = None
    if vis is not None:
        v = np.ascontiguousarray(vis, dtype=np.float32).ravel()
        if v.size != n * 8:
            raise ValueError(f"vis has {v.size} floats, expected {n * 8}")
    if weight is not None:
        w = np.ascontiguousarray(weight, dtype=np.float32).ravel()
        if w.size != n:
            raise ValueError(f"weight has {w.size} floats, expected {n}")
    return uvw, freq, v, w, n_time, n_bl


def map_visibilities(uvw_m, freq_hz, *, grid_size, cell_size, oversample, support, kernel,
                     w_max=1.0, kernel_is_complex=False, table_index=None) -> np.ndarray:
    """Steps 1-4 of the definition per visibility: int32 [n][6] = x0, y0, qx, qy, plane|conj<<8, dropped."""
    a = _Args(grid_size, cell_size, oversample, support, kernel, w_max, kernel_is_complex, table_index)
    uvw, freq, _, _, n_time, n_bl = _inputs(uvw_m, freq_hz)
    out = np.empty((n_time * n_bl * freq.size, 6), dtype=np.int32)
    rc = _load().oracle_map(C.byref(a.p), _ptr(uvw, C.c_double), n_time, n_bl, _ptr(freq, C.c_double),
                            int(freq.size), _ptr(out, C.c_int32))
    if rc:
        raise RuntimeError("oracle_map failed")
    return out


def grid_windows(uvw_m, freq_hz, vis, weight, windows, *, grid_size, cell_size, oversample, support,
                 kernel, w_max=1.0, kernel_is_complex=False, want_abs=True, n_threads=0, out=None,
                 table_index=None):
    """Direct scatter restricted to each window (y_lo, y_hi, x_lo, x_hi).

    Returns (list of complex128 [4][h][w], list of float64 [4][h][w] or None, stats dict).  With
    ``out=(G_list, A_list)`` from an earlier call the sums are added to (used to feed the
    integrations of config 4 one at a time).
    """
    a = _Args(grid_size, cell_size, oversample, support, kernel, w_max, kernel_is_complex, table_index)
    uvw, freq, v, w, n_time, n_bl = _inputs(uvw_m, freq_hz, vis, weight)
    if a.table_index is not None and a.table_index.size != n_time * n_bl:
        raise ValueError("table_index must have n_time * n_baseline entries")
    wins = [tuple(int(x) for x in win) for win in windows]
    sizes = [4 * (y1 - y0) * (x1 - x0) for (y0, y1, x0, x1) in wins]
    offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    if out is None:
        g = np.zeros(int(offs[-1]), dtype=np.complex128)
        ab = np.zeros(int(offs[-1]), dtype=np.float64) if want_abs else None
    else:
        g, ab = out["_g"], out["_a"]
    table = np.array([[y0, y1, x0, x1, offs[k], (y1 - y0) * (x1 - x0), (x1 - x0)]
                      for k, (y0, y1, x0, x1) in enumerate(wins)], dtype=np.int64).reshape(-1, 7)
    stats = np.zeros(2, dtype=np.int64)
    rc = _load().oracle_grid_windows(
        C.byref(a.p), _ptr(uvw, C.c_double), n_time, n_bl, _ptr(freq, C.c_double), int(freq.size),
        _ptr(v, C.c_float), _ptr(w, C.c_float) if w is not None else None, len(wins),
        _ptr(table, C.c_int64), _ptr(g, C.c_double), _ptr(ab, C.c_double) if ab is not None else None,
        _ptr(stats, C.c_int64), int(n_threads))
    if rc:
        raise RuntimeError("oracle_grid_windows: invalid argument")
    res = {"_g": g, "_a": ab, "n_dropped": int(stats[0]), "vis_taps": int(stats[1]), "windows": wins}
    if out is not None:
        res["n_dropped"] += out["n_dropped"]
        res["vis_taps"] += out["vis_taps"]
    res["G"] = [g[offs[k]:offs[k + 1]].reshape(4, y1 - y0, x1 - x0) for k, (y0, y1, x0, x1) in enumerate(wins)]
    res["A"] = None if ab is None else [
        ab[offs[k]:offs[k + 1]].reshape(4, y1 - y0, x1 - x0) for k, (y0, y1, x0, x1) in enumerate(wins)]
    return res


def grid_full(uvw_m, freq_hz, vis, weight=None, *, grid_size, cell_size, oversample, support, kernel,
              w_max=1.0, kernel_is_complex=False, want_abs=True, n_threads=0, table_index=None):
    """The whole grid: complex128 [4][N][N], float64 [4][N][N] (or None), stats.

    Threads own disjoint row bands of the one shared grid (one writer per cell, so the result is
    the same for any thread count); each band is the same direct scatter over all visibilities.
    """
    a = _Args(grid_size, cell_size, oversample, support, kernel, w_max, kernel_is_complex, table_index)
    uvw, freq, v, w, n_time, n_bl = _inputs(uvw_m, freq_hz, vis, weight)
    if a.table_index is not None and a.table_index.size != n_time * n_bl:
        raise ValueError("table_index must have n_time * n_baseline entries")
    n = int(grid_size)
    nt = n_threads if n_threads > 0 else max_threads()
    nb = max(1, min(n, nt))
    edges = [(k * n) // nb for k in range(nb + 1)]
    table = np.array([[edges[k], edges[k + 1], 0, n, edges[k] * n, n * n, n] for k in range(nb)],
                     dtype=np.int64)
    g = np.zeros((4, n, n), dtype=np.complex128)
    ab = np.zeros((4, n, n), dtype=np.float64) if want_abs else None
    stats = np.zeros(2, dtype=np.int64)
    rc = _load().oracle_grid_windows(
        C.byref(a.p), _ptr(uvw, C.c_double), n_time, n_bl, _ptr(freq, C.c_double), int(freq.size),
        _ptr(v, C.c_float), _ptr(w, C.c_float) if w is not None else None, nb,
        _ptr(table, C.c_int64), _ptr(g, C.c_double), _ptr(ab, C.c_double) if ab is not None else None,
        _ptr(stats, C.c_int64), int(nt))
    if rc:
        raise RuntimeError("oracle_grid_windows: invalid argument")
    return g, ab, {"n_dropped": int(stats[0]), "vis_taps": int(stats[1]), "threads": nb}


# ---- row f2: the imaging step after the gridder (test infrastructure, like everything here) --------------
def grid_correction(table_1d, support: int, oversample: int, grid_size: int) -> np.ndarray:
    """1 / c_hat(l_k) for image pixels k = 0..N-1 (l_k = (k - N/2) / N cycles per cell), where
    c_hat(l) = (1/O) sum_j T1[j] cos(2 pi r_j l), r_j = (j - S O / 2) / O: the Fourier transform of the
    (separable, even) tabulated GCF itself (R4; PAPER.md :75 "grid correction")."""
    t1 = np.asarray(table_1d, dtype=np.float64)
    r = (np.arange(support * oversample) - (support * oversample) / 2.0) / oversample
    lk = (np.arange(grid_size) - grid_size // 2) / grid_size
    chat = (t1[None, :] * np.cos(2.0 * np.pi * r[None, :] * lk[:, None])).sum(1) / oversample
    return 1.0 / chat


def image(grid_c: np.ndarray, corr=None) -> np.ndarray:
    """Dirty image of a gridded plane set, complex128 [..., N, N]: the unnormalised inverse DFT with both
    planes centred on cell N/2, times corr[y] corr[x] (PAPER.md :75, :211):
        image[y][x] = corr[y] corr[x] sum_{v,u} G[v][u] exp(+2 pi i ((u-N/2)(x-N/2) + (v-N/2)(y-N/2)) / N).
    Written with the library FFT as the step the definition names; pinned in tests/test_oracle_pins.py against
    the O(N^4) sum written out and (P4) against the direct DFT of a point source."""
    g = np.asarray(grid_c, dtype=np.complex128)
    n = g.shape[-1]
    img = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(g, axes=(-2, -1)), axes=(-2, -1)), axes=(-2, -1)) * (n * n)
    if corr is not None:
        c = np.asarray(corr, dtype=np.float64)
        img = img * (c[:, None] * c[None, :])
    return img
