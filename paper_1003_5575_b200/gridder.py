"""Thin ctypes binding of include/gridder.h -- argument marshalling only.

Every step of the path (map, sort, tile tables, grid, flush) runs inside libgridder.so's CUDA
kernels.  torch is used for device memory and streams and nothing else.  There is no CPU
fallback: if the shared library is missing or cannot be loaded this module raises.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from pathlib import Path

import torch

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libgridder.so"

OK, ERR_INVALID_ARG, ERR_CAPACITY, ERR_WORKSPACE, ERR_CUDA, ERR_NOT_BINNED, ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5, -6

EXPORTS = ("gridder_check_violations", "gridder_bin_channels", "gridder_grid_channels", "gridder_workspace_size", "gridder_plan", "gridder_workspace_size_tuned", "gridder_plan_tuned", "gridder_map_presum",
           "gridder_bin", "gridder_bin_tables", "gridder_grid", "gridder_destroy",
           "gridder_get_stats", "gridder_map", "gridder_scatter_atomic", "gridder_image_workspace_size", "gridder_image",
           "gridder_run_host", "gridder_grid_static", "gridder_sum_parts", "gridder_set_profiling",
           "gridder_get_stage_ms", "gridder_launch_count", "gridder_strerror",
           "gridder_last_cuda_error", "gridder_version")


class GridderError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {strerror(code)} ({code})")
        self.code = code


class _Config(C.Structure):
    _fields_ = [("grid_size", C.c_int32), ("cell_size", C.c_double), ("n_pol", C.c_int32),
                ("oversample", C.c_int32), ("n_wplanes", C.c_int32), ("support", C.POINTER(C.c_int32)),
                ("w_max", C.c_double), ("kernel_is_complex", C.c_int32), ("kernel", C.c_void_p),
                ("max_vis", C.c_int64), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("max_grids", C.c_int32)]


class _Tuning(C.Structure):
    _fields_ = [("tile_log2", C.c_int32), ("chunk", C.c_int32), ("max_warps", C.c_int32), ("merge", C.c_int32),
                ("presum", C.c_int32), ("table_in_tmem", C.c_int32), ("fold_batches", C.c_int32),
                ("force_general", C.c_int32), ("host_slices", C.c_int32), ("host_slice_min_mb", C.c_int32),
                ("reserved", C.c_int32 * 6)]


TUNING_FIELDS = tuple(f[0] for f in _Tuning._fields_ if f[0] != "reserved")


class _Stats(C.Structure):
    _fields_ = [("n_vis", C.c_int64), ("n_dropped", C.c_int64), ("n_entries", C.c_int64),
                ("vis_taps", C.c_int64), ("n_tiles", C.c_int64), ("n_tiles_occupied", C.c_int64),
                ("max_tile_load", C.c_int64), ("n_work_items", C.c_int64), ("tile_size", C.c_int32),
                ("patch_size", C.c_int32), ("chunk_size", C.c_int32), ("grid_warps_per_sm", C.c_int32),
                ("n_records_gridded", C.c_int64), ("n_presum_records", C.c_int64), ("fma_executed", C.c_int64)]


_lib = None


def select_library(path) -> None:
    """Use another build of the library (the GRIDDER_CHECKED one) -- before the first load_library()."""
    global LIB_PATH
    if _lib is not None:
        raise RuntimeError("the library is loaded already")
    LIB_PATH = Path(path)


def check_violations() -> int:
    """Failed index checks so far (GRIDDER_CHECKED build), -1 for the normal build."""
    return int(load_library().gridder_check_violations())


def load_library() -> C.CDLL:
    """dlopen libgridder.so (built by ``python -m paper_1003_5575_b200.build``).  Fails loudly."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_1003_5575_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(str(LIB_PATH))
        lib.gridder_workspace_size.argtypes = [C.POINTER(_Config), C.POINTER(C.c_size_t)]
        lib.gridder_plan.argtypes = [C.POINTER(_Config), C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)]
        lib.gridder_workspace_size_tuned.argtypes = [C.POINTER(_Config), C.POINTER(_Tuning), C.POINTER(C.c_size_t)]
        lib.gridder_plan_tuned.argtypes = [C.POINTER(_Config), C.POINTER(_Tuning), C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)]
        lib.gridder_map_presum.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32,
                                           C.c_void_p, C.c_void_p]
        lib.gridder_bin.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p]
        lib.gridder_bin_tables.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32,
                                           C.c_void_p, C.c_void_p]
        lib.gridder_grid.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
        lib.gridder_bin_channels.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32, C.c_int32,
                                             C.c_void_p]
        lib.gridder_grid_channels.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
        lib.gridder_destroy.argtypes = [C.c_void_p]
        lib.gridder_get_stats.argtypes = [C.c_void_p, C.POINTER(_Stats)]
        lib.gridder_map.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32,
                                    C.c_void_p, C.c_void_p, C.c_void_p]
        lib.gridder_scatter_atomic.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32,
                                               C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
        lib.gridder_sum_parts.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        lib.gridder_image_workspace_size.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        lib.gridder_image.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        lib.gridder_run_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.gridder_grid_static.argtypes = [C.POINTER(_Config), C.POINTER(_Tuning), C.c_void_p, C.c_int32, C.c_int32,
                                            C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                            C.POINTER(C.c_size_t), C.c_void_p]
        lib.gridder_set_profiling.argtypes = [C.c_void_p, C.c_int32]
        lib.gridder_get_stage_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
        lib.gridder_launch_count.argtypes = [C.c_void_p]
        lib.gridder_launch_count.restype = C.c_int64
        lib.gridder_strerror.argtypes = [C.c_int]
        lib.gridder_strerror.restype = C.c_char_p
        lib.gridder_last_cuda_error.argtypes = [C.c_void_p]
        lib.gridder_version.restype = C.c_char_p
        lib.gridder_check_violations.restype = C.c_longlong
        for name in EXPORTS:
            getattr(lib, name)
        _lib = lib
    return _lib


def strerror(code: int) -> str:
    return load_library().gridder_strerror(int(code)).decode()


def version() -> str:
    return load_library().gridder_version().decode()


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev_ptr(t, dtype, what, device=None, numel=None):
    """Pointer of a device buffer after the checks the C ABI cannot make (it sees no sizes): dtype, layout,
    device and element count."""
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise TypeError(f"{what} must be a contiguous CUDA tensor of {dtype}")
    if device is not None and t.device != device:
        raise ValueError(f"{what} is on {t.device}, the plan on {device}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{what} has {t.numel()} elements, expected {numel}")
    return t.data_ptr()


@dataclass
class Stats:
    n_vis: int
    n_dropped: int
    n_entries: int
    vis_taps: int
    n_tiles: int
    n_tiles_occupied: int
    max_tile_load: int
    n_work_items: int
    tile_size: int
    patch_size: int
    chunk_size: int
    grid_warps_per_sm: int
    n_records_gridded: int = 0
    n_presum_records: int = 0
    fma_executed: int = 0


STATIC_WORKSPACE_BYTES = 64 << 20       # GRIDDER_STATIC_WORKSPACE_BYTES (include/gridder.h)


def grid_static(uvw_m: torch.Tensor, freq_hz: torch.Tensor, vis: torch.Tensor, weight, *, grid_size: int, cell_size: float,
                oversample: int, support, kernel: torch.Tensor, n_wplanes: int = 1, w_max: float = 1.0,
                kernel_is_complex: bool = False, tuning: dict | None = None, out: torch.Tensor | None = None,
                accumulate: bool = False, stream=None) -> torch.Tensor:
    """gridder_grid_static: plan + bin + grid of a small cadence on the library's own static 64 MiB workspace -- no
    device allocation by the library or on its behalf (`out` is the caller's grid; without it one torch.empty is made
    here).  Raises GridderError(ERR_WORKSPACE) when the plan needs more than STATIC_WORKSPACE_BYTES.  Synchronises
    the device."""
    lib = load_library()
    device = vis.device
    if device.type != "cuda":
        raise RuntimeError("the gridder runs on a CUDA device only (no CPU fallback)")
    if uvw_m.dim() == 2:
        uvw_m = uvw_m[None]
    n_time, n_bl, three = uvw_m.shape
    if three != 3:
        raise ValueError("uvw_m must be [n_time][n_baseline][3]")
    n = n_time * n_bl * freq_hz.numel()
    sup = [int(s) for s in (support if hasattr(support, "__len__") else [support])]
    c_sup = (C.c_int32 * len(sup))(*sup)
    if kernel.device != device or kernel.dtype != torch.float32 or not kernel.is_contiguous():
        raise ValueError("kernel must be a contiguous float32 tensor on the visibilities' device")
    cfg = _Config(int(grid_size), float(cell_size), 4, int(oversample), int(n_wplanes), c_sup, float(w_max),
                  int(bool(kernel_is_complex)), kernel.data_ptr(), int(max(n, 1)), None, 0, 1)
    tune = _Tuning()
    for k, v in (tuning or {}).items():
        if k not in TUNING_FIELDS:
            raise KeyError(f"unknown gridder_tuning field {k!r}")
        setattr(tune, k, int(v))
    if out is None:
        if accumulate:
            raise ValueError("accumulate needs an existing grid")
        out = torch.empty((4, int(grid_size), int(grid_size), 2), dtype=torch.float32, device=device)
    need = C.c_size_t(0)
    with torch.cuda.device(device):
        rc = lib.gridder_grid_static(
            C.byref(cfg), C.byref(tune), _dev_ptr(uvw_m, torch.float64, "uvw_m", device, 3 * n_time * n_bl), n_time, n_bl,
            _dev_ptr(freq_hz, torch.float64, "freq_hz", device), freq_hz.numel(),
            _dev_ptr(vis, torch.float32, "vis", device, 8 * n), _dev_ptr(weight, torch.float32, "weight", device, n),
            _dev_ptr(out, torch.float32, "grid", device, 8 * int(grid_size) ** 2), int(accumulate), C.byref(need),
            _stream_ptr(stream))
    if rc != OK:
        err = GridderError(rc, "gridder_grid_static")
        err.workspace_needed = need.value
        raise err
    return out


class Gridder:
    """gridder_plan / gridder_bin / gridder_grid / gridder_destroy with torch tensors as buffers."""

    def __init__(self, *, grid_size: int, cell_size: float, oversample: int, support, kernel: torch.Tensor,
                 max_vis: int, n_wplanes: int = 1, w_max: float = 1.0, kernel_is_complex: bool = False,
                 device=None, tuning: dict | None = None, max_grids: int = 1):
        """`tuning`: optional {field of gridder_tuning: value} (include/gridder.h); absent fields are defaults."""
        lib = load_library()
        self._lib = lib
        self._plan = C.c_void_p()
        self.device = torch.device(device if device is not None else kernel.device)
        if self.device.type != "cuda":
            raise RuntimeError("the gridder runs on a CUDA device only (no CPU fallback)")
        support = [int(s) for s in (support if hasattr(support, "__len__") else [support])]
        self._support = (C.c_int32 * len(support))(*support)
        self._kernel = kernel.to(self.device, torch.float32).contiguous()
        self.grid_size = int(grid_size)
        cfg = _Config(int(grid_size), float(cell_size), 4, int(oversample), int(n_wplanes), self._support,
                      float(w_max), int(bool(kernel_is_complex)), self._kernel.data_ptr(), int(max_vis), None, 0,
                      int(max_grids))
        self.n_grids = 1                 # of the last bin
        tune = _Tuning()
        for k, v in (tuning or {}).items():
            if k not in TUNING_FIELDS:
                raise KeyError(f"unknown gridder_tuning field {k!r}")
            setattr(tune, k, int(v))
        self.n_planes = int(n_wplanes)
        self._binned = None          # (n_time, n_baseline, n_chan) of the last bin
        need = C.c_size_t(0)
        with torch.cuda.device(self.device):
            rc = lib.gridder_workspace_size_tuned(C.byref(cfg), C.byref(tune), C.byref(need))
            if rc != OK:
                raise GridderError(rc, "gridder_workspace_size")
            self.workspace = torch.empty(need.value + 256, dtype=torch.uint8, device=self.device)
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            cfg.workspace = base
            cfg.workspace_bytes = need.value
            rc = lib.gridder_plan_tuned(C.byref(cfg), C.byref(tune), C.byref(self._plan), C.byref(need))
        if rc != OK:
            self._plan = C.c_void_p()
            raise GridderError(rc, "gridder_plan")
        self.workspace_bytes = need.value
        self._keep = []

    # -- the four calls ---------------------------------------------------------------------
    def bin(self, uvw_m: torch.Tensor, freq_hz: torch.Tensor, stream=None, table_index=None, chans_per_grid=None) -> None:
        """uvw_m float64 [n_time][n_baseline][3] (metres), freq_hz float64 [n_chan]; table_index (row f3):
        int32 [n_time][n_baseline] choosing each baseline's table from the plan's bank, or None;
        chans_per_grid (row f4): one output grid per block of that many channels (gridder_bin_channels)."""
        if uvw_m.dim() == 2:
            uvw_m = uvw_m[None]
        n_time, n_bl, three = uvw_m.shape
        if three != 3:
            raise ValueError("uvw_m must be [n_time][n_baseline][3]")
        self._keep = [uvw_m, freq_hz, table_index]
        self._binned = None
        if chans_per_grid is not None:
            if table_index is not None:
                raise ValueError("chans_per_grid and table_index cannot be combined")
            rc = self._lib.gridder_bin_channels(self._plan, _dev_ptr(uvw_m, torch.float64, "uvw_m", self.device), n_time, n_bl,
                                                _dev_ptr(freq_hz, torch.float64, "freq_hz", self.device), freq_hz.numel(),
                                                int(chans_per_grid), _stream_ptr(stream))
            if rc != OK:
                raise GridderError(rc, "gridder_bin_channels")
            self.n_grids = max(1, -(-freq_hz.numel() // int(chans_per_grid)))
            self._binned = (n_time, n_bl, freq_hz.numel())
            return
        self.n_grids = 1
        rc = self._lib.gridder_bin_tables(self._plan, _dev_ptr(uvw_m, torch.float64, "uvw_m", self.device), n_time, n_bl,
                                          _dev_ptr(freq_hz, torch.float64, "freq_hz", self.device), freq_hz.numel(),
                                          _dev_ptr(table_index, torch.int32, "table_index", self.device, n_time * n_bl),
                                          _stream_ptr(stream))
        if rc != OK:
            raise GridderError(rc, "gridder_bin")
        self._binned = (n_time, n_bl, freq_hz.numel())

    def grid(self, vis: torch.Tensor, weight=None, out=None, accumulate: bool = False, stream=None) -> torch.Tensor:
        """vis float32 [...][4][2]; returns the grid float32 [4][N][N][2] (after a bin with chans_per_grid:
        [n_grids][4][N][N][2]); asynchronous."""
        shape = (4, self.grid_size, self.grid_size, 2) if self.n_grids == 1 else (self.n_grids, 4, self.grid_size, self.grid_size, 2)
        if out is None:
            if accumulate:
                raise ValueError("accumulate needs an existing grid")
            out = torch.empty(shape, dtype=torch.float32, device=self.device)
        if self._binned is None:
            raise GridderError(ERR_NOT_BINNED, "gridder_grid")
        n = self._binned[0] * self._binned[1] * self._binned[2]
        fn = self._lib.gridder_grid if self.n_grids == 1 else self._lib.gridder_grid_channels
        rc = fn(self._plan, _dev_ptr(vis, torch.float32, "vis", self.device, 8 * n),
                _dev_ptr(weight, torch.float32, "weight", self.device, n),
                _dev_ptr(out, torch.float32, "grid", self.device, 8 * self.grid_size ** 2 * self.n_grids),
                int(accumulate), _stream_ptr(stream))
        if rc != OK:
            raise GridderError(rc, "gridder_grid")
        return out

    def destroy(self) -> None:
        if self._plan:
            self._lib.gridder_destroy(self._plan)
            self._plan = C.c_void_p()

    # -- helpers ------------------------------------------------------------------------------
    def stats(self) -> Stats:
        st = _Stats()
        rc = self._lib.gridder_get_stats(self._plan, C.byref(st))
        if rc != OK:
            raise GridderError(rc, "gridder_get_stats")
        return Stats(*[int(getattr(st, f[0])) for f in _Stats._fields_])

    def set_profiling(self, enable: bool = True) -> None:
        rc = self._lib.gridder_set_profiling(self._plan, int(enable))
        if rc != OK:
            raise GridderError(rc, "gridder_set_profiling")

    STAGES = ("map", "sort", "tables", "grid", "flush", "presum")

    def stage_ms(self) -> dict:
        """Device milliseconds of the last bin/grid per stage (synchronises on their events)."""
        ms = (C.c_float * 6)()
        rc = self._lib.gridder_get_stage_ms(self._plan, ms)
        if rc != OK:
            raise GridderError(rc, "gridder_get_stage_ms")
        return dict(zip(self.STAGES, [float(x) for x in ms]))

    def launch_count(self) -> int:
        return int(self._lib.gridder_launch_count(self._plan))

    def map(self, uvw_m: torch.Tensor, freq_hz: torch.Tensor, stream=None, table_index=None, presum: bool = False) -> torch.Tensor:
        """int32 [n][6] = x0, y0, qx, qy, plane | conj << 8, dropped.  presum=False: map_vis, the device function
        of the per-visibility map kernel; presum=True: the pre-summed path's one-FMA mapper (gridder_map_presum;
        dropped visibilities report 0, 0, 0, 0, 0, 1)."""
        if uvw_m.dim() == 2:
            uvw_m = uvw_m[None]
        n_time, n_bl, _ = uvw_m.shape
        out = torch.empty((n_time * n_bl * freq_hz.numel(), 6), dtype=torch.int32, device=self.device)
        if presum:
            rc = self._lib.gridder_map_presum(self._plan, _dev_ptr(uvw_m, torch.float64, "uvw_m", self.device), n_time, n_bl,
                                              _dev_ptr(freq_hz, torch.float64, "freq_hz", self.device), freq_hz.numel(),
                                              out.data_ptr(), _stream_ptr(stream))
        else:
            rc = self._lib.gridder_map(self._plan, _dev_ptr(uvw_m, torch.float64, "uvw_m", self.device), n_time, n_bl,
                                       _dev_ptr(freq_hz, torch.float64, "freq_hz", self.device), freq_hz.numel(),
                                       _dev_ptr(table_index, torch.int32, "table_index", self.device, n_time * n_bl),
                                       out.data_ptr(), _stream_ptr(stream))
        if rc != OK:
            raise GridderError(rc, "gridder_map")
        return out

    def scatter_atomic(self, uvw_m, freq_hz, vis, weight=None, out=None, accumulate: bool = False, stream=None):
        """per-visibility FP32 atomic scatter (the OpenGL gridder's arithmetic); not deterministic."""
        if uvw_m.dim() == 2:
            uvw_m = uvw_m[None]
        n_time, n_bl, _ = uvw_m.shape
        if out is None:
            if accumulate:
                raise ValueError("accumulate needs an existing grid")
            out = torch.empty((4, self.grid_size, self.grid_size, 2), dtype=torch.float32, device=self.device)
        n = n_time * n_bl * freq_hz.numel()
        rc = self._lib.gridder_scatter_atomic(
            self._plan, _dev_ptr(uvw_m, torch.float64, "uvw_m", self.device), n_time, n_bl,
            _dev_ptr(freq_hz, torch.float64, "freq_hz", self.device), freq_hz.numel(),
            _dev_ptr(vis, torch.float32, "vis", self.device, 8 * n), _dev_ptr(weight, torch.float32, "weight", self.device, n),
            _dev_ptr(out, torch.float32, "grid", self.device, 8 * self.grid_size ** 2), int(accumulate), _stream_ptr(stream))
        if rc != OK:
            raise GridderError(rc, "gridder_scatter_atomic")
        return out

    def image(self, grid: torch.Tensor, corr=None, out=None, stream=None) -> torch.Tensor:
        """centred inverse FFT of the 4 planes with the grid correction fused in (cuFFT inside)."""
        need = C.c_size_t(0)
        rc = self._lib.gridder_image_workspace_size(self._plan, C.byref(need))
        if rc != OK:
            raise GridderError(rc, "gridder_image_workspace_size")
        if getattr(self, "_fft_work", None) is None or self._fft_work.numel() < need.value:
            self._fft_work = torch.empty(max(need.value, 16), dtype=torch.uint8, device=self.device)
        if out is None:
            out = torch.empty_like(grid)
        cells = 8 * self.grid_size ** 2
        rc = self._lib.gridder_image(self._plan, _dev_ptr(grid, torch.float32, "grid", self.device, cells),
                                     _dev_ptr(out, torch.float32, "image", self.device, cells),
                                     _dev_ptr(corr, torch.float32, "corr", self.device, self.grid_size),
                                     self._fft_work.data_ptr(), self._fft_work.numel(), _stream_ptr(stream))
        if rc != OK:
            raise GridderError(rc, "gridder_image")
        return out

    def run_host(self, uvw_m, freq_hz, vis, weight, grid_out, staging: dict, stream=None) -> None:
        """End to end with HOST tensors (pinned for speed): H2D, bin, grid, D2H, synchronise."""
        def hp(t, dtype, what, numel):
            if t is None:
                return None
            if t.is_cuda or not t.is_contiguous() or t.dtype != dtype:
                raise TypeError(f"{what} must be a contiguous host tensor of {dtype}")
            if t.numel() != numel:
                raise ValueError(f"{what} has {t.numel()} elements, expected {numel}")
            return t.data_ptr()
        if uvw_m.dim() == 2:
            uvw_m = uvw_m[None]
        n_time, n_bl, _ = uvw_m.shape
        n_chan = freq_hz.numel()
        n = n_time * n_bl * n_chan
        cells = 8 * self.grid_size ** 2
        need = {"uvw": (torch.float64, 3 * n_time * n_bl), "freq": (torch.float64, n_chan), "vis": (torch.float32, 8 * n),
                "grid": (torch.float32, cells)}
        if weight is not None:
            need["weight"] = (torch.float32, n)
        for name, (dt, cnt) in need.items():     # staging buffers may be larger than one call needs
            t = staging.get(name)
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.device == self.device and t.is_contiguous()
                    and t.dtype == dt and t.numel() >= cnt):
                raise ValueError(f"staging[{name!r}] must be a contiguous {dt} tensor on {self.device} with >= {cnt} elements")
        self._binned = None
        rc = self._lib.gridder_run_host(
            self._plan, hp(uvw_m, torch.float64, "uvw_m", 3 * n_time * n_bl), n_time, n_bl,
            hp(freq_hz, torch.float64, "freq_hz", n_chan), n_chan, hp(vis, torch.float32, "vis", 8 * n),
            hp(weight, torch.float32, "weight", n), hp(grid_out, torch.float32, "grid_out", cells),
            staging["uvw"].data_ptr(), staging["freq"].data_ptr(),
            staging["vis"].data_ptr(), staging["weight"].data_ptr() if weight is not None else None,
            staging["grid"].data_ptr(), _stream_ptr(stream))
        if rc != OK:
            raise GridderError(rc, "gridder_run_host")

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
