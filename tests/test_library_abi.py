"""CPU-side checks of the boundary: the shared library builds, loads and exports every symbol
include/gridder.h declares; argument checks that need no device return the documented codes."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def lib():
    from paper_1003_5575_b200 import build, gridder
    build.build()
    return gridder.load_library()


def test_every_declared_symbol_is_exported(lib):
    header = (ROOT / "include" / "gridder.h").read_text()
    declared = set(re.findall(r"GRIDDER_API\s+[\w\s\*]+?\b(gridder_\w+)\s*\(", header))
    assert {"gridder_plan", "gridder_bin", "gridder_grid", "gridder_destroy"} <= declared
    from paper_1003_5575_b200 import gridder
    assert declared == set(gridder.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_version_and_strerror(lib):
    from paper_1003_5575_b200 import gridder
    assert re.fullmatch(r"\d+\.\d+\.\d+", gridder.version())
    assert gridder.strerror(0) == "ok"
    for code in range(-6, 0):
        assert "unknown" not in gridder.strerror(code)
    assert "unknown" in gridder.strerror(-99)


def test_null_and_invalid_arguments_need_no_device(lib):
    from paper_1003_5575_b200 import gridder
    need = C.c_size_t(0)
    assert lib.gridder_workspace_size(None, C.byref(need)) == gridder.ERR_INVALID_ARG
    sup = (C.c_int32 * 1)(16)
    def cfg(**kw):
        base = dict(grid_size=256, cell_size=1.0, n_pol=4, oversample=4, n_wplanes=1, support=sup, w_max=1.0,
                    kernel_is_complex=0, kernel=None, max_vis=1000, workspace=None, workspace_bytes=0, max_grids=0)
        base.update(kw)
        return gridder._Config(*[base[f[0]] for f in gridder._Config._fields_])
    for bad in (dict(grid_size=255), dict(grid_size=0), dict(cell_size=0.0), dict(n_pol=2), dict(oversample=0),
                dict(n_wplanes=0), dict(max_vis=-1), dict(support=(C.c_int32 * 1)(0)),
                dict(support=(C.c_int32 * 1)(33)), dict(support=(C.c_int32 * 1)(7), oversample=1)):
        assert lib.gridder_workspace_size(C.byref(cfg(**bad)), C.byref(need)) == gridder.ERR_INVALID_ARG, bad
    # complex tables, w-planes and supports up to 32 are sized without a device
    assert lib.gridder_workspace_size(C.byref(cfg(kernel_is_complex=1)), C.byref(need)) == gridder.OK and need.value > 0
    sup3 = (C.c_int32 * 3)(8, 16, 32)
    assert lib.gridder_workspace_size(C.byref(cfg(n_wplanes=3, support=sup3, w_max=10.0)), C.byref(need)) == gridder.OK
    assert lib.gridder_workspace_size(C.byref(cfg(n_wplanes=3, support=sup3, w_max=0.0)), C.byref(need)) == gridder.ERR_INVALID_ARG
    # the largest grid is sized too (its key has no room for the sub-cell bits: general path)
    assert lib.gridder_workspace_size(C.byref(cfg(grid_size=32768)), C.byref(need)) == gridder.OK
    # a table bank of 2 GB and more is beyond the 32-bit table offsets
    sup64 = (C.c_int32 * 64)(*([32] * 64))
    assert lib.gridder_workspace_size(C.byref(cfg(n_wplanes=64, support=sup64, oversample=64, kernel_is_complex=1,
                                                  w_max=1.0)), C.byref(need)) == gridder.ERR_UNSUPPORTED
    # tuning: a zeroed struct is the default plan, a field outside its range is refused, several grids are sized
    tune = gridder._Tuning()
    assert lib.gridder_workspace_size_tuned(C.byref(cfg()), C.byref(tune), C.byref(need)) == gridder.OK
    one = need.value
    assert lib.gridder_workspace_size(C.byref(cfg()), C.byref(need)) == gridder.OK and need.value == one
    for field, bad in (("tile_log2", 5), ("chunk", 7), ("merge", 3), ("presum", -1), ("fold_batches", 3), ("table_in_tmem", 9)):
        t = gridder._Tuning()
        setattr(t, field, bad)
        assert lib.gridder_workspace_size_tuned(C.byref(cfg()), C.byref(t), C.byref(need)) == gridder.ERR_INVALID_ARG, field
    assert lib.gridder_workspace_size(C.byref(cfg(max_grids=12)), C.byref(need)) == gridder.OK and need.value > one
    assert lib.gridder_workspace_size(C.byref(cfg(max_grids=-1)), C.byref(need)) == gridder.ERR_INVALID_ARG
    assert lib.gridder_bin_channels(None, None, 1, 1, None, 1, 1, None) == gridder.ERR_INVALID_ARG
    plan = C.c_void_p()
    assert lib.gridder_plan(C.byref(cfg(grid_size=255)), C.byref(plan), None) == gridder.ERR_INVALID_ARG
    assert lib.gridder_plan(C.byref(cfg()), None, None) == gridder.ERR_INVALID_ARG
    assert lib.gridder_bin(None, None, 1, 1, None, 1, None) == gridder.ERR_INVALID_ARG
    assert lib.gridder_grid(None, None, None, None, 0, None) == gridder.ERR_INVALID_ARG
    assert lib.gridder_destroy(None) == gridder.ERR_INVALID_ARG
    assert lib.gridder_get_stats(None, None) == gridder.ERR_INVALID_ARG
    # row f4's summation kernel: argument checks come before any CUDA call
    buf = C.c_void_p(256)
    assert lib.gridder_sum_parts(None, 2, 8, 8, buf, None) == gridder.ERR_INVALID_ARG
    assert lib.gridder_sum_parts(buf, 0, 8, 8, buf, None) == gridder.ERR_INVALID_ARG          # no parts
    assert lib.gridder_sum_parts(buf, 2, 6, 8, buf, None) == gridder.ERR_INVALID_ARG          # len not a multiple of 4
    assert lib.gridder_sum_parts(buf, 2, 8, 4, buf, None) == gridder.ERR_INVALID_ARG          # stride < len
    assert lib.gridder_sum_parts(C.c_void_p(260), 2, 8, 8, buf, None) == gridder.ERR_INVALID_ARG   # misaligned
    assert lib.gridder_sum_parts(buf, 2, 0, 0, buf, None) == gridder.OK                       # nothing to do


def test_binding_refuses_cpu_tensors():
    import torch
    from paper_1003_5575_b200 import gridder
    with pytest.raises(RuntimeError):
        gridder.Gridder(grid_size=64, cell_size=1.0, oversample=4, support=[8],
                        kernel=torch.zeros(32 * 32), max_vis=10)
