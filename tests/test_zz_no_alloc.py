"""gridder_grid_static (csrc/static_ws.cu): the path on the library's own static 64 MiB workspace, for callers that
may not allocate device memory.  Two different problems back to back on the shared, dirty array, each compared with
the existing path (gridder_plan + gridder_bin + gridder_grid on a caller-owned workspace) within the tests'
tolerance, and with the oracle; a plan beyond the array is refused.  (Named to be collected last.)"""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import ATOL, RTOL_ABS, as_complex, assert_parity

pytestmark = pytest.mark.gpu
C_M_S = 299_792_458.0


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5575_b200 import gridder
    gridder.load_library()
    return torch.device("cuda:0")


def _case(seed, N, S, O, nt, nb, nf):
    rng = np.random.default_rng(seed)
    uvw = np.zeros((nt, nb, 3))
    uvw[:, :, :2] = rng.uniform(-N / 2 - 1, N / 2 + 1, (nt, nb, 2))
    uvw[:, :8, :2] = 3.25                                            # a hot point: one tile takes many entries
    freq = C_M_S * (1.0 + 2e-3 * np.arange(nf))
    vis = rng.standard_normal((nt, nb, nf, 4, 2)).astype(np.float32)
    w = rng.uniform(0.5, 1.5, (nt, nb, nf)).astype(np.float32)
    return uvw, freq, vis, w, synth.spheroidal_table(S, O).astype(np.float32)


def _existing_path(dev, uvw, freq, vis, w, table, *, N, S, O, accumulate_onto=None):
    from paper_1003_5575_b200 import gridder
    g = gridder.Gridder(grid_size=N, cell_size=1.0, oversample=O, support=[S],
                        kernel=torch.from_numpy(table.ravel()).to(dev), max_vis=vis.size // 8, tuning={"presum": 2})
    g.bin(torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev))
    if accumulate_onto is None:
        out = g.grid(torch.from_numpy(vis).to(dev), torch.from_numpy(w).to(dev))
    else:
        out = torch.from_numpy(accumulate_onto.copy()).to(dev)
        g.grid(torch.from_numpy(vis).to(dev), torch.from_numpy(w).to(dev), out=out, accumulate=True)
    res = out.cpu().numpy()
    g.destroy()
    return res


def _static_path(dev, uvw, freq, vis, w, table, *, N, S, O, accumulate_onto=None):
    from paper_1003_5575_b200 import gridder
    d = dict(grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=torch.from_numpy(table.ravel()).to(dev))
    args = (torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev), torch.from_numpy(vis).to(dev),
            torch.from_numpy(w).to(dev))
    if accumulate_onto is None:
        out = torch.full((4, N, N, 2), float("nan"), dtype=torch.float32, device=dev)     # every cell must be written
        gridder.grid_static(*args, out=out, **d)
    else:
        out = torch.from_numpy(accumulate_onto.copy()).to(dev)
        gridder.grid_static(*args, out=out, accumulate=True, **d)
    return out.cpu().numpy()


def test_static_workspace_two_calls_in_a_row_match_the_existing_path(dev):
    shapes = [dict(seed=31, N=128, S=16, O=4, nt=3, nb=180, nf=12),      # 16-cell patches, 6 480 visibilities
              dict(seed=32, N=256, S=7, O=8, nt=2, nb=150, nf=9)]        # 8-cell patches: another layout of the array
    cases = [(_case(**sh), dict(N=sh["N"], S=sh["S"], O=sh["O"])) for sh in shapes]
    # the two static calls run back to back: the second finds the array as the first left it
    got = [_static_path(dev, *c, **kw) for c, kw in cases]
    for (c, kw), g in zip(cases, got):
        uvw, freq, vis, w, table = c
        ref, ab, _ = oracle.grid_full(uvw, freq, vis, w, grid_size=kw["N"], cell_size=1.0, oversample=kw["O"],
                                      support=[kw["S"]], kernel=table.ravel())
        assert np.isfinite(g).all()
        assert_parity(g, ref, ab, f"static workspace, N = {kw['N']}")
        old = _existing_path(dev, *c, **kw)
        err = np.abs(as_complex(g) - as_complex(old))
        assert (err <= RTOL_ABS * ab + ATOL).all(), float((err / (RTOL_ABS * ab + ATOL)).max())
        assert np.array_equal(g, old)                                    # the same code on another workspace: same bits
    # and once more the first problem, now accumulating onto a grid: the array holds the second problem's leftovers
    (c, kw) = cases[0]
    base = np.random.default_rng(33).standard_normal((4, kw["N"], kw["N"], 2)).astype(np.float32)
    a = _static_path(dev, *c, accumulate_onto=base, **kw)
    b = _existing_path(dev, *c, accumulate_onto=base, **kw)
    assert np.array_equal(a, b)


def test_static_workspace_refuses_what_does_not_fit(dev):
    from paper_1003_5575_b200 import gridder
    N, S, O = 1024, 16, 4
    table = torch.from_numpy(synth.spheroidal_table(S, O).astype(np.float32).ravel()).to(dev)
    n = 300_000
    uvw = torch.zeros((1, n, 3), dtype=torch.float64, device=dev)
    freq = torch.full((1,), C_M_S, dtype=torch.float64, device=dev)
    vis = torch.zeros((n, 4, 2), dtype=torch.float32, device=dev)
    out = torch.full((4, N, N, 2), 7.0, dtype=torch.float32, device=dev)
    with pytest.raises(gridder.GridderError) as e:
        gridder.grid_static(uvw, freq, vis, None, grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=table, out=out)
    assert e.value.code == gridder.ERR_WORKSPACE and "workspace too small" in str(e.value)
    assert e.value.workspace_needed > gridder.STATIC_WORKSPACE_BYTES
    assert bool((out == 7.0).all())                                      # nothing was enqueued
