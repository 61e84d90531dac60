"""Full-size parity (BASELINE.json configs 2, 3 and 4 at their real sizes, in the launch configuration
bench.py times: default tile, chunk and warps).  The oracle cannot grid 4096^2 x 10^8..10^9 in test
time, so it computes sampled windows of the grid one by one (oracle.grid_windows: the same direct
scatter restricted to a window) -- hot centre, mid-radius, sparse outskirts, a strip crossing many
tiles -- and every cell of every window must satisfy |delta| <= 1e-5 * sum|w V C| + 1e-6.  Counts
(visibilities, dropped, vis*taps) are compared exactly and the rerun must be bit-identical."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import as_complex, oracle_kwargs, RTOL_ABS, ATOL

pytestmark = pytest.mark.gpu

N = 4096
WINDOWS = [                       # (y_lo, y_hi, x_lo, x_hi)
    (2032, 2064, 2032, 2064),     # the hottest tiles (18 antennas within 1.5 m of the centre)
    (2060, 2084, 1990, 2014),     # core, off-centre
    (2000, 2008, 1800, 2296),     # a strip across 124 tiles through the core
    (2400, 2424, 1700, 1724),     # mid radius
    (1500, 1524, 2600, 2624),
    (3000, 3024, 1200, 1224),     # outskirts
    (700, 724, 3100, 3124),
    (40, 64, 2040, 2064),         # near the grid edge (the longest baselines)
]


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5575_b200 import gridder
    gridder.load_library()
    if torch.cuda.get_device_properties(0).total_memory < 100 * 2 ** 30:
        pytest.skip("needs a 180 GB class GPU")
    return torch.device("cuda:0")


def _run_full(dev, cfg):
    """Grid config `cfg` at full size on the GPU; the oracle's windows are fed one integration at a time."""
    from paper_1003_5575_b200 import gridder
    wl = synth.make_workload(cfg)
    nt, nb, nf = wl.n_time, wl.n_baseline, wl.n_chan
    vis = torch.empty((nt, nb, nf, 4, 2), dtype=torch.float32, device=dev)
    weight = torch.empty((nt, nb, nf), dtype=torch.float32, device=dev) if wl.random_weights else None
    res = None
    kw = oracle_kwargs(wl)
    for t in range(nt):
        vis[t] = wl.vis_block(t, dev)
        if weight is not None:
            weight[t] = wl.weight_block(t, dev)
        h_vis = vis[t].cpu().numpy()
        h_w = None if weight is None else weight[t].cpu().numpy()
        res = oracle.grid_windows(wl.uvw[t:t + 1], wl.freq, h_vis, h_w, WINDOWS, out=res, **kw)
        del h_vis, h_w
    g = gridder.Gridder(grid_size=wl.grid_size, cell_size=wl.cell_size, oversample=wl.oversample, support=wl.support,
                        kernel=torch.from_numpy(wl.kernel).to(dev), max_vis=wl.n_vis, n_wplanes=wl.n_wplanes,
                        w_max=wl.w_max, kernel_is_complex=wl.kernel_is_complex)
    g.bin(torch.from_numpy(wl.uvw).to(dev), torch.from_numpy(wl.freq).to(dev))
    grid = g.grid(vis, weight)
    st = g.stats()
    first = [grid[:, y0:y1, x0:x1].cpu().numpy() for (y0, y1, x0, x1) in WINDOWS]
    checksum = grid.view(torch.int32).sum(dtype=torch.int64).item()
    grid2 = g.grid(vis, weight)
    same = bool(torch.equal(grid, grid2)) and grid2.view(torch.int32).sum(dtype=torch.int64).item() == checksum
    g.destroy()
    del vis, weight, grid, grid2
    torch.cuda.empty_cache()
    return wl, st, first, res, same


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_full_size_sampled_windows(dev, cfg):
    wl, st, got, res, same = _run_full(dev, cfg)
    assert same, "rerun at full size is not bit-identical"
    assert st.n_vis == wl.n_vis and st.n_dropped == res["n_dropped"] == 0
    assert st.vis_taps == res["vis_taps"]
    if wl.n_wplanes == 1:
        assert st.vis_taps == wl.n_vis * wl.support[0] ** 2
    worst, busiest = 0.0, 0.0
    for k, win in enumerate(WINDOWS):
        ref, ab = res["G"][k], res["A"][k]
        err = np.abs(as_complex(got[k]) - ref)
        tol = RTOL_ABS * ab + ATOL
        bad = err > tol
        assert not bad.any(), (f"config {cfg} window {win}: {int(bad.sum())} cells out of tolerance, "
                               f"worst err/tol {float((err / tol).max()):.3f}")
        worst = max(worst, float((err / tol).max()))
        busiest = max(busiest, float(ab.max()))
    assert busiest > 1e3, "the sampled windows must include heavily loaded cells"
    print(f"config {cfg}: worst err/tol {worst:.3f} over {len(WINDOWS)} windows, busiest cell sum|wVC| {busiest:.3g}, "
          f"{st.n_work_items} work items, max tile load {st.max_tile_load}")
