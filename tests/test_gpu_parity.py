"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Integer work (the mapping, counts) must be bit-exact; grid cells must satisfy
BASELINE.json's |delta| <= 1e-5 * sum|w V C| + 1e-6; reruns must be bit-identical."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import as_complex, assert_parity, oracle_kwargs

pytestmark = pytest.mark.gpu
C = 299_792_458.0


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5575_b200 import gridder
    gridder.load_library()           # must exist: there is no fallback
    return torch.device("cuda:0")


def _gridder(dev, *, N, du, O, S, table, max_vis, tuning=None):
    """A plan; `tuning` = fields of gridder_tuning (include/gridder.h) that steer it onto the path under test."""
    from paper_1003_5575_b200 import gridder
    return gridder.Gridder(grid_size=N, cell_size=du, oversample=O, support=[S],
                           kernel=torch.from_numpy(np.ascontiguousarray(table, np.float32).ravel()).to(dev),
                           max_vis=max_vis, tuning=tuning)


def _run(dev, uvw, freq, vis, weight, *, N, du, O, S, table, tuning=None, accumulate_onto=None):
    uvw = np.ascontiguousarray(uvw, np.float64)
    uvw = uvw[None] if uvw.ndim == 2 else uvw
    n = uvw.shape[0] * uvw.shape[1] * len(freq)
    g = _gridder(dev, N=N, du=du, O=O, S=S, table=table, max_vis=max(n, 1), tuning=tuning)
    g.bin(torch.from_numpy(uvw).to(dev), torch.tensor(np.asarray(freq, np.float64), device=dev))
    d_vis = torch.from_numpy(np.ascontiguousarray(vis, np.float32)).to(dev)
    d_w = None if weight is None else torch.from_numpy(np.ascontiguousarray(weight, np.float32)).to(dev)
    if accumulate_onto is not None:
        out = torch.from_numpy(accumulate_onto.copy()).to(dev)
        g.grid(d_vis, d_w, out=out, accumulate=True)
    else:
        out = g.grid(d_vis, d_w)
    res = out.cpu().numpy()
    st = g.stats()
    g.destroy()
    return res, st


def _oracle(uvw, freq, vis, weight, *, N, du, O, S, table):
    uvw = np.ascontiguousarray(uvw, np.float64)
    uvw = uvw[None] if uvw.ndim == 2 else uvw
    return oracle.grid_full(uvw, freq, vis, weight, grid_size=N, cell_size=du, oversample=O, support=[S],
                            kernel=np.ascontiguousarray(table, np.float32).ravel())


def _random_case(rng, n, N, S, spread=None, lattice_ties=True):
    half = N / 2
    spread = half + 1 if spread is None else spread
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = rng.uniform(-spread, spread, (n, 2))
    if lattice_ties and n >= 100:
        uvw[0, :40, :2] = (np.floor(uvw[0, :40, :2] * 8) + 0.5) / 8          # rounding ties
        uvw[0, 40:60, :2] = np.round(uvw[0, 40:60, :2])                      # cell centres
        uvw[0, 60, :2] = (-half + S / 2, -half + S / 2)                      # first legal origin
        uvw[0, 61, :2] = (half - S / 2 - 0.125, half - S / 2 - 0.125)        # last legal origin
        uvw[0, 62, :2] = (-half + S / 2 - 0.125, 0.0)                        # just off the left edge
    vis = rng.standard_normal((n, 4, 2)).astype(np.float32)
    w = rng.uniform(0.5, 1.5, n).astype(np.float32)
    return uvw, vis, w


# ------------------------------------------------------------------------------------ the mapping
@pytest.mark.parametrize("cfg", [0, 1])
def test_map_kernel_is_bit_exact_on_configs(dev, cfg):
    wl = synth.make_workload(cfg)
    g = _gridder(dev, N=wl.grid_size, du=wl.cell_size, O=wl.oversample, S=wl.support[0], table=wl.kernel,
                 max_vis=wl.n_vis)
    got = g.map(torch.from_numpy(wl.uvw).to(dev), torch.from_numpy(wl.freq).to(dev)).cpu().numpy()
    g.destroy()
    ref = oracle.map_visibilities(wl.uvw, wl.freq, **oracle_kwargs(wl))
    assert np.array_equal(got, ref)


@pytest.mark.parametrize("S,O,N", [(16, 4, 512), (7, 8, 256), (15, 8, 128), (8, 2, 64), (1, 2, 32)])
def test_map_kernel_is_bit_exact_on_adversarial_positions(dev, S, O, N):
    rng = np.random.default_rng(100 + S)
    n = 200_000
    pos = rng.uniform(-N / 2 - 3, N / 2 + 3, (n, 2))
    pos[:50_000] = (np.floor(pos[:50_000] * O) + 0.5) / O                     # exact half sub-cells
    pos[50_000:60_000] = np.round(pos[50_000:60_000] * O) / O                 # exact lattice points
    pos[60_000:70_000] = np.nextafter((np.floor(pos[60_000:70_000] * O) + 0.5) / O, -np.inf)
    pos[70_000:80_000] = np.nextafter((np.floor(pos[70_000:80_000] * O) + 0.5) / O, np.inf)
    pos[80_000] = (1e30, -1e30)
    pos[80_001] = (-1e18, 3.0)
    du = 0.37
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = pos * du                      # wavelengths; freq list below rescales them
    freq = np.array([C, C * (1 + 2.0 ** -20), 0.75 * C])
    table = np.zeros((S * O) ** 2, np.float32)
    g = _gridder(dev, N=N, du=du, O=O, S=S, table=table, max_vis=n * 3)
    got = g.map(torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev)).cpu().numpy()
    g.destroy()
    ref = oracle.map_visibilities(uvw, freq, grid_size=N, cell_size=du, oversample=O, support=[S], kernel=table)
    assert np.array_equal(got, ref)
    assert 0 < ref[:, 5].sum() < len(ref)


def _check_presum_map(got, ref):
    """gridder_map_presum reports a dropped visibility as 0, 0, 0, 0, 0, 1; everything else as gridder_map."""
    assert np.array_equal(got[:, 5], ref[:, 5])
    keep = ref[:, 5] == 0
    assert np.array_equal(got[keep], ref[keep])
    assert not got[~keep, :5].any()


@pytest.mark.parametrize("S,O,N", [(16, 4, 512), (7, 8, 256), (15, 8, 128), (8, 2, 64), (16, 1, 64)])
def test_presum_mapper_is_bit_exact_on_adversarial_positions(dev, S, O, N):
    """The PRODUCTION mapper of configs 2 and 4 (FastMap2: one FMA per axis, screened; csrc/map.cuh) on the
    same 600 000 adversarial positions -- exact half sub-cells, lattice points, their FP64 neighbours, far
    outliers -- with integer equality against the oracle's mapping."""
    rng = np.random.default_rng(100 + S)
    n = 200_000
    pos = rng.uniform(-N / 2 - 3, N / 2 + 3, (n, 2))
    pos[:50_000] = (np.floor(pos[:50_000] * O) + 0.5) / O
    pos[50_000:60_000] = np.round(pos[50_000:60_000] * O) / O
    pos[60_000:70_000] = np.nextafter((np.floor(pos[60_000:70_000] * O) + 0.5) / O, -np.inf)
    pos[70_000:80_000] = np.nextafter((np.floor(pos[70_000:80_000] * O) + 0.5) / O, np.inf)
    pos[80_000] = (1e30, -1e30)
    pos[80_001] = (-1e18, 3.0)
    pos[80_002] = (N * 1.4, 0.0)                   # beyond the fast range of the screen, inside the slow one
    du = 0.37
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = pos * du
    freq = np.array([C, C * (1 + 2.0 ** -20), 0.75 * C])
    table = np.zeros((S * O) ** 2, np.float32)
    g = _gridder(dev, N=N, du=du, O=O, S=S, table=table, max_vis=n * 3)
    got = g.map(torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev), presum=True).cpu().numpy()
    g.destroy()
    ref = oracle.map_visibilities(uvw, freq, grid_size=N, cell_size=du, oversample=O, support=[S], kernel=table)
    _check_presum_map(got, ref)
    assert 0 < ref[:, 5].sum() < len(ref)


def test_presum_mapper_is_bit_exact_on_config_2(dev):
    """Every visibility of BASELINE.json config 2 (130 816 baselines x 768 channels) through the production
    mapper, against the oracle's mapping, in blocks of 96 channels."""
    wl = synth.make_workload(2)
    g = _gridder(dev, N=wl.grid_size, du=wl.cell_size, O=wl.oversample, S=wl.support[0], table=wl.kernel, max_vis=1024)
    d_uvw = torch.from_numpy(wl.uvw).to(dev)
    for f0 in range(0, wl.n_chan, 96):
        freq = wl.freq[f0:f0 + 96]
        got = g.map(d_uvw, torch.from_numpy(freq).to(dev), presum=True).cpu().numpy()
        ref = oracle.map_visibilities(wl.uvw, freq, **oracle_kwargs(wl))
        _check_presum_map(got, ref)
    g.destroy()


# ------------------------------------------------------------------------------------ full grids
@pytest.mark.parametrize("cfg", [0, 1])
def test_parity_full_grid_configs(dev, cfg):
    wl = synth.make_workload(cfg)
    vis = wl.visibilities("cpu").numpy()
    got, st = _run(dev, wl.uvw, wl.freq, vis, None, N=wl.grid_size, du=wl.cell_size, O=wl.oversample,
                   S=wl.support[0], table=wl.kernel)
    ref, ab, ost = oracle.grid_full(wl.uvw, wl.freq, vis, None, **oracle_kwargs(wl))
    assert st.n_vis == wl.n_vis and st.n_dropped == ost["n_dropped"] == 0
    assert st.vis_taps == ost["vis_taps"] == wl.n_vis * wl.support[0] ** 2
    assert_parity(got, ref, ab, f"config {cfg}")


@pytest.mark.parametrize("S,O,N,n", [(16, 4, 96, 6000), (15, 8, 80, 5000), (7, 8, 64, 4000), (8, 4, 48, 3000),
                                     (9, 2, 70, 3000), (12, 4, 66, 3000), (3, 2, 34, 500), (1, 2, 20, 300)])
def test_parity_random_small(dev, S, O, N, n):
    rng = np.random.default_rng(S * 1000 + N)
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    uvw, vis, w = _random_case(rng, n, N, S)
    got, st = _run(dev, uvw, [C], vis, w, N=N, du=1.0, O=O, S=S, table=table)
    ref, ab, ost = _oracle(uvw, [C], vis, w, N=N, du=1.0, O=O, S=S, table=table)
    assert 0 < ost["n_dropped"] == st.n_dropped
    assert st.vis_taps == ost["vis_taps"] and st.n_entries == n - st.n_dropped
    assert_parity(got, ref, ab, f"S={S} O={O} N={N}")


@pytest.mark.parametrize("tlog", [2, 3, 4])
@pytest.mark.parametrize("S,O", [(16, 4), (7, 8)])
def test_parity_tile_sizes_and_ragged_grid(dev, S, O, tlog):
    """N not a multiple of the tile edge; every tile size the kernels are instantiated for."""
    rng = np.random.default_rng(7 + tlog)
    N, n = 90, 5000
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    uvw, vis, w = _random_case(rng, n, N, S)
    got, st = _run(dev, uvw, [C], vis, w, N=N, du=1.0, O=O, S=S, table=table, tuning={"tile_log2": tlog})
    ref, ab, ost = _oracle(uvw, [C], vis, w, N=N, du=1.0, O=O, S=S, table=table)
    assert st.tile_size == 1 << tlog and st.n_dropped == ost["n_dropped"]
    assert_parity(got, ref, ab, f"T={1 << tlog}")


def test_parity_hot_tile_is_split_into_chunks(dev):
    """All visibilities inside one tile, many more than K: the bounded overflow path."""
    rng = np.random.default_rng(11)
    N, S, O, n = 64, 16, 4, 20_000
    table = synth.spheroidal_table(S, O)
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = rng.uniform(-3.0, 3.0, (n, 2))
    vis = (rng.standard_normal((n, 4, 2)) + 3.0).astype(np.float32)          # coherent: sums grow
    got, st = _run(dev, uvw, [C], vis, None, N=N, du=1.0, O=O, S=S, table=table, tuning={"chunk": 512})
    ref, ab, _ = _oracle(uvw, [C], vis, None, N=N, du=1.0, O=O, S=S, table=table)
    assert st.chunk_size == 512 and st.n_work_items >= n // 512 and st.max_tile_load > 512
    assert st.n_work_items <= st.n_tiles_occupied + n // 512
    assert_parity(got, ref, ab, "hot tile")


def test_empty_and_single_inputs(dev):
    N, S, O = 32, 7, 8
    table = synth.spheroidal_table(S, O)
    got, st = _run(dev, np.zeros((1, 0, 3)), [C], np.zeros((0, 4, 2), np.float32), None, N=N, du=1.0, O=O, S=S,
                   table=table)
    assert st.n_vis == 0 and st.n_work_items == 0 and not got.any()
    uvw = np.zeros((1, 1, 3))
    vis = np.zeros((1, 4, 2), np.float32)
    vis[0, 3] = (2.0, -1.0)
    got, st = _run(dev, uvw, [C], vis, None, N=N, du=1.0, O=O, S=S, table=table)
    ref, ab, _ = _oracle(uvw, [C], vis, None, N=N, du=1.0, O=O, S=S, table=table)
    assert st.n_work_items == 1
    assert_parity(got, ref, ab, "single")
    # everything off the grid: nothing gridded, grid overwritten with zeros
    uvw[0, 0, :2] = (100.0, 0.0)
    got, st = _run(dev, uvw, [C], vis, None, N=N, du=1.0, O=O, S=S, table=table)
    assert st.n_dropped == 1 and st.vis_taps == 0 and not got.any()


def test_accumulate_and_zero_weights(dev):
    rng = np.random.default_rng(12)
    N, S, O, n = 64, 15, 8, 3000
    table = synth.spheroidal_table(S, O)
    uvw, vis, w = _random_case(rng, n, N, S, spread=20)
    w[::3] = 0.0
    base = rng.standard_normal((4, N, N, 2)).astype(np.float32)
    got, _ = _run(dev, uvw, [C], vis, w, N=N, du=1.0, O=O, S=S, table=table, accumulate_onto=base)
    ref, ab, _ = _oracle(uvw, [C], vis, w, N=N, du=1.0, O=O, S=S, table=table)
    assert_parity(got, ref + as_complex(base), ab + np.abs(as_complex(base)), "accumulate")
    keep = w != 0
    got2, _ = _run(dev, uvw[:, keep], [C], vis[keep], None, N=N, du=1.0, O=O, S=S, table=table)
    got1, _ = _run(dev, uvw, [C], vis, np.where(keep, 1.0, 0.0).astype(np.float32), N=N, du=1.0, O=O, S=S,
                   table=table)
    assert_parity(got1, as_complex(got2), ab, "zero weights contribute nothing")


# ------------------------------------------------------------------------------------ determinism
def test_reruns_and_launch_shapes_are_bit_identical(dev):
    wl = synth.make_workload(1, n_time=2)
    vis = wl.visibilities("cpu").numpy()
    kw = dict(N=wl.grid_size, du=wl.cell_size, O=wl.oversample, S=wl.support[0], table=wl.kernel)
    a, _ = _run(dev, wl.uvw, wl.freq, vis, None, **kw)
    b, _ = _run(dev, wl.uvw, wl.freq, vis, None, **kw)
    assert np.array_equal(a, b)
    # the number of resident warps changes which warp takes which work item, never the result
    c, st = _run(dev, wl.uvw, wl.freq, vis, None, tuning={"max_warps": 4}, **kw)
    assert st.grid_warps_per_sm == 4 and np.array_equal(a, c)
    # same plan: bin once, grid twice, and re-bin
    g = _gridder(dev, max_vis=wl.n_vis, **kw)
    d_uvw, d_f, d_v = torch.from_numpy(wl.uvw).to(dev), torch.from_numpy(wl.freq).to(dev), torch.from_numpy(vis).to(dev)
    g.bin(d_uvw, d_f)
    o1 = g.grid(d_v).cpu().numpy()
    o2 = g.grid(d_v).cpu().numpy()
    g.bin(d_uvw, d_f)
    o3 = g.grid(d_v).cpu().numpy()
    g.destroy()
    assert np.array_equal(o1, a) and np.array_equal(o2, a) and np.array_equal(o3, a)


def test_error_paths_on_device(dev):
    from paper_1003_5575_b200 import gridder
    table = torch.zeros(64 * 64, device=dev)
    g = gridder.Gridder(grid_size=64, cell_size=1.0, oversample=4, support=[16], kernel=table, max_vis=100)
    vis = torch.zeros((10, 4, 2), device=dev)
    with pytest.raises(gridder.GridderError) as e:
        g.grid(vis)
    assert e.value.code == gridder.ERR_NOT_BINNED
    with pytest.raises(gridder.GridderError) as e:
        g.bin(torch.zeros((1, 101, 3), dtype=torch.float64, device=dev), torch.tensor([C], dtype=torch.float64, device=dev))
    assert e.value.code == gridder.ERR_CAPACITY
    with pytest.raises(gridder.GridderError) as e:
        g.stats()
    assert e.value.code == gridder.ERR_NOT_BINNED
    g.destroy()
    with pytest.raises(gridder.GridderError) as e:
        gridder.Gridder(grid_size=64, cell_size=1.0, oversample=64, support=[32] * 64, n_wplanes=64, w_max=1.0,
                        kernel_is_complex=True, kernel=torch.zeros(8, device=dev), max_vis=100)
    assert e.value.code == gridder.ERR_UNSUPPORTED


# ------------------------------------------------------------------------------------ host buffers end to end
def test_run_host_sliced_copy_compute_overlap_matches_oracle(dev):
    """gridder_run_host on config 1 with pinned host buffers, forced into its sliced mode (copy of slice
    k+1 on a second stream while slice k is binned and gridded): within tolerance of the oracle, equal to
    the single-shot mode within a few FP32 roundings, and bit-identical between two calls."""
    from paper_1003_5575_b200 import gridder
    wl = synth.make_workload(1)
    vis = wl.visibilities("cpu").contiguous()
    h_uvw, h_freq = torch.from_numpy(wl.uvw).pin_memory(), torch.from_numpy(wl.freq).pin_memory()
    h_vis = vis.pin_memory()
    staging = {"uvw": torch.empty_like(h_uvw, device=dev), "freq": torch.empty_like(h_freq, device=dev),
               "vis": torch.empty_like(h_vis, device=dev), "weight": None,
               "grid": torch.empty((4, wl.grid_size, wl.grid_size, 2), dtype=torch.float32, device=dev)}
    outs = []
    for min_mb in (1, 1, 100000):                      # sliced, sliced again, single shot
        g = gridder.Gridder(grid_size=wl.grid_size, cell_size=wl.cell_size, oversample=wl.oversample, support=wl.support,
                            kernel=torch.from_numpy(wl.kernel).to(dev), max_vis=wl.n_vis,
                            tuning={"host_slice_min_mb": min_mb})
        h_grid = torch.empty((4, wl.grid_size, wl.grid_size, 2), dtype=torch.float32).pin_memory()
        g.run_host(h_uvw, h_freq, h_vis, None, h_grid, staging)
        outs.append(h_grid.numpy().copy())
        g.destroy()
    ref, ab, _ = oracle.grid_full(wl.uvw, wl.freq, vis.numpy(), None, **oracle_kwargs(wl))
    assert np.array_equal(outs[0], outs[1])
    assert_parity(outs[0], ref, ab, "run_host, sliced")
    assert_parity(outs[2], ref, ab, "run_host, single shot")
    assert np.abs(as_complex(outs[0]) - as_complex(outs[2])).max() <= 2e-6 * np.abs(ref).max()


def test_large_grid_takes_the_general_path(dev):
    """N = 16384 with O = 4: tile + origin + sub-cell bits need 33 key bits, so the plan switches to the
    general path (sub-cell offsets in the sort value).  Windows around a few visibilities against the oracle."""
    from paper_1003_5575_b200 import gridder
    rng = np.random.default_rng(16384)
    N, S, O, n = 16384, 16, 4, 4000
    table = synth.spheroidal_table(S, O)
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = rng.uniform(-N / 2 + 40, N / 2 - 40, (n, 2))
    uvw[0, :200, :2] = rng.uniform(-30.0, 30.0, (200, 2))                 # a busy patch in the middle
    vis = rng.standard_normal((n, 4, 2)).astype(np.float32)
    g = gridder.Gridder(grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=torch.from_numpy(table.ravel()).to(dev),
                        max_vis=n)
    g.bin(torch.from_numpy(uvw).to(dev), torch.tensor([C], dtype=torch.float64, device=dev))
    grid = g.grid(torch.from_numpy(vis).to(dev))
    st = g.stats()
    wins = [(N // 2 - 48, N // 2 + 48, N // 2 - 48, N // 2 + 48)]
    for k in (300, 1000, 2500, 3999):
        cx, cy = int(uvw[0, k, 0]) + N // 2, int(uvw[0, k, 1]) + N // 2
        wins.append((cy - 12, cy + 12, cx - 12, cx + 12))
    got = [grid[:, y0:y1, x0:x1].cpu().numpy() for (y0, y1, x0, x1) in wins]
    total = float(grid[..., 0].double().sum().item())
    g.destroy()
    del grid
    torch.cuda.empty_cache()
    res = oracle.grid_windows(uvw, [C], vis, None, wins, grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=table)
    assert st.n_dropped == res["n_dropped"] == 0 and st.vis_taps == res["vis_taps"] == n * S * S
    for k in range(len(wins)):
        assert res["A"][k].max() > 0
        assert_parity(got[k], res["G"][k], res["A"][k], f"N=16384 window {wins[k]}")
    # nothing is lost outside the windows either: total of the real parts = sum_i Re V_i * (per-offset table sum)
    m = oracle.map_visibilities(uvw, [C], grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=table)
    t64 = table.astype(np.float64)
    csum = np.array([[t64[qy::O, qx::O].sum() for qx in range(O)] for qy in range(O)])
    want = (vis[:, :, 0].astype(np.float64).sum(1) * csum[m[:, 3], m[:, 2]]).sum()
    assert abs(total - want) <= 1e-4 * np.abs(vis[:, :, 0]).sum() * csum.max() * 1e-1 + 1e-2


# ------------------------------------------------------------------------------------ merging
def test_merging_of_equal_origin_and_offset_entries(dev):
    """The grid kernel sums entries of a batch that share patch origin and sub-cell offset before gridding
    them (exact by linearity).  Many visibilities on few lattice points: the merged and the unmerged runs
    both match the oracle, the counters say what was executed, and a dense case really is merged."""
    rng = np.random.default_rng(91)
    N, S, O, n = 64, 16, 4, 20_000
    table = synth.spheroidal_table(S, O)
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = rng.integers(-6, 7, (n, 2)) / 2.0               # 13 x 13 lattice points: heavy duplication
    uvw[0, ::7, :2] += rng.uniform(-0.2, 0.2, (len(uvw[0, ::7]), 2))
    vis = (rng.standard_normal((n, 4, 2)) + 1.0).astype(np.float32)
    w = rng.uniform(0.5, 1.5, n).astype(np.float32)
    kw = dict(N=N, du=1.0, O=O, S=S, table=table)
    ref, ab, _ = _oracle(uvw, [C], vis, w, **kw)
    a, st_a = _run(dev, uvw, [C], vis, w, **kw)
    a2, _ = _run(dev, uvw, [C], vis, w, **kw)
    b, st_b = _run(dev, uvw, [C], vis, w, tuning={"merge": 2}, **kw)
    assert np.array_equal(a, a2)
    assert_parity(a, ref, ab, "merging on")
    assert_parity(b, ref, ab, "merging off")
    assert st_b.n_records_gridded == st_b.n_vis == n                 # unmerged: one record per entry (none dropped)
    assert st_b.fma_executed == n * 256 * 8
    assert st_a.n_records_gridded < n // 3 and st_a.fma_executed == st_a.n_records_gridded * 256 * 8
    # one work item per tile: with the per-origin bins carried from batch to batch the grid kernel grids every
    # distinct (origin, offset) exactly once -- the count is the oracle's number of distinct lattice points
    c, st_c = _run(dev, uvw, [C], vis, w, tuning={"chunk": 32768}, **kw)
    m = oracle.map_visibilities(np.ascontiguousarray(uvw), [C], grid_size=N, cell_size=1.0, oversample=O, support=[S],
                                kernel=np.ascontiguousarray(table, np.float32).ravel())
    live = m[m[:, 5] == 0]
    assert st_c.n_records_gridded == len(np.unique(live[:, :4], axis=0))
    assert_parity(c, ref, ab, "merging on, one item per tile")


@pytest.mark.parametrize("S,O,N,n,tuning", [(16, 4, 96, 6000, {}), (12, 4, 66, 3000, {"merge": 2}),
                                            (16, 4, 80, 8000, {"tile_log2": 3}), (7, 8, 64, 3000, {})])
def test_table_in_tensor_memory(dev, S, O, N, n, tuning):
    """table_in_tmem: the GCF table is read with tcgen05.ld instead of LDS (the default for pre-summed plans,
    where the grid kernel runs on partial records); same bits as the shared-memory table."""
    rng = np.random.default_rng(S + N + n)
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    uvw, vis, w = _random_case(rng, n, N, S)
    kw = dict(N=N, du=1.0, O=O, S=S, table=table)
    a, _ = _run(dev, uvw, [C], vis, w, tuning=dict(tuning, table_in_tmem=1), **kw)
    b, _ = _run(dev, uvw, [C], vis, w, tuning=dict(tuning, table_in_tmem=2), **kw)
    ref, ab, _ = _oracle(uvw, [C], vis, w, **kw)
    assert np.array_equal(a, b)
    assert_parity(a, ref, ab, f"tensor-memory table S={S} O={O}")


def test_table_too_large_for_shared_memory_takes_the_general_path(dev):
    """S = 16 with O = 16 is a 256 KB table: more than an SM's shared memory.  The plan must not fail: it reads
    the table from global memory (the general path) and still matches the oracle."""
    rng = np.random.default_rng(1616)
    N, S, O, n = 96, 16, 16, 3000
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    uvw, vis, w = _random_case(rng, n, N, S)
    kw = dict(N=N, du=1.0, O=O, S=S, table=table)
    got, st = _run(dev, uvw, [C], vis, w, **kw)
    ref, ab, ost = _oracle(uvw, [C], vis, w, **kw)
    assert st.n_dropped == ost["n_dropped"] and st.vis_taps == ost["vis_taps"]
    assert_parity(got, ref, ab, "S=16 O=16")
