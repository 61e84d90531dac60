"""GPU parity of the general path: several w-planes, variable support 1..32 (8-, 16- and 2x2x16-cell
patch classes), complex tables conjugated for w < 0 (BASELINE.json config 3; R13), and real
tables read from global memory.  Same bar as test_gpu_parity.py: integer work bit-exact, grid cells
within 1e-5 * sum|w V C| + 1e-6, reruns bit-identical."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import assert_parity

pytestmark = pytest.mark.gpu
C = 299_792_458.0


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5575_b200 import gridder
    gridder.load_library()
    return torch.device("cuda:0")


def _tables(rng, supports, O, cplx):
    parts = []
    for s in supports:
        shape = (s * O, s * O, 2) if cplx else (s * O, s * O)
        parts.append(rng.standard_normal(shape).astype(np.float32).ravel())
    return np.concatenate(parts)


def _case(rng, n, N, w_max, n_tie=40):
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = rng.uniform(-N / 2 - 1, N / 2 + 1, (n, 2))
    uvw[0, :, 2] = rng.uniform(-1.05 * w_max, 1.05 * w_max, n)          # beyond w_max: clamps to the last plane
    uvw[0, :n_tie, :2] = (np.floor(uvw[0, :n_tie, :2] * 4) + 0.5) / 4    # rounding ties
    uvw[0, n_tie:2 * n_tie, 2] = 0.0                                     # w = 0: plane 0, not conjugated
    vis = rng.standard_normal((n, 4, 2)).astype(np.float32)
    w = rng.uniform(0.5, 1.5, n).astype(np.float32)
    return uvw, vis, w


def _both(dev, uvw, freq, vis, weight, *, N, du, O, supports, table, w_max, cplx, tuning=None):
    from paper_1003_5575_b200 import gridder
    n = uvw.shape[0] * uvw.shape[1] * len(freq)
    g = gridder.Gridder(grid_size=N, cell_size=du, oversample=O, support=list(supports),
                        kernel=torch.from_numpy(table).to(dev), max_vis=max(n, 1), n_wplanes=len(supports),
                        w_max=w_max, kernel_is_complex=cplx, tuning=tuning)
    d_uvw = torch.from_numpy(np.ascontiguousarray(uvw)).to(dev)
    d_f = torch.tensor(np.asarray(freq, np.float64), device=dev)
    got_map = g.map(d_uvw, d_f).cpu().numpy()
    g.bin(d_uvw, d_f)
    d_vis = torch.from_numpy(np.ascontiguousarray(vis)).to(dev)
    d_w = None if weight is None else torch.from_numpy(np.ascontiguousarray(weight)).to(dev)
    out1 = g.grid(d_vis, d_w).cpu().numpy()
    out2 = g.grid(d_vis, d_w).cpu().numpy()
    st = g.stats()
    g.destroy()
    kw = dict(grid_size=N, cell_size=du, oversample=O, support=list(supports), kernel=table, w_max=w_max,
              kernel_is_complex=cplx)
    ref_map = oracle.map_visibilities(uvw, freq, **kw)
    ref, ab, ost = oracle.grid_full(uvw, freq, vis, weight, **kw)
    assert np.array_equal(got_map, ref_map), "map (x0, y0, qx, qy, plane|conj, dropped) differs from the oracle"
    assert st.n_dropped == ost["n_dropped"] and st.vis_taps == ost["vis_taps"]
    assert np.array_equal(out1, out2), "rerun is not bit-identical"
    return out1, ref, ab, st, ost


@pytest.mark.parametrize("S,O,N,n", [(16, 4, 96, 5000), (7, 8, 64, 4000), (15, 8, 80, 3000), (3, 2, 34, 500)])
def test_general_path_equals_oracle_on_single_real_table(dev, S, O, N, n):
    """The global-table kernels (MODE 1) on the shapes the fast path also handles."""
    rng = np.random.default_rng(S * 7 + N)
    table = _tables(rng, [S], O, False)
    uvw, vis, w = _case(rng, n, N, 1.0)
    got, ref, ab, st, _ = _both(dev, uvw, [C], vis, w, N=N, du=1.0, O=O, supports=[S], table=table, w_max=1.0,
                                cplx=False, tuning={"force_general": 1})
    assert st.n_dropped > 0
    assert_parity(got, ref, ab, f"general real S={S}")


@pytest.mark.parametrize("S,O,N,n", [(17, 2, 80, 3000), (24, 4, 96, 3000), (32, 4, 120, 3000), (31, 2, 100, 2000)])
def test_large_support_uses_four_sub_patches(dev, S, O, N, n):
    rng = np.random.default_rng(S)
    table = _tables(rng, [S], O, False)
    uvw, vis, w = _case(rng, n, N, 1.0)
    got, ref, ab, st, _ = _both(dev, uvw, [C], vis, w, N=N, du=1.0, O=O, supports=[S], table=table, w_max=1.0,
                                cplx=False)
    assert st.patch_size == 32
    assert_parity(got, ref, ab, f"real S={S}")


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("tlog", [2, 3])
def test_wplanes_mixed_supports_all_three_patch_classes(dev, cplx, tlog):
    rng = np.random.default_rng(5 + tlog + 10 * cplx)
    supports = [4, 8, 8, 10, 14, 16, 18, 26, 32]
    O, N, n, w_max = 4, 128, 12000, 37.5
    table = _tables(rng, supports, O, cplx)
    uvw, vis, w = _case(rng, n, N, w_max)
    vis2 = np.stack([vis, vis[::-1]], 1).copy()               # [n][2 channels][4][2]
    w2 = np.stack([w, w[::-1]], 1).copy()
    got, ref, ab, st, ost = _both(dev, uvw, [C, 0.9 * C], vis2, w2, N=N, du=1.0, O=O, supports=supports, table=table,
                                  w_max=w_max, cplx=cplx, tuning={"tile_log2": tlog})
    assert st.tile_size == 1 << tlog and 0 < st.n_dropped < 2 * n
    assert_parity(got, ref, ab, f"w-planes cplx={cplx} T={1 << tlog}")


def test_wplanes_hot_tile_chunks_and_unit_weights(dev):
    rng = np.random.default_rng(77)
    supports = [8, 12, 20]
    O, N, n, w_max = 2, 64, 9000, 3.0
    table = _tables(rng, supports, O, True)
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = rng.uniform(-2.0, 2.0, (n, 2))
    uvw[0, :, 2] = rng.uniform(-3.0, 3.0, n)
    vis = (rng.standard_normal((n, 4, 2)) + 2.0).astype(np.float32)
    got, ref, ab, st, _ = _both(dev, uvw, [C], vis, None, N=N, du=1.0, O=O, supports=supports, table=table, w_max=w_max,
                                cplx=True, tuning={"chunk": 256})
    assert st.chunk_size == 256 and st.max_tile_load > 256 and st.n_work_items > n // 256
    assert_parity(got, ref, ab, "w-planes hot tile")


def test_config3_reduced_full_grid(dev):
    """BASELINE.json config 3 (32 complex w-planes, support 8..32, 4096^2 grid), first 2 channels."""
    wl = synth.make_workload(3, n_chan=2)
    vis = wl.visibilities("cpu").numpy()
    got, ref, ab, st, ost = _both(dev, wl.uvw, wl.freq, vis, None, N=wl.grid_size, du=wl.cell_size, O=wl.oversample,
                                  supports=wl.support, table=wl.kernel, w_max=wl.w_max, cplx=True)
    assert st.n_dropped == 0 and st.n_vis == wl.n_vis
    assert_parity(got, ref, ab, "config 3 (2 channels)")


@pytest.mark.parametrize("cplx", [False, True])
def test_per_baseline_tables_row_f3(dev, cplx):
    """gridder_bin_tables: every (integration, baseline) names its own table of the plan's bank
    (PAPER.md :73, :179); indices outside the bank drop the baseline; w only decides conjugation."""
    from paper_1003_5575_b200 import gridder
    rng = np.random.default_rng(61 + cplx)
    supports = [6, 8, 12, 16, 22, 32]
    O, N, nb, nf, w_max = 2, 128, 3000, 3, 1.0
    table = _tables(rng, supports, O, cplx)
    uvw = np.zeros((2, nb, 3))
    uvw[:, :, :2] = rng.uniform(-N / 2 - 1, N / 2 + 1, (2, nb, 2)) / 1.1
    uvw[:, :, 2] = rng.uniform(-3.0, 3.0, (2, nb))
    freq = C * np.array([1.0, 1.05, 1.1])
    idx = rng.integers(0, len(supports), (2, nb)).astype(np.int32)
    idx[0, :4] = (-1, len(supports), 1 << 20, -(1 << 20))
    vis = rng.standard_normal((2, nb, nf, 4, 2)).astype(np.float32)
    w = rng.uniform(0.5, 1.5, (2, nb, nf)).astype(np.float32)
    g = gridder.Gridder(grid_size=N, cell_size=1.0, oversample=O, support=supports, kernel=torch.from_numpy(table).to(dev),
                        max_vis=2 * nb * nf, n_wplanes=len(supports), w_max=w_max, kernel_is_complex=cplx)
    d_uvw, d_f = torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev)
    d_idx = torch.from_numpy(idx).to(dev)
    got_map = g.map(d_uvw, d_f, table_index=d_idx).cpu().numpy()
    g.bin(d_uvw, d_f, table_index=d_idx)
    out1 = g.grid(torch.from_numpy(vis).to(dev), torch.from_numpy(w).to(dev)).cpu().numpy()
    out2 = g.grid(torch.from_numpy(vis).to(dev), torch.from_numpy(w).to(dev)).cpu().numpy()
    st = g.stats()
    g.destroy()
    kw = dict(grid_size=N, cell_size=1.0, oversample=O, support=supports, kernel=table, w_max=w_max,
              kernel_is_complex=cplx, table_index=idx)
    assert np.array_equal(got_map, oracle.map_visibilities(uvw, freq, **kw))
    ref, ab, ost = oracle.grid_full(uvw, freq, vis, w, **kw)
    assert st.n_dropped == ost["n_dropped"] >= 4 * nf and st.vis_taps == ost["vis_taps"]
    assert np.array_equal(out1, out2)
    assert_parity(out1, ref, ab, f"per-baseline tables, complex={cplx}")


@pytest.mark.parametrize("presum", [1, 2])
def test_per_baseline_tables_bank_of_one_on_the_fast_path(dev, presum):
    """A bank of ONE real table takes the fast path, where there is nothing to choose -- but an index outside
    the bank must still drop its baseline (include/gridder.h), as the oracle does.  Whether or not the plan
    would pre-sum: a table_index always goes through the per-visibility map."""
    from paper_1003_5575_b200 import gridder
    rng = np.random.default_rng(71)
    S, O, N, nb, nf = 16, 4, 96, 2000, 4
    table = _tables(rng, [S], O, False)
    uvw = np.zeros((1, nb, 3))
    uvw[:, :, :2] = rng.uniform(-N / 2 + S, N / 2 - S, (1, nb, 2)) / 1.1
    freq = C * np.array([1.0, 1.01, 1.02, 1.03])
    idx = np.zeros((1, nb), np.int32)
    idx[0, ::7] = -1
    idx[0, 3::11] = 1
    vis = rng.standard_normal((1, nb, nf, 4, 2)).astype(np.float32)
    g = gridder.Gridder(grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=torch.from_numpy(table).to(dev),
                        max_vis=nb * nf, tuning={"presum": presum})
    d_uvw, d_f, d_idx = torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev), torch.from_numpy(idx).to(dev)
    got_map = g.map(d_uvw, d_f, table_index=d_idx).cpu().numpy()
    g.bin(d_uvw, d_f, table_index=d_idx)
    out = g.grid(torch.from_numpy(vis).to(dev)).cpu().numpy()
    st = g.stats()
    g.destroy()
    kw = dict(grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=table, table_index=idx)
    assert np.array_equal(got_map, oracle.map_visibilities(uvw, freq, **kw))
    ref, ab, ost = oracle.grid_full(uvw, freq, vis, None, **kw)
    n_bad = int(((idx < 0) | (idx > 0)).sum()) * nf
    assert st.n_dropped == ost["n_dropped"] == n_bad and st.vis_taps == ost["vis_taps"] and st.n_presum_records == 0
    assert_parity(out, ref, ab, "bank of one table with indices outside it")


@pytest.mark.parametrize("cplx", [False, True])
def test_carried_bins_grid_every_plane_origin_offset_once(dev, cplx):
    """Long runs of one (plane, origin) across many batches, both signs of w, every sub-cell offset: with the per-run
    bins (grid.cu stage_write_bins) the grid kernel grids each distinct (plane, conjugate, origin, offset) of a work
    item exactly once -- the count is pinned against the oracle's mapping -- and the sums stay within tolerance."""
    rng = np.random.default_rng(91 + cplx)
    supports = [12, 16]                                       # one patch class (16 cells), two tables
    O, N, n, w_max = 4, 64, 7000, 2.0
    table = _tables(rng, supports, O, cplx)
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = rng.uniform(-1.4, 1.4, (n, 2))            # a handful of origins, all of one 8 x 8 tile or two
    uvw[0, :, 2] = rng.uniform(-2.0, 2.0, n)
    uvw[0, :200, :2] = 0.3                                    # and one lattice point met 200 times
    vis = rng.standard_normal((n, 4, 2)).astype(np.float32)
    w = rng.uniform(0.5, 1.5, n).astype(np.float32)
    got, ref, ab, st, ost = _both(dev, uvw, [C], vis, w, N=N, du=1.0, O=O, supports=supports, table=table, w_max=w_max,
                                  cplx=cplx, tuning={"chunk": 16384})
    m = oracle.map_visibilities(uvw, [C], grid_size=N, cell_size=1.0, oversample=O, support=supports, kernel=table,
                                w_max=w_max, kernel_is_complex=cplx)
    live = m[m[:, 5] == 0]
    if not cplx:
        live = live.copy()
        live[:, 4] &= 255                                     # real tables: the sign of w changes nothing
    distinct = len(np.unique(live[:, :5], axis=0))
    assert st.n_dropped == 0 and st.n_work_items <= 4
    assert st.n_records_gridded == distinct < n // 4
    assert_parity(got, ref, ab, f"carried bins cplx={cplx}")
