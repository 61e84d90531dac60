"""SURVEY 8(f) row f4, second half: batched per-channel grids (PAPER.md :108-120 -- a GPU holds 12 consecutive
channels and makes one image of each).  One gridder_bin_channels over all channels, one gridder_grid_channels
writing one grid per channel block; every grid against an ORACLE run on that block's channels alone."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import as_complex, assert_parity

pytestmark = pytest.mark.gpu
C = 299_792_458.0


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5575_b200 import gridder
    gridder.load_library()
    return torch.device("cuda:0")


def _case(rng, nt, nb, nf, N, band):
    uvw = np.zeros((nt, nb, 3))
    uvw[0, :, :2] = rng.uniform(-N / 2 - 2, N / 2 + 2, (nb, 2)) / (1.0 + band * nf)
    rot = 4e-4 * np.arange(nt)[:, None]
    uvw[:, :, 0] = uvw[0, :, 0] * np.cos(rot) - uvw[0, :, 1] * np.sin(rot)
    uvw[:, :, 1] = uvw[0, :, 0] * np.sin(rot) + uvw[0, :, 1] * np.cos(rot)
    uvw[:, :, 2] = rng.uniform(-1.0, 1.0, (1, nb))
    freq = C * (1.0 + band * np.arange(nf))
    vis = rng.standard_normal((nt, nb, nf, 4, 2)).astype(np.float32)
    w = rng.uniform(0.5, 1.5, (nt, nb, nf)).astype(np.float32)
    return uvw, freq, vis, w


@pytest.mark.parametrize("tuning", [{"presum": 1}, {"presum": 2}, {"presum": 1, "tile_log2": 2, "chunk": 64}])
def test_twelve_channel_grids_against_twelve_oracle_runs(dev, tuning):
    from paper_1003_5575_b200 import gridder
    rng = np.random.default_rng(1212)
    nt, nb, nf, N, S, O, per = 4, 400, 12, 128, 16, 4, 1          # the paper's shape: 12 channels, one grid each
    table = synth.spheroidal_table(S, O).astype(np.float32)
    uvw, freq, vis, w = _case(rng, nt, nb, nf, N, 3e-3)
    g = gridder.Gridder(grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=torch.from_numpy(table.ravel()).to(dev),
                        max_vis=nt * nb * nf, max_grids=12, tuning=tuning)
    d_uvw, d_f = torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev)
    d_v, d_w = torch.from_numpy(vis).to(dev), torch.from_numpy(w).to(dev)
    g.bin(d_uvw, d_f, chans_per_grid=per)
    out1 = g.grid(d_v, d_w).cpu().numpy()
    out2 = g.grid(d_v, d_w).cpu().numpy()
    st = g.stats()
    g.destroy()
    assert out1.shape == (12, 4, N, N, 2) and np.array_equal(out1, out2)
    dropped = taps = 0
    for k in range(12):
        sl = slice(k * per, (k + 1) * per)
        ref, ab, ost = oracle.grid_full(uvw, freq[sl], np.ascontiguousarray(vis[:, :, sl]), np.ascontiguousarray(w[:, :, sl]),
                                        grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=table.ravel())
        dropped += ost["n_dropped"]
        taps += ost["vis_taps"]
        assert np.abs(ref).max() > 0
        assert_parity(out1[k], ref, ab, f"channel grid {k} {tuning}")
    assert st.n_dropped == dropped > 0 and st.vis_taps == taps


def test_channel_blocks_ragged_accumulate_wplanes_and_errors(dev):
    """26 channels in blocks of 4 (the last grid holds 2), complex w-plane tables (the general path), accumulate
    onto existing grids; plain gridder_grid after a multi-grid bin and too many grids are refused."""
    from paper_1003_5575_b200 import gridder
    rng = np.random.default_rng(2626)
    nt, nb, nf, N, O, per = 2, 500, 26, 96, 2, 4
    supports = [8, 12, 22]
    table = np.concatenate([rng.standard_normal((s * O, s * O, 2)).astype(np.float32).ravel() for s in supports])
    uvw, freq, vis, w = _case(rng, nt, nb, nf, N, 2e-3)
    n_grids = 7
    g = gridder.Gridder(grid_size=N, cell_size=1.0, oversample=O, support=supports, kernel=torch.from_numpy(table).to(dev),
                        max_vis=nt * nb * nf, n_wplanes=3, w_max=1.0, kernel_is_complex=True, max_grids=8)
    d_uvw, d_f = torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev)
    d_v, d_w = torch.from_numpy(vis).to(dev), torch.from_numpy(w).to(dev)
    g.bin(d_uvw, d_f, chans_per_grid=per)
    base = rng.standard_normal((n_grids, 4, N, N, 2)).astype(np.float32)
    out = torch.from_numpy(base.copy()).to(dev)
    g.grid(d_v, d_w, out=out, accumulate=True)
    got = out.cpu().numpy()
    # binned for 7 grids: the one-grid call is refused
    assert g._lib.gridder_grid(g._plan, d_v.data_ptr(), d_w.data_ptr(), out.data_ptr(), 0, None) == gridder.ERR_INVALID_ARG
    with pytest.raises(gridder.GridderError) as e:
        g.bin(d_uvw, d_f, chans_per_grid=2)                  # 13 grids > max_grids = 8
    assert e.value.code == gridder.ERR_CAPACITY
    g.bin(d_uvw, d_f)                                        # and back to one grid on the same plan
    one = g.grid(d_v, d_w).cpu().numpy()
    g.destroy()
    kw = dict(grid_size=N, cell_size=1.0, oversample=O, support=supports, kernel=table, w_max=1.0, kernel_is_complex=True)
    total = np.zeros((4, N, N), np.complex128)
    total_ab = np.zeros((4, N, N))
    for k in range(n_grids):
        sl = slice(k * per, min(nf, (k + 1) * per))
        ref, ab, _ = oracle.grid_full(uvw, freq[sl], np.ascontiguousarray(vis[:, :, sl]), np.ascontiguousarray(w[:, :, sl]), **kw)
        assert_parity(got[k], ref + as_complex(base[k]), ab + np.abs(as_complex(base[k])), f"accumulated channel grid {k}")
        total += ref
        total_ab += ab
    assert_parity(one, total, total_ab, "all channels on one grid")
