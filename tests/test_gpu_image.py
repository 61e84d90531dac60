"""the imaging step (centred inverse FFT + grid correction) against the oracle's imager.
Tolerance (written out here because north_star states none for this row): every image pixel is a sum of
N^2 grid cells times unit-modulus factors, so an FP32 FFT can be off by a few ulp times log2(N^2) of the
L1 norm at worst; the test allows 2e-6 * corr[y] corr[x] * sum|G| -- tight enough that any wrong sign,
shift or transposition fails, because the sparse cases below have |image| ~ sum|G|."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import as_complex

pytestmark = pytest.mark.gpu
RTOL_L1 = 2e-6


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5575_b200 import gridder
    gridder.load_library()
    return torch.device("cuda:0")


def _plan(dev, N):
    from paper_1003_5575_b200 import gridder
    return gridder.Gridder(grid_size=N, cell_size=1.0, oversample=4, support=[16],
                           kernel=torch.from_numpy(synth.spheroidal_table(16, 4).ravel()).to(dev), max_vis=16)


@pytest.mark.parametrize("N,sparse", [(64, False), (64, True), (96, True), (250, False)])
def test_image_matches_oracle_small(dev, N, sparse):
    rng = np.random.default_rng(N + sparse)
    grid = rng.standard_normal((4, N, N, 2)).astype(np.float32)
    if sparse:
        keep = np.zeros((4, N, N, 1), np.float32)
        idx = rng.integers(0, N, (12, 3))
        keep[idx[:, 0] % 4, idx[:, 1], idx[:, 2]] = 1.0
        grid *= keep
    corr = rng.uniform(0.5, 2.0, N).astype(np.float32)
    g = _plan(dev, N)
    d_grid = torch.from_numpy(grid).to(dev)
    got = g.image(d_grid, torch.from_numpy(corr).to(dev)).cpu().numpy()
    plain = g.image(d_grid).cpu().numpy()
    inplace = g.image(d_grid, torch.from_numpy(corr).to(dev), out=d_grid).cpu().numpy()
    g.destroy()
    gc = as_complex(grid)
    ref = oracle.image(gc, corr.astype(np.float64))
    l1 = np.abs(gc).sum(axis=(1, 2))[:, None, None]
    tol = RTOL_L1 * l1 * (corr[:, None] * corr[None, :])[None] + 1e-6
    err = np.abs(as_complex(got) - ref)
    assert (err <= tol).all(), f"worst err/tol {(err / tol).max():.3f}"
    assert (np.abs(as_complex(plain) - oracle.image(gc)) <= RTOL_L1 * l1 + 1e-6).all()
    assert np.array_equal(inplace, got), "in-place imaging must give the same bits"


def test_image_full_size_sampled_pixels(dev):
    """N = 4096 (the configs' grid): a grid with 60 non-zero cells, image pixels sampled and summed directly."""
    N = 4096
    rng = np.random.default_rng(9)
    cells = np.stack([rng.integers(0, 4, 60), rng.integers(0, N, 60), rng.integers(0, N, 60)], 1)
    vals = rng.standard_normal(60) + 1j * rng.standard_normal(60)
    t1 = synth.spheroidal_1d(16, 4)
    corr = oracle.grid_correction(t1.astype(np.float32), 16, 4, N)
    corr[np.abs(np.arange(N) - N // 2) > 0.45 * N] = 1.0          # the taper's zero is at the very edge
    g = _plan(dev, N)
    d_grid = torch.zeros((4, N, N, 2), dtype=torch.float32, device=dev)
    h = np.zeros((60, 2), np.float32)
    h[:, 0], h[:, 1] = vals.real, vals.imag
    d_grid[cells[:, 0], cells[:, 1], cells[:, 2]] = torch.from_numpy(h).to(dev)
    img = g.image(d_grid, torch.from_numpy(corr.astype(np.float32)).to(dev))
    v32 = h[:, 0].astype(np.float64) + 1j * h[:, 1].astype(np.float64)
    px = np.stack([rng.integers(0, 4, 200), rng.integers(0, N, 200), rng.integers(0, N, 200)], 1)
    px[:4] = [[0, N // 2, N // 2], [1, 0, 0], [2, N - 1, N - 1], [3, N // 2, 0]]
    got = as_complex(img[px[:, 0], px[:, 1], px[:, 2]].cpu().numpy())
    g.destroy()
    c32 = corr.astype(np.float32).astype(np.float64)
    worst = 0.0
    for (pol, y, x), gv in zip(px, got):
        m = cells[:, 0] == pol
        ph = np.exp(2j * np.pi * ((cells[m, 2] - N // 2) * (x - N // 2) + (cells[m, 1] - N // 2) * (y - N // 2)) / N)
        want = c32[y] * c32[x] * (v32[m] * ph).sum()
        tol = RTOL_L1 * c32[y] * c32[x] * np.abs(v32[m]).sum() + 1e-6
        worst = max(worst, abs(gv - want) / tol)
    assert worst <= 1.0, f"worst err/tol {worst:.3f}"
