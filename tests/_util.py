"""Shared helpers of the GPU parity tests (comparison only; no gridding arithmetic here)."""
import numpy as np

RTOL_ABS = 1e-5     # BASELINE.json north_star: |delta| <= 1e-5 * sum|w V C| + 1e-6 per cell
ATOL = 1e-6


def as_complex(grid_f32):
    g = np.asarray(grid_f32)
    return g[..., 0].astype(np.float64) + 1j * g[..., 1].astype(np.float64)


def assert_parity(got_f32, ref_c128, abs_f64, what=""):
    """Per cell and polarisation: |G_gpu - G| <= 1e-5 * Abs + 1e-6 (complex modulus)."""
    err = np.abs(as_complex(got_f32) - ref_c128)
    tol = RTOL_ABS * abs_f64 + ATOL
    bad = err > tol
    worst = float((err / tol).max()) if err.size else 0.0
    assert not bad.any(), f"{what}: {int(bad.sum())} cells out of tolerance, worst err/tol = {worst:.3f}"
    return worst


def oracle_kwargs(wl):
    return dict(grid_size=wl.grid_size, cell_size=wl.cell_size, oversample=wl.oversample,
                support=wl.support, kernel=wl.kernel, w_max=wl.w_max,
                kernel_is_complex=wl.kernel_is_complex)
