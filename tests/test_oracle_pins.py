"""Pins for the oracle (oracle/gridder_oracle.c): it is checked against what the paper and the
mathematics fix, never against itself and never against the CUDA path.  All CPU, no GPU.

P1 unit visibility reproduces the table (BASELINE.json invariant 1)
P2 linearity (invariant 2)            P3 total-sum identity (invariant 3)
P4 grid -> inverse FFT -> grid correction == brute-force direct DFT within 1e-3 (invariant 4)
P5 brute-force gather restatement   P6 "around 60 visibilities per pixel" (:183)
P7 the spheroidal table against its textbook definition
"""
from pathlib import Path

import numpy as np
import pytest

import oracle
from synth import kernels

C = 299_792_458.0   # with freq = C the oracle's scale f/c is exactly 1: "metres" are wavelengths


def _grid(uv, vis, weight=None, *, N, S, O, table, du=1.0, w=None, **kw):
    uvw = np.zeros((1, len(uv), 3))
    uvw[0, :, :2] = uv
    if w is not None:
        uvw[0, :, 2] = w
    g, a, st = oracle.grid_full(uvw, [C], vis, weight, grid_size=N, cell_size=du, oversample=O,
                                support=S if isinstance(S, (list, tuple)) else [S], kernel=table, **kw)
    return g, a, st


def _vis(n, rng):
    return rng.standard_normal((n, 4, 2)).astype(np.float32)


def _gather_bruteforce(uv, vis, weight, N, S, O, table2d, du=1.0):
    """PAPER.md:181/:195 as a gather: every cell looks at every visibility, measures the distance
    from the (1/O-lattice) visibility position to its own centre and, if the table covers that
    distance, takes table[distance] * w * V.  No patch origin, no offset index: only
    'sample j of the table sits at r = (j - S*O/2)/O cells'."""
    out = np.zeros((4, N, N), dtype=np.complex128)
    v = vis[..., 0].astype(np.float64) + 1j * vis[..., 1].astype(np.float64)
    n_drop = 0
    for i, (u_, v_) in enumerate(uv):
        X = int(np.floor((u_ / du + N // 2) * O + 0.5))
        Y = int(np.floor((v_ / du + N // 2) * O + 0.5))
        cells_x = [c for c in range(-4 * S, N + 4 * S) if 0 <= c * O - X + (S * O) // 2 < S * O]
        cells_y = [c for c in range(-4 * S, N + 4 * S) if 0 <= c * O - Y + (S * O) // 2 < S * O]
        if min(cells_x) < 0 or max(cells_x) >= N or min(cells_y) < 0 or max(cells_y) >= N:
            n_drop += 1     # reading R7: a visibility with any tap off the grid is dropped whole
            continue
        wgt = 1.0 if weight is None else float(weight[i])
        for cy in cells_y:
            jy = cy * O - Y + (S * O) // 2
            for cx in cells_x:
                jx = cx * O - X + (S * O) // 2
                out[:, cy, cx] += wgt * v[i] * float(table2d[jy, jx])
    return out, n_drop


# ----------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("S,O", [(7, 8), (16, 4), (15, 8), (8, 4), (6, 2)])
def test_p1_unit_visibility_reproduces_table(S, O):
    N = 64
    rng = np.random.default_rng(1)
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)   # any table: no symmetry to hide behind
    k_x, k_y = 30, 35
    for my in range(O):
        for mx in range(O):
            uv = np.array([[k_x - N // 2 + mx / O, k_y - N // 2 + my / O]])
            vis = np.zeros((1, 4, 2), np.float32)
            vis[0, 2, 0] = 1.0                                       # unit, one polarisation
            g, a, st = _grid(uv, vis, N=N, S=S, O=O, table=table)
            assert st["n_dropped"] == 0 and st["vis_taps"] == S * S
            # expected straight from the table's meaning: cell c sees distance r = c - (k + m/O),
            # i.e. table sample j = r*O + S*O/2
            exp = np.zeros((N, N))
            for cy in range(N):
                jy = (cy - k_y) * O - my + (S * O) // 2
                if not 0 <= jy < S * O:
                    continue
                for cx in range(N):
                    jx = (cx - k_x) * O - mx + (S * O) // 2
                    if 0 <= jx < S * O:
                        exp[cy, cx] = table[jy, jx]
            assert np.array_equal(g[2].real, exp)                    # exact: 1.0 * table value
            assert not g[2].imag.any() and not g[[0, 1, 3]].any()
            assert np.array_equal(a[2], np.abs(exp))


def test_p1_centre_conventions_even_and_odd_support():
    N, k = 32, 16
    uv = np.array([[0.0, 0.0]])                                       # exactly on cell centre (N/2, N/2)
    vis = np.zeros((1, 4, 2), np.float32)
    vis[0, 0, 0] = 1.0
    # even S: offset 0, patch [k - S/2, k + S/2), tap t at distance t - S/2
    S, O = 8, 4
    t = kernels.spheroidal_table(S, O)
    g, _, _ = _grid(uv, vis, N=N, S=S, O=O, table=t)
    assert np.array_equal(g[0, k - 4:k + 4, k - 4:k + 4].real, t[0::O, 0::O])
    assert np.count_nonzero(g[0]) <= S * S
    # odd S: offset O/2, patch [k - 3, k + 3], integer distances, centre tap psi(0)^2 = 1 on k
    S, O = 7, 8
    t = kernels.spheroidal_table(S, O)
    g, _, _ = _grid(uv, vis, N=N, S=S, O=O, table=t)
    assert np.array_equal(g[0, k - 3:k + 4, k - 3:k + 4].real, t[O // 2::O, O // 2::O])
    assert g[0, k, k].real == pytest.approx(1.0, abs=1e-6)
    assert abs(g[0]).argmax() == k * N + k


# ----------------------------------------------------------------------------------------- P2
def test_p2_linearity():
    rng = np.random.default_rng(2)
    N, S, O, n = 48, 7, 8, 300
    table = kernels.spheroidal_table(S, O)
    uv = rng.uniform(-15, 15, (n, 2))
    # values exactly representable in float32 so alpha*V1 + beta*V2 is formed without rounding
    v1 = rng.integers(-64, 64, (n, 4, 2)).astype(np.float32)
    v2 = rng.integers(-64, 64, (n, 4, 2)).astype(np.float32)
    w = (rng.integers(1, 8, n) / 4.0).astype(np.float32)
    alpha, beta = 3.0, -0.5
    g1, _, _ = _grid(uv, v1, w, N=N, S=S, O=O, table=table)
    g2, _, _ = _grid(uv, v2, w, N=N, S=S, O=O, table=table)
    g12, _, _ = _grid(uv, (alpha * v1 + beta * v2).astype(np.float32), w, N=N, S=S, O=O, table=table)
    ref = alpha * g1 + beta * g2
    assert np.abs(g12 - ref).max() <= 1e-12 * np.abs(ref).max()


# ----------------------------------------------------------------------------------------- P3
@pytest.mark.parametrize("S,O", [(7, 8), (16, 4)])
def test_p3_total_sum(S, O):
    rng = np.random.default_rng(3)
    N, n = 64, 500
    t1 = kernels.spheroidal_1d(S, O)
    table = np.outer(t1, t1).astype(np.float32)
    uv = rng.uniform(-20, 20, (n, 2))
    vis = _vis(n, rng)
    w = rng.uniform(0.5, 1.5, n).astype(np.float32)
    g, a, st = _grid(uv, vis, w, N=N, S=S, O=O, table=table)
    assert st["n_dropped"] == 0
    # sum of the taps a visibility uses depends on its sub-cell offset: taps are the table samples
    # congruent to (S*O/2 - X) mod O.  (the per-offset sum, not one constant.)
    t64 = table.astype(np.float64)
    X = np.floor((uv[:, 0] + N // 2) * O + 0.5).astype(np.int64)
    Y = np.floor((uv[:, 1] + N // 2) * O + 0.5).astype(np.int64)
    rx = ((S * O) // 2 - X) % O
    ry = ((S * O) // 2 - Y) % O
    sum_c = np.array([t64[ry_::O, rx_::O].sum() for ry_, rx_ in zip(ry, rx)])
    v = vis[..., 0].astype(np.float64) + 1j * vis[..., 1].astype(np.float64)
    exp = (w.astype(np.float64)[:, None] * v * sum_c[:, None]).sum(0)
    got = g.reshape(4, -1).sum(1)
    assert np.abs(got - exp).max() <= 1e-10 * np.abs(exp).max()
    exp_abs = (w.astype(np.float64)[:, None] * np.abs(v) * sum_c[:, None]).sum(0)   # table >= 0 here
    assert np.abs(a.reshape(4, -1).sum(1) - exp_abs).max() <= 1e-10 * exp_abs.max()


# ----------------------------------------------------------------------------------------- P4
@pytest.mark.parametrize("src", [(0.0, 0.0), (2 / 16, -1 / 16), (5 / 16, 3 / 16)])
def test_p4_three_antennas_fft_image_matches_direct_dft(src):
    """3 antennas, 16^2 grid, S=7, O=8: grid -> inverse FFT -> grid correction vs the direct DFT
    of a point source, within 1e-3 of the peak on the inner half of the image; baselines snapped
    to the 1/O lattice (the table lookup is nearest-sub-cell)."""
    N, S, O = 16, 7, 8
    rng = np.random.default_rng(4)
    t1 = kernels.spheroidal_1d(S, O)
    table = np.outer(t1, t1).astype(np.float32)
    ant = np.round(rng.uniform(-2.0, 2.0, (3, 2)) * O) / O
    i, j = np.triu_indices(3, 1)
    uv = ant[j] - ant[i]
    l0, m0 = src                                                     # cycles per cell (du = 1)
    vis_c = np.exp(-2j * np.pi * (uv[:, 0] * l0 + uv[:, 1] * m0))
    vis = np.zeros((3, 4, 2), np.float32)
    vis[:, 0, 0], vis[:, 0, 1] = vis_c.real, vis_c.imag
    g, _, st = _grid(uv, vis, N=N, S=S, O=O, table=table)
    assert st["n_dropped"] == 0
    lk = (np.arange(N) - N // 2) / N                                 # image pixel centres
    # the oracle's imager (row f2) is what is pinned here against the direct DFT
    img_c = oracle.image(g[0], oracle.grid_correction(t1.astype(np.float32), S, O, N))
    v32 = vis[:, 0, 0].astype(np.float64) + 1j * vis[:, 0, 1].astype(np.float64)
    dft = np.zeros((N, N), complex)
    for (u_, v_), vv in zip(uv, v32):
        dft += vv * np.exp(2j * np.pi * (u_ * lk[None, :] + v_ * lk[:, None]))
    inner = slice(N // 4 + 1, 3 * N // 4)
    err = np.abs(img_c - dft)[inner, inner].max() / np.abs(dft).max()
    assert err < 1e-3
    # and the source is where it was put (sign and centre conventions, R9/R10)
    if max(abs(round(l0 * N)), abs(round(m0 * N))) < N // 4:
        peak = np.unravel_index(np.abs(img_c[inner, inner]).argmax(), (N // 2 - 1, N // 2 - 1))
        assert (peak[1] + N // 4 + 1 - N // 2, peak[0] + N // 4 + 1 - N // 2) == (round(l0 * N), round(m0 * N))


def test_p4b_imager_equals_the_centred_inverse_dft_written_out():
    """oracle.image against the O(N^4) definition on a random 8 x 8 plane, with a non-trivial correction."""
    N = 8
    rng = np.random.default_rng(44)
    g = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    corr = rng.uniform(0.5, 2.0, N)
    k = np.arange(N) - N // 2
    want = np.zeros((N, N), complex)
    for y in range(N):
        for x in range(N):
            ph = np.exp(2j * np.pi * (k[None, :] * k[x] + k[:, None] * k[y]) / N)       # [v][u]
            want[y, x] = corr[y] * corr[x] * (g * ph).sum()
    assert np.abs(oracle.image(g, corr) - want).max() < 1e-12 * np.abs(want).max()


# ----------------------------------------------------------------------------------------- P5
@pytest.mark.parametrize("S,O,N", [(7, 8, 32), (16, 4, 48), (6, 2, 24)])
def test_p5_scatter_equals_bruteforce_gather(S, O, N):
    rng = np.random.default_rng(5)
    n = 400
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    half = N / 2
    uv = rng.uniform(-half - 1, half + 1, (n, 2))                     # some fall off the grid
    uv[:40] = np.round(uv[:40] * O) / O                               # exact lattice points
    uv[40:80] = (np.floor(uv[40:80] * O) + 0.5) / O                   # exact rounding ties
    uv[80:90] = np.round(uv[80:90])                                   # cell centres
    uv[90] = (-half + S / 2, -half + S / 2)                           # grid-edge cases
    uv[91] = (half - S / 2 - 1.0 / O, half - S / 2 - 1.0 / O)
    uv[92] = (-half + S / 2 - 1.0 / O, 0.0)
    uv[93] = (0.0, half - S / 2 + 1.0 / O)
    vis = _vis(n, rng)
    w = rng.uniform(0.5, 1.5, n).astype(np.float32)
    g, _, st = _grid(uv, vis, w, N=N, S=S, O=O, table=table)
    ref, n_drop = _gather_bruteforce(uv, vis, w, N, S, O, table)
    assert 0 < n_drop < n and st["n_dropped"] == n_drop
    assert st["vis_taps"] == (n - n_drop) * S * S
    assert np.abs(g - ref).max() <= 1e-12 * np.abs(ref).max()


def test_p5_cell_size_and_frequency_scaling():
    """u_lambda = u_m * f / c and cell = u_lambda / du + N/2."""
    rng = np.random.default_rng(6)
    N, S, O, n = 40, 7, 8, 60
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    du = 2.5
    freqs = np.array([100e6, 150e6, 200e6])
    uvw = np.zeros((2, n, 3))
    uvw[:, :, :2] = rng.uniform(-60, 60, (2, n, 2))                  # metres
    vis = _vis(2 * n * 3, rng)
    g, _, st = oracle.grid_full(uvw, freqs, vis, None, grid_size=N, cell_size=du, oversample=O,
                                support=[S], kernel=table)
    # flatten (t, b, f) -> per-visibility wavelengths, then the same brute force at du
    uvl = (uvw[:, :, None, :2] * (freqs / C)[None, None, :, None]).reshape(-1, 2)
    ref, n_drop = _gather_bruteforce(uvl, vis, None, N, S, O, table, du=du)
    assert st["n_dropped"] == n_drop
    assert np.abs(g - ref).max() <= 1e-12 * np.abs(ref).max()


# ----------------------------------------------------------------------------------------- P6
def test_p6_paper_vis_per_pixel_closed_form(repo_root):
    vals = {}
    for line in (Path(repo_root) / "tests/golden/paper_section5_vis_per_pixel.txt").read_text().splitlines():
        if line and not line.startswith("#"):
            k, v = line.split()
            vals[k] = float(v)
    mean = vals["baselines"] * vals["patch"] ** 2 / vals["image"] ** 2
    assert abs(mean - vals["stated_vis_per_pixel"]) <= vals["stated_tolerance"]      # 59.5 ~ "around 60"
    # the same closed form on the oracle: all-ones table, unit visibilities => every tap adds 1,
    # so the grid total is n*S^2 and the mean per cell n*S^2/N^2
    rng = np.random.default_rng(7)
    N, S, O, n = 96, 24, 2, 2000
    uv = rng.uniform(-N / 2 + S / 2 + 1, N / 2 - S / 2 - 1, (n, 2))
    vis = np.zeros((n, 4, 2), np.float32)
    vis[:, 0, 0] = 1.0
    g, a, st = _grid(uv, vis, N=N, S=S, O=O, table=np.ones((S * O, S * O), np.float32))
    assert st["n_dropped"] == 0 and st["vis_taps"] == n * S * S
    assert g[0].real.sum() == n * S * S and a[0].sum() == n * S * S
    assert g[0].real.mean() == pytest.approx(n * S * S / N ** 2)


# ----------------------------------------------------------------------------------------- P7
@pytest.mark.parametrize("S,O", [(7, 8), (15, 8), (16, 4)])
def test_p7_spheroidal_table_is_the_textbook_function(S, O):
    from scipy.special import pro_ang1
    t1 = kernels.spheroidal_1d(S, O)
    n = S * O
    assert t1[n // 2] == pytest.approx(1.0, abs=1e-12)
    assert np.allclose(t1[1:], t1[1:][::-1], atol=1e-12)             # even about r = 0 (sample n/2)
    assert np.all(np.diff(t1[: n // 2 + 1]) > 0) and np.all(t1 > 0)
    c = np.pi * S / 2
    eta = 2.0 * ((np.arange(n) - n / 2) / O) / S
    inner = np.abs(eta) < 1
    ref = np.array([pro_ang1(0, 0, c, e)[0] for e in eta[inner]]) / pro_ang1(0, 0, c, 0.0)[0]
    assert np.abs(t1[inner] - ref).max() < 1e-6


# --------------------------------------------------------------------- other parts of the definition
def test_windows_are_restrictions_and_thread_count_is_immaterial():
    rng = np.random.default_rng(8)
    N, S, O, n = 64, 7, 8, 800
    table = kernels.spheroidal_table(S, O)
    uv = rng.uniform(-28, 28, (n, 2))
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = uv
    vis = _vis(n, rng)
    kw = dict(grid_size=N, cell_size=1.0, oversample=O, support=[S], kernel=table)
    g1, a1, _ = oracle.grid_full(uvw, [C], vis, None, n_threads=1, **kw)
    g5, a5, _ = oracle.grid_full(uvw, [C], vis, None, n_threads=5, **kw)
    assert np.array_equal(g1, g5) and np.array_equal(a1, a5)
    wins = [(0, 8, 0, 8), (20, 41, 13, 30), (63, 64, 0, 64)]
    res = oracle.grid_windows(uvw, [C], vis, None, wins, **kw)
    for (y0, y1, x0, x1), gw, aw in zip(wins, res["G"], res["A"]):
        assert np.array_equal(gw, g1[:, y0:y1, x0:x1]) and np.array_equal(aw, a1[:, y0:y1, x0:x1])
    # feeding the visibilities in two calls adds up (used for config 4, one integration at a time)
    r1 = oracle.grid_windows(uvw[:, :300], [C], vis[:300], None, wins, **kw)
    r2 = oracle.grid_windows(uvw[:, 300:], [C], vis[300:], None, wins, out=r1, **kw)
    for gw, ga in zip(r2["G"], res["G"]):
        assert np.abs(gw - ga).max() <= 1e-12 * np.abs(ga).max()


def test_weights_multiply_and_zero_weight_contributes_nothing():
    rng = np.random.default_rng(9)
    N, S, O, n = 32, 6, 2, 50
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    uv = rng.uniform(-10, 10, (n, 2))
    vis = _vis(n, rng)
    w = np.ones(n, np.float32)
    w[::2] = 0.0
    g, a, _ = _grid(uv, vis, w, N=N, S=S, O=O, table=table)
    g_odd, a_odd, _ = _grid(uv[1::2], vis[1::2], None, N=N, S=S, O=O, table=table)
    assert np.array_equal(g, g_odd) and np.array_equal(a, a_odd)
    g2, _, _ = _grid(uv, vis, 2.0 * np.ones(n, np.float32), N=N, S=S, O=O, table=table)
    g1, _, _ = _grid(uv, vis, None, N=N, S=S, O=O, table=table)
    assert np.array_equal(g2, 2.0 * g1)


def test_wplanes_variable_support_and_conjugate():
    """Reading R13: plane = min(P-1, floor(|w|/w_max * P)), support per plane, conj table for w<0."""
    rng = np.random.default_rng(10)
    N, O = 64, 4
    supports = [4, 6, 8]
    tabs = [(rng.standard_normal((s * O, s * O)) + 1j * rng.standard_normal((s * O, s * O))).astype(np.complex64)
            for s in supports]
    kernel = np.concatenate([t.view(np.float32).ravel() for t in tabs])
    w_max = 30.0
    kw = dict(N=N, S=supports, O=O, table=kernel, w_max=w_max, kernel_is_complex=True)
    vis = np.zeros((1, 4, 2), np.float32)
    vis[0, 1] = (1.0, 0.0)
    k = N // 2
    for w_l, plane in [(0.0, 0), (9.99, 0), (10.0, 1), (-15.0, 1), (20.0, 2), (30.0, 2), (-45.0, 2)]:
        g, a, st = _grid(np.zeros((1, 2)), vis, w=np.array([w_l]), **kw)
        s = supports[plane]
        exp = tabs[plane][0::O, 0::O].astype(np.complex128)
        if w_l < 0:
            exp = exp.conj()
        assert st["vis_taps"] == s * s
        assert np.array_equal(g[1, k - s // 2:k + s // 2, k - s // 2:k + s // 2], exp)
        assert np.count_nonzero(g) == np.count_nonzero(exp)
        assert np.allclose(a[1, k - s // 2:k + s // 2, k - s // 2:k + s // 2], np.abs(exp), rtol=1e-15)
    # a complex visibility times a complex tap is a complex product
    vis[0, 1] = (0.5, -2.0)
    g, _, _ = _grid(np.zeros((1, 2)), vis, w=np.array([12.0]), **kw)
    s = supports[1]
    exp = (0.5 - 2.0j) * tabs[1][0::O, 0::O].astype(np.complex128)
    assert np.allclose(g[1, k - s // 2:k + s // 2, k - s // 2:k + s // 2], exp, rtol=1e-15)


def test_per_baseline_tables_reduce_to_single_table_gridding():
    """Row f3 (PAPER.md :73, :179 "a unique GCF for each visibility"): with table_index the GCF of a baseline
    is the caller's choice, not |w|'s.  Pin: by linearity the grid equals the sum, over the tables j, of
    gridding the baselines that use j with a single-table problem -- the case P1-P5 pin; an index outside
    the bank drops the baseline; the conjugate is still taken for w < 0."""
    rng = np.random.default_rng(33)
    N, O, nb = 48, 2, 300
    supports = [5, 8, 12, 20]
    tabs = [(rng.standard_normal((s * O, s * O)) + 1j * rng.standard_normal((s * O, s * O))).astype(np.complex64)
            for s in supports]
    kernel = np.concatenate([t.view(np.float32).ravel() for t in tabs])
    uv = rng.uniform(-N / 2 + 1, N / 2 - 1, (nb, 2))
    w = rng.uniform(-5.0, 5.0, nb)
    idx = rng.integers(0, len(supports), nb).astype(np.int32)
    idx[:3] = (-1, len(supports), 99)                              # not in the bank: dropped
    vis, wt = _vis(nb, rng), rng.uniform(0.5, 1.5, nb).astype(np.float32)
    g, a, st = _grid(uv, vis, wt, N=N, S=supports, O=O, table=kernel, w=w, w_max=1.0, kernel_is_complex=True,
                     table_index=idx)
    want, want_a, taps, dropped = np.zeros_like(g), np.zeros_like(a), 0, 3
    for j, s_j in enumerate(supports):
        m = idx == j
        gj, aj, sj = _grid(uv[m], vis[m], wt[m], N=N, S=[s_j], O=O, table=tabs[j].view(np.float32).ravel(), w=w[m],
                           kernel_is_complex=True)
        want += gj; want_a += aj; taps += sj["vis_taps"]; dropped += sj["n_dropped"]
    assert st["vis_taps"] == taps and st["n_dropped"] == dropped
    assert np.abs(g - want).max() <= 1e-12 * np.abs(want).max()
    assert np.abs(a - want_a).max() <= 1e-12 * want_a.max()
    m = oracle.map_visibilities(np.concatenate([uv, w[:, None]], 1)[None], [C], grid_size=N, cell_size=1.0, oversample=O,
                                support=supports, kernel=kernel, kernel_is_complex=True, table_index=idx)
    assert np.array_equal(m[3:, 4] & 0xFF, idx[3:]) and np.array_equal(m[3:, 4] >> 8, (w[3:] < 0).astype(np.int32))
    assert m[:3, 5].all()


def test_map_matches_gather_algebra():
    """oracle.map_visibilities (what the CUDA map kernel is compared with) against the gather view:
    the patch is exactly the set of cells whose centre the table reaches."""
    rng = np.random.default_rng(11)
    N, S, O, n = 128, 15, 8, 3000
    uv = rng.uniform(-70, 70, (n, 2))
    uv[:200] = (np.floor(uv[:200] * O) + 0.5) / O
    uvw = np.zeros((1, n, 3))
    uvw[0, :, :2] = uv
    m = oracle.map_visibilities(uvw, [C], grid_size=N, cell_size=1.0, oversample=O, support=[S],
                                kernel=np.zeros((S * O) ** 2, np.float32))
    X = np.floor((uv + N // 2) * O + 0.5).astype(np.int64)
    for axis, (c0, q) in enumerate([(m[:, 0], m[:, 2]), (m[:, 1], m[:, 3])]):
        c0 = c0.astype(np.int64)
        j0 = c0 * O - X[:, axis] + (S * O) // 2                       # table sample of the first tap
        assert np.array_equal(j0, q) and (q >= 0).all() and (q < O).all()
        assert ((c0 - 1) * O - X[:, axis] + (S * O) // 2 < 0).all()   # the cell before is out of reach
        assert ((c0 + S - 1) * O - X[:, axis] + (S * O) // 2 < S * O).all()   # last tap inside
        assert ((c0 + S) * O - X[:, axis] + (S * O) // 2 >= S * O).all()      # the cell after is not
    off = (m[:, 0] < 0) | (m[:, 0] + S > N) | (m[:, 1] < 0) | (m[:, 1] + S > N)
    assert np.array_equal(off, m[:, 5].astype(bool)) and off.any() and not off.all()
