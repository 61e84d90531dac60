"""Pre-summation in input order (csrc/presum.cu) against the CPU oracle: multi-channel, multi-integration
inputs where neighbouring channels / integrations of a baseline share their lattice point, ragged group
shapes, dropped visibilities, adversarial key sequences, and bit-identical reruns."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import as_complex, assert_parity, oracle_kwargs
from test_gpu_parity import _gridder, _oracle, _run, C

pytestmark = pytest.mark.gpu
PS = {"presum": 1}


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1003_5575_b200 import gridder
    gridder.load_library()
    return torch.device("cuda:0")


def test_presum_config1_full_grid(dev):
    wl = synth.make_workload(1)
    vis = wl.visibilities("cpu").numpy()
    kw = dict(N=wl.grid_size, du=wl.cell_size, O=wl.oversample, S=wl.support[0], table=wl.kernel)
    a, st = _run(dev, wl.uvw, wl.freq, vis, None, tuning=PS, **kw)
    b, _ = _run(dev, wl.uvw, wl.freq, vis, None, tuning=PS, **kw)
    ref, ab, ost = oracle.grid_full(wl.uvw, wl.freq, vis, None, **oracle_kwargs(wl))
    assert 0 < st.n_presum_records < wl.n_vis
    assert st.n_dropped == ost["n_dropped"] == 0 and st.vis_taps == ost["vis_taps"]
    assert np.array_equal(a, b)
    assert_parity(a, ref, ab, "presum config 1")


@pytest.mark.parametrize("nt,nb,nf,band", [(8, 300, 64, 2e-3), (1, 517, 100, 2e-3), (3, 200, 33, 5e-4), (9, 150, 70, 1e-3),
                                           (11, 97, 31, 3e-3), (16, 64, 32, 1e-4), (2, 400, 5, 1e-2)])
def test_presum_ragged_groups_weights_and_drops(dev, nt, nb, nf, band):
    rng = np.random.default_rng(nt * 1000 + nf)
    N, S, O = 256, 16, 4
    table = synth.spheroidal_table(S, O)
    uvw = np.zeros((nt, nb, 3))
    uvw[0, :, :2] = rng.uniform(-112.0, 112.0, (nb, 2))
    rot = 3e-4 * np.arange(nt)[:, None]                               # a slow rotation with the integration
    uvw[:, :, 0] = uvw[0, :, 0] * np.cos(rot) - uvw[0, :, 1] * np.sin(rot)
    uvw[:, :, 1] = uvw[0, :, 0] * np.sin(rot) + uvw[0, :, 1] * np.cos(rot)
    uvw[:, :5, :2] = 0.0                                              # everything of these rows on one point
    freq = C * (1.0 + band * np.arange(nf))
    vis = rng.standard_normal((nt, nb, nf, 4, 2)).astype(np.float32)
    w = rng.uniform(0.0, 1.5, (nt, nb, nf)).astype(np.float32)
    kw = dict(N=N, du=1.0, O=O, S=S, table=table)
    a, st = _run(dev, uvw, freq, vis, w, tuning=PS, **kw)
    a2, _ = _run(dev, uvw, freq, vis, w, tuning=PS, **kw)
    ref, ab, ost = _oracle(uvw, freq, vis, w, **kw)
    assert st.n_presum_records > 0
    assert st.n_dropped == ost["n_dropped"] and st.vis_taps == ost["vis_taps"]
    assert np.array_equal(a, a2)
    assert_parity(a, ref, ab, f"presum {nt}x{nb}x{nf}")
    # the classic per-visibility path agrees within tolerance too
    c, st_c = _run(dev, uvw, freq, vis, w, tuning={"presum": 2}, **kw)
    assert st_c.n_presum_records == 0
    assert_parity(c, ref, ab, "classic")


def test_presum_adversarial_key_sequences(dev):
    """Keys that come back (A B A down the integrations, A B A along the channels), rows identical to their
    neighbours, everything dropped in places: records may split, sums must not change."""
    rng = np.random.default_rng(5)
    N, S, O, nt, nb, nf = 128, 16, 4, 8, 64, 48
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    uvw = np.zeros((nt, nb, 3))
    pts = rng.uniform(-40.0, 40.0, (3, nb, 2))
    pat = [0, 1, 0, 0, 2, 1, 1, 0]                                    # the lattice point of integration t
    for t in range(nt):
        uvw[t, :, :2] = pts[pat[t]]
    uvw[:, 10:20, :2] = 1000.0                                        # always off the grid
    uvw[3, 20:30, :2] = -1000.0                                       # off the grid in one integration only
    freq = np.full(nf, C)
    freq[::3] = C * 1.01                                              # channels alternate between two scales
    freq[7] = C * 40.0                                                # one channel off the grid for most rows
    vis = rng.standard_normal((nt, nb, nf, 4, 2)).astype(np.float32)
    w = rng.uniform(0.5, 1.5, (nt, nb, nf)).astype(np.float32)
    kw = dict(N=N, du=1.0, O=O, S=S, table=table)
    a, st = _run(dev, uvw, freq, vis, w, tuning=PS, **kw)
    ref, ab, ost = _oracle(uvw, freq, vis, w, **kw)
    assert st.n_presum_records > 0 and 0 < st.n_dropped == ost["n_dropped"]
    assert st.vis_taps == ost["vis_taps"]
    assert_parity(a, ref, ab, "presum adversarial")


def test_presum_nothing_to_merge_and_shapes_that_fall_back(dev):
    """Channels at unrelated frequencies: every visibility is its own record.  A larger input that does not
    merge either is handed to the per-visibility path."""
    rng = np.random.default_rng(6)
    N, S, O, nb, nf = 96, 15, 8, 100, 32      # (3 200 visibilities: inside the record capacity of 3n/4 + 1024)
    table = rng.standard_normal((S * O, S * O)).astype(np.float32)
    uvw = np.zeros((1, nb, 3))
    uvw[0, :, :2] = rng.uniform(-N / 2 - 1, N / 2 + 1, (nb, 2))
    freq = C * rng.uniform(0.2, 1.0, nf)
    vis = rng.standard_normal((1, nb, nf, 4, 2)).astype(np.float32)
    kw = dict(N=N, du=1.0, O=O, S=S, table=table)
    a, st = _run(dev, uvw, freq, vis, None, tuning=PS, **kw)
    ref, ab, ost = _oracle(uvw, freq, vis, None, **kw)
    assert st.n_dropped == ost["n_dropped"] > 0
    assert 0.9 * (nb * nf - st.n_dropped) <= st.n_presum_records <= nb * nf - st.n_dropped
    assert_parity(a, ref, ab, "presum, one record per visibility")
    # one channel, random positions, 20 000 visibilities: nothing merges, the plan kernel counts more than
    # 3 n / 4 + 1024 records, and gridder_bin takes the per-visibility path instead (decided from the data)
    nb1 = 20000
    uvw1 = np.zeros((1, nb1, 3))
    uvw1[0, :, :2] = rng.uniform(-N / 2 - 1, N / 2 + 1, (nb1, 2))
    vis1 = rng.standard_normal((1, nb1, 1, 4, 2)).astype(np.float32)
    b, st_b = _run(dev, uvw1, freq[:1], vis1, None, tuning=PS, **kw)
    ref, ab, ost = _oracle(uvw1, freq[:1], vis1, None, **kw)
    assert st_b.n_presum_records == 0 and st_b.n_dropped == ost["n_dropped"] and st_b.vis_taps == ost["vis_taps"]
    assert_parity(b, ref, ab, "nothing merges: per-visibility path")


def test_presum_bin_once_grid_twice_accumulate_and_empty(dev):
    rng = np.random.default_rng(7)
    N, S, O, nt, nb, nf = 64, 16, 4, 4, 50, 40
    table = synth.spheroidal_table(S, O)
    kw = dict(N=N, du=1.0, O=O, S=S, table=table)
    got, st = _run(dev, np.zeros((1, 0, 3)), [C], np.zeros((0, 4, 2), np.float32), None, tuning=PS, **kw)
    assert st.n_vis == 0 and st.n_work_items == 0 and not got.any()
    uvw = np.zeros((nt, nb, 3))
    uvw[:, :, :2] = rng.uniform(-20.0, 20.0, (1, nb, 2))
    freq = C * (1.0 + 1e-3 * np.arange(nf))
    vis = rng.standard_normal((nt, nb, nf, 4, 2)).astype(np.float32)
    w = rng.uniform(0.5, 1.5, (nt, nb, nf)).astype(np.float32)
    ref, ab, _ = _oracle(uvw, freq, vis, w, **kw)
    base = rng.standard_normal((4, N, N, 2)).astype(np.float32)
    got, _ = _run(dev, uvw, freq, vis, w, tuning=PS, accumulate_onto=base, **kw)
    assert_parity(got, ref + as_complex(base), ab + np.abs(as_complex(base)), "presum accumulate")
    g = _gridder(dev, max_vis=nt * nb * nf, tuning=PS, **kw)
    d_uvw, d_f = torch.from_numpy(uvw).to(dev), torch.from_numpy(freq).to(dev)
    d_v, d_w = torch.from_numpy(vis).to(dev), torch.from_numpy(w).to(dev)
    g.bin(d_uvw, d_f)
    o1 = g.grid(d_v, d_w).cpu().numpy()
    o2 = g.grid(d_v, d_w).cpu().numpy()
    o4 = g.grid(2.0 * d_v, d_w).cpu().numpy()
    g.bin(d_uvw, d_f)
    o3 = g.grid(d_v, d_w).cpu().numpy()
    g.destroy()
    assert np.array_equal(o1, o2) and np.array_equal(o1, o3) and np.array_equal(o4, 2.0 * o1)
    assert_parity(o1, ref, ab, "presum, bin once grid twice")


def test_presum_randomised_sweep(dev):
    """40 seeded random multi-channel problems through the pre-summed path: shapes around the 8-row x 32-channel
    group (ragged in both), tiles 4/8/16, chunks down to one batch, table in shared or tensor memory, with and
    without weights, bands from 'every channel on one point' to 'every channel elsewhere'."""
    rng = np.random.default_rng(2025)
    for it in range(40):
        S = int(rng.choice([9, 12, 13, 15, 16]))
        O = int(rng.choice([1, 2, 4])) if S % 2 == 0 else int(rng.choice([2, 4, 8]))
        N = int(rng.choice([48, 64, 96, 130]))
        nt = int(rng.choice([1, 2, 3, 5, 8, 9, 17]))
        nb = int(rng.choice([1, 7, 8, 9, 40, 150]))
        nf = int(rng.choice([1, 2, 31, 32, 33, 64, 100]))
        if nt * nb * nf > 60_000:
            nb = max(1, 60_000 // (nt * nf))
        spread = float(rng.choice([0.4, 3.0, N / 3, N / 2 + 1]))
        band = float(rng.choice([0.0, 1e-4, 2e-3, 3e-2]))
        table = rng.standard_normal((S * O, S * O)).astype(np.float32)
        uvw = np.zeros((nt, nb, 3))
        uvw[0, :, :2] = rng.uniform(-spread, spread, (nb, 2))
        rot = float(rng.choice([0.0, 1e-4, 1e-2])) * np.arange(nt)[:, None]
        uvw[:, :, 0] = uvw[0, :, 0] * np.cos(rot) - uvw[0, :, 1] * np.sin(rot)
        uvw[:, :, 1] = uvw[0, :, 0] * np.sin(rot) + uvw[0, :, 1] * np.cos(rot)
        if rng.random() < 0.3:
            uvw[:, :, :2] = np.round(uvw[:, :, :2] * O) / O
        freq = C * (1.0 + band * np.arange(nf))
        vis = rng.standard_normal((nt, nb, nf, 4, 2)).astype(np.float32)
        w = None if rng.random() < 0.3 else rng.uniform(0.0, 1.5, (nt, nb, nf)).astype(np.float32)
        kw = dict(N=N, du=1.0, O=O, S=S, table=table)
        tuning = {"presum": 1, "tile_log2": int(rng.choice([2, 3, 4])), "chunk": int(rng.choice([32, 64, 100, 256, 4096])),
                  "table_in_tmem": int(rng.choice([1, 2]))}
        got, st = _run(dev, uvw, freq, vis, w, tuning=tuning, **kw)
        ref, ab, ost = _oracle(uvw, freq, vis, w, **kw)
        what = f"sweep case {it}: {nt}x{nb}x{nf} S={S} O={O} N={N} {tuning}"
        assert st.n_dropped == ost["n_dropped"] and st.vis_taps == ost["vis_taps"], what
        assert_parity(got, ref, ab, what)
