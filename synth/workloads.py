"""The five seeded synthetic array workloads of BASELINE.json (``configs[0..4]``).

Shapes follow PAPER.md Table 1 (:47-55: 512 tiles, 130 816 baselines, 768 x 40 kHz channels),
4 polarisations (:45) and the 8 s cadence (:11, :59).  The MWA data the paper measured on is not
public, so these stand in for it.  Every reading of an under-specified config item is listed in
DESIGN.md ("Input recipe"); the seeds are ``10035575 + config``.

Nothing here maps uvw to cells or touches a grid: this module only makes the arrays that the
oracle and the CUDA library are both given.  Small pieces (antennas, uvw, frequencies, tables)
are numpy on the host; visibilities and weights are made per integration with torch on the
device asked for (CPU for configs 0-1, the GPU for the 10^8-10^9 sample configs) so both paths
read identical bytes.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

from . import kernels

C_M_PER_S = 299_792_458.0
SIDEREAL_DAY_S = 86164.0905
LATITUDE_DEG = -26.7033
SEED0 = 10035575
CONFIG_IDS = (0, 1, 2, 3, 4)

_SPEC = {
    #      n_ant  n_chan  n_time dt_s  N     S    O  f0_hz    df_hz   wplanes
    0: dict(n_ant=32, n_chan=1, n_time=8, dt=8.0, grid=256, support=7, oversample=8,
            f0=150.0e6, df=0.0, wplanes=1),
    1: dict(n_ant=128, n_chan=32, n_time=8, dt=8.0, grid=1024, support=15, oversample=8,
            f0=140.0e6, df=40.0e3, wplanes=1),
    2: dict(n_ant=512, n_chan=768, n_time=1, dt=8.0, grid=4096, support=16, oversample=4,
            f0=140.0e6, df=40.0e3, wplanes=1),
    3: dict(n_ant=512, n_chan=768, n_time=1, dt=8.0, grid=4096, support=None, oversample=4,
            f0=140.0e6, df=40.0e3, wplanes=32),
    4: dict(n_ant=512, n_chan=768, n_time=8, dt=1.0, grid=4096, support=16, oversample=4,
            f0=140.0e6, df=40.0e3, wplanes=1),
}


def _antennas(cfg: int, rng: np.random.Generator, n_ant: int) -> np.ndarray:
    """East/North positions in metres ("1.5 km disk" read as a 1.5 km *diameter*)."""
    if cfg == 0:
        r = 750.0 * np.sqrt(rng.random(n_ant))
    elif cfg == 1:
        n_core = round(0.2 * n_ant)
        r = np.concatenate([750.0 * np.sqrt(rng.random(n_ant - n_core)),
                            50.0 * np.sqrt(rng.random(n_core))])
    else:
        # surface density ~ r^-1.5  =>  N(<r) ~ sqrt(r); half of the antennas inside 150 m
        half = n_ant // 2
        u = rng.random(n_ant)
        r = np.empty(n_ant)
        r[:half] = 150.0 * u[:half] ** 2
        r[half:] = (np.sqrt(150.0) + u[half:] * (np.sqrt(750.0) - np.sqrt(150.0))) ** 2
    th = 2.0 * np.pi * rng.random(n_ant)
    return np.stack([r * np.cos(th), r * np.sin(th)], axis=1)


def _uvw(enu: np.ndarray, hour_angles: np.ndarray, dec: float) -> np.ndarray:
    """Baseline vectors (u, v, w) in metres, [n_time][n_baseline][3]; textbook rotation (ref [6])."""
    lat = np.deg2rad(LATITUDE_DEG)
    east, north = enu[:, 0], enu[:, 1]
    x, y, z = -np.sin(lat) * north, east, np.cos(lat) * north
    i, j = np.triu_indices(enu.shape[0], 1)
    lx, ly, lz = x[j] - x[i], y[j] - y[i], z[j] - z[i]
    out = np.empty((hour_angles.size, i.size, 3))
    for t, h in enumerate(hour_angles):
        sh, ch, sd, cd = np.sin(h), np.cos(h), np.sin(dec), np.cos(dec)
        out[t, :, 0] = sh * lx + ch * ly
        out[t, :, 1] = -sd * ch * lx + sd * sh * ly + cd * lz
        out[t, :, 2] = cd * ch * lx - cd * sh * ly + sd * lz
    return out


@dataclass
class Workload:
    cfg: int
    name: str
    n_ant: int
    n_time: int
    n_baseline: int
    n_chan: int
    grid_size: int
    oversample: int
    support: list            # taps per axis, one entry per w-plane
    n_wplanes: int
    w_max: float             # wavelengths (1.0 when there is a single plane)
    kernel_is_complex: bool
    cell_size: float         # wavelengths per cell
    uvw: np.ndarray          # float64 [n_time][n_baseline][3], metres
    freq: np.ndarray         # float64 [n_chan], Hz
    kernel: np.ndarray       # float32, plane-major, plane p is [S_p*O][S_p*O] (x2 if complex)
    src_l: np.ndarray = field(repr=False, default=None)
    src_m: np.ndarray = field(repr=False, default=None)
    src_flux: np.ndarray = field(repr=False, default=None)
    noise_sigma: float = 0.1
    random_weights: bool = False
    w_term: bool = False
    band: int = 0

    @property
    def n_vis(self) -> int:
        return self.n_time * self.n_baseline * self.n_chan

    # -- per-integration sample blocks -------------------------------------------------------
    def vis_block(self, t: int, device="cpu", baseline_chunk: int = 16384) -> torch.Tensor:
        """float32 [n_baseline][n_chan][4][2] for integration ``t`` (pol order XX, XY, YX, YY).

        XX = YY = sum_s S_s exp(-2 pi i (u l_s + v m_s [+ w (n_s - 1)])), XY = YX = 0, then
        independent N(0, sigma) noise on each of the 8 real components; phases in float64.
        """
        dev = torch.device(device)
        gen = torch.Generator(device=dev)
        gen.manual_seed((SEED0 + self.cfg) * 1000 + 17 * t + 1 + 100003 * self.band)
        out = torch.empty((self.n_baseline, self.n_chan, 4, 2), dtype=torch.float32, device=dev)
        scale = torch.as_tensor(self.freq / C_M_PER_S, dtype=torch.float64, device=dev)
        uvw_t = torch.as_tensor(self.uvw[t], dtype=torch.float64, device=dev)
        l = torch.as_tensor(self.src_l, dtype=torch.float64, device=dev)
        m = torch.as_tensor(self.src_m, dtype=torch.float64, device=dev)
        flux = torch.as_tensor(self.src_flux, dtype=torch.float64, device=dev)
        nm1 = torch.sqrt(1.0 - l * l - m * m) - 1.0 if self.w_term else torch.zeros_like(l)
        for b0 in range(0, self.n_baseline, baseline_chunk):
            b1 = min(self.n_baseline, b0 + baseline_chunk)
            u, v, w = uvw_t[b0:b1, 0], uvw_t[b0:b1, 1], uvw_t[b0:b1, 2]
            re = torch.zeros((b1 - b0, self.n_chan), dtype=torch.float64, device=dev)
            im = torch.zeros_like(re)
            for s in range(l.numel()):
                metres = u * l[s] + v * m[s] + w * nm1[s]
                ph = (-2.0 * np.pi) * metres[:, None] * scale[None, :]
                re += flux[s] * torch.cos(ph)
                im += flux[s] * torch.sin(ph)
            blk = out[b0:b1]
            blk.normal_(0.0, self.noise_sigma, generator=gen)
            blk[:, :, 0, 0] += re.float()
            blk[:, :, 0, 1] += im.float()
            blk[:, :, 3, 0] += re.float()
            blk[:, :, 3, 1] += im.float()
        return out

    def weight_block(self, t: int, device="cpu"):
        """float32 [n_baseline][n_chan], or None for unit weights (configs 0-3)."""
        if not self.random_weights:
            return None
        dev = torch.device(device)
        gen = torch.Generator(device=dev)
        gen.manual_seed((SEED0 + self.cfg) * 1000 + 17 * t + 2 + 100003 * self.band)
        w = torch.empty((self.n_baseline, self.n_chan), dtype=torch.float32, device=dev)
        w.normal_(1.0, 0.25, generator=gen)
        return w.clamp_(0.5, 1.5)

    def visibilities(self, device="cpu") -> torch.Tensor:
        """float32 [n_time][n_baseline][n_chan][4][2] (all integrations)."""
        return torch.stack([self.vis_block(t, device) for t in range(self.n_time)])

    def weights(self, device="cpu"):
        if not self.random_weights:
            return None
        return torch.stack([self.weight_block(t, device) for t in range(self.n_time)])


def config_shape(cfg: int) -> dict:
    """The full sizes of config ``cfg``: n_ant, n_baseline, n_chan, n_time, grid, oversample, wplanes."""
    sp = dict(_SPEC[cfg])
    sp["n_baseline"] = sp["n_ant"] * (sp["n_ant"] - 1) // 2
    return sp


def make_workload(cfg: int, n_time: int | None = None, n_chan: int | None = None, band: int = 0, n_bands: int = 1) -> Workload:
    """Build config ``cfg``.  ``n_time`` / ``n_chan`` may shrink the sample axes (bounded CPU
    samples of the same workload); geometry, cell size and tables stay those of the full config.
    ``band`` > 0 moves the whole band up by ``band`` bandwidths (another GPU's channel block in the
    paper's channel decomposition, PAPER.md :112-118).  ``n_bands`` is the number of bands of the whole job: the
    cell size is fitted to the top of the highest one, so that all ranks of a channel-sharded job grid onto the
    SAME uv cells and their grids may be summed (multi-frequency synthesis)."""
    sp = _SPEC[cfg]
    rng = np.random.default_rng(SEED0 + cfg)
    enu = _antennas(cfg, rng, sp["n_ant"])
    lat = np.deg2rad(LATITUDE_DEG)
    dec = lat + np.deg2rad(30.0) if cfg == 3 else np.deg2rad(-27.0)
    hours = np.arange(sp["n_time"]) * sp["dt"] * 2.0 * np.pi / SIDEREAL_DAY_S
    uvw = _uvw(enu, hours, dec)
    freq = sp["f0"] + band * sp["n_chan"] * sp["df"] + sp["df"] * np.arange(sp["n_chan"], dtype=np.float64)
    o = sp["oversample"]
    if sp["wplanes"] > 1:
        support = kernels.wplane_supports(sp["wplanes"])
        table = kernels.wplane_tables(support, o)
        w_max = float(np.abs(uvw[:, :, 2]).max() * freq.max() / C_M_PER_S)
        is_complex = True
    else:
        support = [sp["support"]]
        table = kernels.spheroidal_table(sp["support"], o).ravel()
        w_max, is_complex = 1.0, False
    # fit-to-grid cell size: no visibility of the full config is dropped
    top = sp["f0"] + (max(n_bands, band + 1) * sp["n_chan"] - 1) * sp["df"] if sp["n_chan"] > 1 else freq.max()
    max_uv = float(np.abs(uvw[:, :, :2]).max() * max(top, freq.max()) / C_M_PER_S)
    n = sp["grid"]
    cell = max_uv / (n / 2 - max(support) / 2 - 2)
    # 20 sources, dN/dS ~ S^-2 on [0.1, 10] Jy, (l, m) uniform in (-0.3, 0.3)
    src_u = rng.random(20)
    flux = 1.0 / (10.0 - 9.9 * src_u)
    src_l = rng.uniform(-0.3, 0.3, 20)
    src_m = rng.uniform(-0.3, 0.3, 20)
    nt = sp["n_time"] if n_time is None else int(n_time)
    nc = sp["n_chan"] if n_chan is None else int(n_chan)
    return Workload(
        cfg=cfg, name=f"config{cfg}", n_ant=sp["n_ant"], n_time=nt, n_baseline=uvw.shape[1],
        n_chan=nc, grid_size=n, oversample=o, support=support, n_wplanes=sp["wplanes"],
        w_max=w_max, kernel_is_complex=is_complex, cell_size=cell,
        uvw=np.ascontiguousarray(uvw[:nt]), freq=np.ascontiguousarray(freq[:nc]),
        kernel=np.ascontiguousarray(table, dtype=np.float32),
        src_l=src_l, src_m=src_m, src_flux=flux, random_weights=(cfg == 4), w_term=(cfg == 3), band=band)
