"""Benchmark of the gridder hot path (map + bin + grid + flush) on the seeded synthetic arrays.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

One "step" is one pass of the whole hot path (gridder_bin + gridder_grid: SURVEY.md section 8(a)
rows a1-a5) over one synthetic cadence of BASELINE.json config C (default 4: 512 antennas, 768
channels, 8 integrations -- the configuration the metric "512-tile 8 s cadence time" is quoted on).
Prints ONE JSON line (rank 0).  Contract and field meanings: DESIGN.md section 8.

  value      visibility-taps gridded per second, whole job, inputs resident in HBM
  e2e        the same through gridder_run_host: pinned HOST buffers, H2D and D2H inside the timing
  roofline   the grid kernel's FP32-FMA rate (16 flop per visibility-tap) from CUDA events recorded
             around it inside the library on the launching stream, against the FMA-pipe peak
  cpu_baseline  the oracle as it stands, timed on this box's host cores on a bounded sample

Under torchrun (N > 1) every rank grids its own cadence (its own 30.72 MHz band, the paper's
channel decomposition, PAPER.md :108-120): no data-path collective, "scaling": "weak".
`--impl reference` times the oracle only (rank 0), none of the CUDA library is loaded.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "visibility_taps_gridded_per_s"
UNIT = "vis*taps/s"
FLOP_PER_VIS_TAP = 16            # 4 pol x complex x (mul + add), real GCF table
FP32_LANES_PER_SM = 128          # guide: 4 SMSP x 32 lanes, one FFMA per lane per clock
BAND_HZ = 768 * 40.0e3           # one rank's band; rank r starts at 140 MHz + r * BAND_HZ
# dram__bytes_read.sum + dram__bytes_write.sum of one grid_kernel launch from the committed
# `ncu --set full` capture (profiles/), keyed by config; None until a capture exists for it.
NCU_GRID_KERNEL_TRAFFIC_BYTES = {
    4: 4_177_715_000,     # profiles/r01f_grid_kernel_on_records_config4_ncu_full.csv: 1.763335 GB read + 2.414380 GB written
    2: 3_500_273_000,     # profiles/r01f_grid_kernel_on_records_config2_ncu_full.csv: 1.150321 GB read + 2.349952 GB written
}
# the same for reduce_kernel (dense plans: it is the longest kernel of the step there)
NCU_REDUCE_KERNEL_TRAFFIC_BYTES = {
    4: 50_401_785_000,    # profiles/r01f_reduce_kernel_config4_ncu_full.csv: 48.661029 GB read + 1.740756 GB written
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config id (default: the metric's)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (development only)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle leg (development only)")
    ap.add_argument("--no-unmerged", action="store_true", help="skip the merging-off leg (development only)")
    ap.add_argument("--mfs", action="store_true",
                    help="row f4: with N > 1 ranks also sum the per-rank grids inside every timed step "
                         "(deterministic all-to-all + FP64 sum + all-gather); default: no collective")
    ap.add_argument("--atomic", action="store_true",
                    help="also time the atomic-scatter gridder (SURVEY row f1) once on the same workload")
    return ap.parse_args()


def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return json.loads(p.read_text())
        except Exception:
            pass
    return {}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons of one GPU while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------------------------
# The oracle leg: cpu_baseline of our arm, and the whole of `--impl reference`.
# --------------------------------------------------------------------------------------------
class OracleSample:
    """A bounded sample of config `cfg` for the CPU oracle: the first n_time integrations and the
    first n_chan channels of every baseline."""

    def __init__(self, cfg: int, n_time: int, n_chan: int):
        import numpy as np
        import synth
        self.wl = synth.make_workload(cfg, n_time=n_time, n_chan=n_chan)
        self.vis = self.wl.visibilities("cpu").numpy()
        w = self.wl.weights("cpu")
        self.weight = None if w is None else np.ascontiguousarray(w.numpy())
        self.n_time, self.n_chan = n_time, n_chan

    def run(self):
        """One timed oracle gridding (wall clock of the gridding call only) -> (vis_taps, seconds, threads)."""
        import oracle
        wl = self.wl
        t0 = time.perf_counter()
        _, _, st = oracle.grid_full(wl.uvw, wl.freq, self.vis, self.weight, grid_size=wl.grid_size,
                                    cell_size=wl.cell_size, oversample=wl.oversample, support=wl.support,
                                    kernel=wl.kernel, w_max=wl.w_max, kernel_is_complex=wl.kernel_is_complex,
                                    want_abs=False)
        return st["vis_taps"], time.perf_counter() - t0, st["threads"]

    def describe(self) -> str:
        wl = self.wl
        return (f"config {wl.cfg}: integrations 0..{self.n_time - 1}, channels 0..{self.n_chan - 1}, all "
                f"{wl.n_baseline} baselines ({wl.n_vis} visibilities), {wl.grid_size}^2 grid, "
                f"double-precision direct scatter")


def sized_oracle_sample(cfg: int, target_s: float) -> OracleSample:
    """Pick the channel (then integration) count so one oracle run takes about target_s on this box."""
    import synth
    shape = synth.config_shape(cfg)
    full_chan, full_time = shape["n_chan"], shape["n_time"]
    probe_chan = min(full_chan, 2)
    probe = OracleSample(cfg, 1, probe_chan)
    probe.run()                                   # page in the library and the grids
    _, dt, _ = probe.run()
    per_chan = max(dt / probe_chan, 1e-5)
    n_chan = int(max(1, min(full_chan, round(target_s / per_chan))))
    n_time = 1
    if n_chan == full_chan:
        n_time = int(max(1, min(full_time, round(target_s / (per_chan * full_chan)))))
    if (n_time, n_chan) == (1, probe_chan):
        return probe
    return OracleSample(cfg, n_time, n_chan)


def cpu_baseline(cfg: int, target_s: float) -> dict:
    s = sized_oracle_sample(cfg, target_s)
    taps, dt, threads = s.run()
    return {"value": taps / dt, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": s.describe(),
            "seconds": dt}


def run_reference(args) -> dict:
    """`--impl reference`: the oracle, as it stands, on this box's host cores (rank 0 only)."""
    import oracle
    oracle.build()
    n_runs = args.steps + args.warmup
    per_step = max(1.0, min(args.cpu_seconds, 150.0 / max(1, n_runs)))
    s = sized_oracle_sample(args.config, per_step)
    for _ in range(args.warmup):
        s.run()
    taps, secs, threads = 0, 0.0, 0
    for _ in range(args.steps):
        t, dt, threads = s.run()
        taps += t
        secs += dt
    value = taps / secs if secs > 0 else 0.0
    wl = s.wl
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config{wl.cfg}", "sample": s.describe(), "n_vis_per_step": wl.n_vis,
                   "grid": wl.grid_size, "support": max(wl.support), "oversample": wl.oversample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": s.describe()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


# --------------------------------------------------------------------------------------------
# Our arm: the CUDA library through the thin binding, one process per GPU.
# --------------------------------------------------------------------------------------------
def shard_plan(world: int, rank: int) -> dict:
    """Which part of the job a rank owns: its own band (channel block), nothing shared."""
    if not (0 <= rank < world):
        raise ValueError("rank outside the world")
    return {"band": rank, "f0_hz": 140.0e6 + rank * BAND_HZ, "collective": None}


def aggregate(per_rank_ms, per_rank_units, steps: int) -> dict:
    """Whole-job figures from per-rank device times and per-rank units per step (max over ranks)."""
    ms = max(per_rank_ms)
    units = sum(per_rank_units) * steps
    return {"ms_total": ms, "ms_per_step": ms / max(1, steps), "value": units / (ms * 1e-3) if ms > 0 else 0.0}


def _host_budget_bytes(world: int) -> int:
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 64 << 30
    return int(0.6 * avail / max(1, world))


def run_ours(args) -> dict | None:
    import numpy as np
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the gridder has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    from paper_1003_5575_b200 import gridder
    gridder.load_library()                       # fails loudly if libgridder.so is missing
    import synth

    shard = shard_plan(world, rank)
    wl = synth.make_workload(args.config, band=shard["band"])
    nt, nb, nf, n = wl.n_time, wl.n_baseline, wl.n_chan, wl.n_vis
    vis = torch.empty((nt, nb, nf, 4, 2), dtype=torch.float32, device=dev)
    weight = torch.empty((nt, nb, nf), dtype=torch.float32, device=dev) if wl.random_weights else None
    for t in range(nt):
        vis[t] = wl.vis_block(t, dev)
        if weight is not None:
            weight[t] = wl.weight_block(t, dev)
    d_uvw = torch.from_numpy(wl.uvw).to(dev)
    d_freq = torch.from_numpy(wl.freq).to(dev)
    g = gridder.Gridder(grid_size=wl.grid_size, cell_size=wl.cell_size, oversample=wl.oversample,
                        support=wl.support, kernel=torch.from_numpy(wl.kernel).to(dev), max_vis=n,
                        n_wplanes=wl.n_wplanes, w_max=wl.w_max, kernel_is_complex=wl.kernel_is_complex)
    grid = torch.empty((4, wl.grid_size, wl.grid_size, 2), dtype=torch.float32, device=dev)

    mfs_on = bool(args.mfs and world > 1)
    if mfs_on:
        from paper_1003_5575_b200 import mfs

    def step():
        g.bin(d_uvw, d_freq)
        g.grid(vis, weight, out=grid)
        if mfs_on:
            mfs.reduce_grids(grid)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    st = g.stats()
    g.set_profiling(True)
    launches0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_rank = e0.elapsed_time(e1)
    stage = g.stage_ms()
    st_exec = g.stats()                   # records gridded / FMAs executed by the last gridder_grid
    launches = g.launch_count() - launches0 + (args.steps if mfs_on else 0)      # + gridder_sum_parts per step
    g.set_profiling(False)
    checksum = float(grid[0, wl.grid_size // 2, wl.grid_size // 2, 0].item())

    def gather(x: float):
        if world == 1:
            return [x]
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        out = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(out, t)
        return [float(o.item()) for o in out]

    agg = aggregate(gather(ms_rank), gather(float(st.vis_taps)), args.steps)

    # ---- end to end: pinned host buffers through gridder_run_host ---------------------------
    e2e = None
    if not args.no_e2e:
        per_t = nb * nf * (32 + (4 if weight is not None else 0))
        nt_e = int(max(1, min(nt, _host_budget_bytes(world) // max(1, per_t))))
        h_vis = torch.empty((nt_e, nb, nf, 4, 2), dtype=torch.float32, pin_memory=True)
        h_vis.copy_(vis[:nt_e])
        h_w = None
        if weight is not None:
            h_w = torch.empty((nt_e, nb, nf), dtype=torch.float32, pin_memory=True)
            h_w.copy_(weight[:nt_e])
        h_uvw = torch.from_numpy(np.ascontiguousarray(wl.uvw[:nt_e])).pin_memory()
        h_freq = torch.from_numpy(wl.freq).pin_memory()
        h_grid = torch.empty(grid.shape, dtype=torch.float32, pin_memory=True)
        staging = {"uvw": d_uvw, "freq": d_freq, "vis": vis, "weight": weight, "grid": grid}
        e_steps = max(1, min(args.steps, 3))
        g.run_host(h_uvw, h_freq, h_vis, h_w, h_grid, staging)            # warm-up
        taps_e = st.vis_taps * nt_e // nt        # (run_host grids in slices; the plan's stats are the last slice's)
        barrier()
        e0.record()
        for _ in range(e_steps):
            g.run_host(h_uvw, h_freq, h_vis, h_w, h_grid, staging)
        e1.record()
        barrier()
        agg_e = aggregate(gather(e0.elapsed_time(e1)), gather(float(taps_e)), e_steps)
        h2d = h_vis.numel() * 4 + (h_w.numel() * 4 if h_w is not None else 0) + h_uvw.numel() * 8 + h_freq.numel() * 8
        e2e = {"value": agg_e["value"], "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(h_grid.numel() * 4), "ms_per_step": agg_e["ms_per_step"],
               "steps": e_steps, "n_time": nt_e, "result_checksum": float(h_grid[0, wl.grid_size // 2, wl.grid_size // 2, 0])}
        del h_vis, h_w, h_grid
    f1 = None
    if args.atomic:
        # row f1: per-visibility FP32 atomic scatter, same inputs, one warm-up and one timed pass
        g.scatter_atomic(d_uvw, d_freq, vis, weight, out=grid)
        barrier()
        e0.record()
        g.scatter_atomic(d_uvw, d_freq, vis, weight, out=grid)
        e1.record()
        barrier()
        ms_f1 = e0.elapsed_time(e1)
        f1 = {"ms": ms_f1, "value": st.vis_taps / (ms_f1 * 1e-3), "unit": UNIT,
              "note": "gridder_scatter_atomic: no binning, red.global.add.v2.f32 per (tap, pol); not deterministic"}
    g.destroy()
    # the same kernel with merging off: every entry gridded on its own (what per-visibility GCFs would need)
    unmerged = None
    if world == 1 and not args.no_unmerged:
        g.workspace = None                        # (the first plan's workspace goes back to the allocator)
        torch.cuda.empty_cache()
        g2 = gridder.Gridder(grid_size=wl.grid_size, cell_size=wl.cell_size, oversample=wl.oversample,
                             support=wl.support, kernel=torch.from_numpy(wl.kernel).to(dev), max_vis=n,
                             n_wplanes=wl.n_wplanes, w_max=wl.w_max, kernel_is_complex=wl.kernel_is_complex,
                             tuning={"merge": 2})
        g2.bin(d_uvw, d_freq)
        g2.grid(vis, weight, out=grid)
        torch.cuda.synchronize()
        g2.set_profiling(True)
        for _ in range(2):
            g2.grid(vis, weight, out=grid)
        torch.cuda.synchronize()
        st2, stage2 = g2.stats(), g2.stage_ms()
        g2.destroy()
        unmerged = {"grid_kernel_ms": stage2["grid"], "fma_executed": st2.fma_executed,
                    "records_gridded": st2.n_records_gridded}
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return None

    # ---- roofline of the dominant kernel (the grid kernel) ----------------------------------
    peaks = measured_peaks()
    props = torch.cuda.get_device_properties(dev)
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    fma_peak_tf = props.multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    flop_per_tap = FLOP_PER_VIS_TAP * (2 if wl.kernel_is_complex else 1)
    grid_ms = stage["grid"]
    # The grid kernel sums entries with equal patch origin and table offset before gridding them
    # (exact by linearity), so it executes fewer FMAs than 8 per visibility-tap.  The roofline
    # fraction is claimed on the FMAs it EXECUTED (gridder_get_stats: records x padded patch cells x
    # 8 or 16); the nominal rate (16 flop per visibility-tap gridded) is given beside it.
    alg_bytes = n * (32 + (4 if weight is not None else 0)) + nt * nb * 24 + nf * 8 + 32 * wl.grid_size ** 2
    exec_flop = 2.0 * st_exec.fma_executed
    achieved_tf = exec_flop / (grid_ms * 1e-3) / 1e12 if grid_ms > 0 else 0.0
    nominal_tf = flop_per_tap * st.vis_taps / (grid_ms * 1e-3) / 1e12 if grid_ms > 0 else 0.0
    roofline = {
        "bound": "alu", "kernel": "grid_kernel", "achieved": achieved_tf, "peak": fma_peak_tf, "unit": "TFLOP/s",
        "frac": achieved_tf / fma_peak_tf if fma_peak_tf else None,
        "traffic": NCU_GRID_KERNEL_TRAFFIC_BYTES.get(args.config),
        "peak_source": f"derived: {props.multi_processor_count} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x "
                       f"{sm_max_mhz:.0f} MHz (clocks.max.sm); DESIGN.md section 7",
        "kernel_ms": grid_ms, "kernel_share_of_step": grid_ms / agg["ms_per_step"] if agg["ms_per_step"] else None,
        "flop_per_launch": exec_flop, "records_gridded": st_exec.n_records_gridded,
        "merge_factor": st.n_entries / st_exec.n_records_gridded if st_exec.n_records_gridded else None,
        "nominal": {"tflops": nominal_tf, "frac": nominal_tf / fma_peak_tf if fma_peak_tf else None,
                    "flop_per_launch": flop_per_tap * st.vis_taps,
                    "note": "16 (32) flop per visibility-tap gridded; above 1 is possible because of the merging"},
        "frac_at_sampled_clock": (achieved_tf / (fma_peak_tf * clocks["sm_mhz"] / sm_max_mhz)
                                  if clocks.get("sm_mhz") else None),
        "hbm": {"algorithmic_bytes_per_step": int(alg_bytes),
                "gbs_at_step_time": alg_bytes / (agg["ms_per_step"] * 1e-3) / 1e9 if agg["ms_per_step"] else None,
                "peak_gbs": peaks.get("hbm_gbs", 6650.0),
                "peak_source": "MEASURED_PEAKS.json" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md)"},
    }
    reduce_ms = stage.get("reduce", 0.0)
    if reduce_ms > grid_ms:
        # Dense plan: the pre-summation (reduce_kernel) is the longest kernel.  It streams every sorted
        # (key, index) pair, gathers the visibility (and weight) it names, and writes the records:
        # HBM-bound.  Algorithmic bytes per launch: 8 + 32 (+ 4) per entry, 36 per record.
        red_bytes = st.n_entries * (8 + 32 + (4 if weight is not None else 0)) + st_exec.n_records_gridded * 36
        gbs = red_bytes / (reduce_ms * 1e-3) / 1e9
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        roofline = {
            "bound": "hbm", "kernel": "reduce_kernel", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
            "frac": gbs / hbm_peak, "traffic": NCU_REDUCE_KERNEL_TRAFFIC_BYTES.get(args.config),
            "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy bandwidth)" if "hbm_gbs" in peaks
                           else "fallback (B200_PROFILING.md)",
            "kernel_ms": reduce_ms, "kernel_share_of_step": reduce_ms / agg["ms_per_step"] if agg["ms_per_step"] else None,
            "bytes_per_launch": int(red_bytes), "entries": st.n_entries, "records": st_exec.n_records_gridded,
            "merge_factor": roofline["merge_factor"],
            "grid_kernel": roofline,              # the second kernel of the stage, on the records: FP32-FMA bound
            "hbm": roofline["hbm"],
        }
    out = {
        "metric": METRIC, "value": agg["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": agg["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{wl.cfg}", "n_antennas": wl.n_ant, "n_baselines": nb, "n_chan": nf,
                   "n_time": nt, "n_vis_per_gpu": n, "grid": wl.grid_size, "support": max(wl.support),
                   "oversample": wl.oversample, "n_wplanes": wl.n_wplanes, "weights": weight is not None,
                   "parallelism": (f"channel-block x{world} + grid sum (all-to-all, FP64 fixed-order sum, all-gather)"
                                   if mfs_on else f"channel-block x{world} (no collective)"),
                   "l2": "inputs per step exceed the 126 MB L2" if n * 32 > (126 << 20) else "L2-resident inputs",
                   "tile": st.tile_size, "chunk": st.chunk_size, "work_items": st.n_work_items,
                   "grid_warps_per_sm": st.grid_warps_per_sm},
        "gflops": flop_per_tap * agg["value"] / 1e9,
        "stage_ms": stage, "grid_only_ms": stage["grid"] + stage["flush"] + stage.get("reduce", 0.0) + stage.get("presum", 0.0),     # gridder_grid alone (a bin serves many)
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
        "cadence_budget_s": 8.0, "result_checksum": checksum,
    }
    if unmerged is not None and unmerged["grid_kernel_ms"] > 0:
        tf = 2.0 * unmerged["fma_executed"] / (unmerged["grid_kernel_ms"] * 1e-3) / 1e12
        unmerged.update({"achieved": tf, "frac": tf / fma_peak_tf, "unit": "TFLOP/s",
                         "note": "GRIDDER_MERGE=0: every entry gridded on its own, same kernel"})
        out["roofline"]["without_merging"] = unmerged
    if f1 is not None:
        out["f1_atomic_scatter"] = f1
    if e2e is not None:
        out["e2e"] = e2e
    if world == 1 and not args.no_cpu:
        import oracle
        oracle.build()
        out["cpu_baseline"] = cpu_baseline(args.config, args.cpu_seconds)
    return out


def main():
    args = parse_args()
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        print(json.dumps(run_reference(args)), flush=True)
        return
    out = run_ours(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
