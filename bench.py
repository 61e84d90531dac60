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
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures of this round
# (profiles/r02_kernels_config4_ncu_full.csv; historical, i.e. not measured by this run), keyed by kernel and config.
NCU_TRAFFIC_BYTES = {
    # profiles/r02_kernels_config4_ncu_full.csv
    ("presum_kernel", 4): 32_686_298_000,      # 29.923058 GB read + 2.763240 GB written
    ("grid_kernel", 4): 6_077_384_000,         # 3.773518 GB read + 2.303866 GB written
    ("presum_plan_kernel", 4): 1_299_012_000,  # 0.116209 GB read + 1.182803 GB written
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
    ap.add_argument("--no-per-config", action="store_true", help="skip the compact legs on configs 0-3 (development only)")
    ap.add_argument("--spawn-check", action="store_true",
                    help="host-logic check of the launcher (tests): every rank joins a gloo group and reports its "
                         "shard, rank 0 prints one JSON line; no GPU work")
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

    def run(self, n_threads: int = 0):
        """One timed oracle gridding (wall clock of the gridding call only) -> (vis_taps, seconds, threads)."""
        import oracle
        wl = self.wl
        t0 = time.perf_counter()
        _, _, st = oracle.grid_full(wl.uvw, wl.freq, self.vis, self.weight, grid_size=wl.grid_size,
                                    cell_size=wl.cell_size, oversample=wl.oversample, support=wl.support,
                                    kernel=wl.kernel, w_max=wl.w_max, kernel_is_complex=wl.kernel_is_complex,
                                    want_abs=False, n_threads=n_threads)
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


def _self_spawn(args) -> int:
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves (torchrun's own module, one
    process per GPU, rendezvous on 127.0.0.1) and hand its exit code back.  NCCL's communicator lines stay on."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve())] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    return subprocess.call(cmd, env=env)


def spawn_check(args) -> dict | None:
    """What every rank of a launched job does before any GPU work, on gloo: join the group, exchange shard plans."""
    import torch
    import torch.distributed as dist
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    mine = torch.tensor([float(shard_plan(world, rank)["f0_hz"])], dtype=torch.float64)
    got = [torch.zeros_like(mine) for _ in range(world)]
    if world > 1:
        dist.all_gather(got, mine)
        dist.destroy_process_group()
    else:
        got = [mine]
    if rank != 0:
        return None
    return {"spawn_check": True, "n_gpus": world, "requested_gpus": args.gpus, "f0_hz": [float(x.item()) for x in got]}


class Loaded:
    """One config resident in HBM: inputs, plan, output grid."""

    def __init__(self, cfg: int, dev, band: int = 0, tuning=None, n_bands: int = 1):
        import torch
        import synth
        from paper_1003_5575_b200 import gridder
        wl = synth.make_workload(cfg, band=band, n_bands=n_bands)       # one cell size for all ranks' bands
        self.wl = wl
        nt, nb, nf = wl.n_time, wl.n_baseline, wl.n_chan
        self.vis = torch.empty((nt, nb, nf, 4, 2), dtype=torch.float32, device=dev)
        self.weight = torch.empty((nt, nb, nf), dtype=torch.float32, device=dev) if wl.random_weights else None
        for t in range(nt):
            self.vis[t] = wl.vis_block(t, dev)
            if self.weight is not None:
                self.weight[t] = wl.weight_block(t, dev)
        self.uvw = torch.from_numpy(wl.uvw).to(dev)
        self.freq = torch.from_numpy(wl.freq).to(dev)
        self.table = torch.from_numpy(wl.kernel).to(dev)
        self.grid = torch.empty((4, wl.grid_size, wl.grid_size, 2), dtype=torch.float32, device=dev)
        self.dev = dev
        self.g = self.plan(tuning)

    def plan(self, tuning=None):
        from paper_1003_5575_b200 import gridder
        wl = self.wl
        return gridder.Gridder(grid_size=wl.grid_size, cell_size=wl.cell_size, oversample=wl.oversample, support=wl.support,
                               kernel=self.table, max_vis=wl.n_vis, n_wplanes=wl.n_wplanes, w_max=wl.w_max,
                               kernel_is_complex=wl.kernel_is_complex, tuning=tuning)

    def step(self):
        self.g.bin(self.uvw, self.freq)
        self.g.grid(self.vis, self.weight, out=self.grid)

    def close(self):
        self.g.destroy()
        self.g.workspace = None


def timed_steps(step, steps: int, barrier) -> list:
    """Device milliseconds of each of `steps` calls of step(): CUDA events around every step on the current stream
    (the stream the library launches on), a barrier + synchronise on both sides of the whole region."""
    import torch
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    barrier()
    ev[0].record()
    for k in range(steps):
        step()
        ev[k + 1].record()
    barrier()
    return [ev[k].elapsed_time(ev[k + 1]) for k in range(steps)]


def _median(xs):
    xs = sorted(xs)
    m = len(xs) // 2
    return xs[m] if len(xs) % 2 else 0.5 * (xs[m - 1] + xs[m])


def kernel_rooflines(L: "Loaded", stage: dict, st, st_exec, ms_per_step: float, fma_peak_tf: float, hbm_peak: float,
                     hbm_source: str, fma_source: str) -> dict:
    """the longest kernel of the step against the roofline that bounds it -- 16 (32) flop per
    visibility-tap against the FP32-FMA peak, or 32 B + 4 B per visibility (+ uvw, + the grid once) against HBM --
    and the same for the whole step.  Every number here reproduces from stage_ms, config and the stats."""
    wl, cfg = L.wl, L.wl.cfg
    n, nt, nb, nf = wl.n_vis, wl.n_time, wl.n_baseline, wl.n_chan
    has_w = L.weight is not None
    flop_per_tap = FLOP_PER_VIS_TAP * (2 if wl.kernel_is_complex else 1)
    grid_bytes = 32 * wl.grid_size ** 2
    alg_bytes = n * (32 + (4 if has_w else 0)) + nt * nb * 24 + nf * 8 + grid_bytes
    exec_flop = 2.0 * st_exec.fma_executed
    nominal_flop = float(flop_per_tap * st.vis_taps)
    kernels = {}

    def alu(name, ms, flop, extra=None):
        tf = flop / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
        d = {"bound": "alu", "kernel": name, "achieved": tf, "peak": fma_peak_tf, "unit": "TFLOP/s",
             "frac": tf / fma_peak_tf if fma_peak_tf else None, "kernel_ms": ms, "flop_per_launch": flop,
             "kernel_share_of_step": ms / ms_per_step if ms_per_step else None, "peak_source": fma_source,
             "traffic": NCU_TRAFFIC_BYTES.get((name, cfg)),
             "traffic_source": "profiles/r02 ncu --set full capture (historical)" if (name, cfg) in NCU_TRAFFIC_BYTES else None}
        d.update(extra or {})
        return d

    def hbm(name, ms, nbytes, extra=None):
        gbs = nbytes / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
        d = {"bound": "hbm", "kernel": name, "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
             "kernel_ms": ms, "bytes_per_launch": int(nbytes), "kernel_share_of_step": ms / ms_per_step if ms_per_step else None,
             "peak_source": hbm_source, "frac_of_8tbs": gbs / 8000.0, "traffic": NCU_TRAFFIC_BYTES.get((name, cfg)),
             "traffic_source": "profiles/r02 ncu --set full capture (historical)" if (name, cfg) in NCU_TRAFFIC_BYTES else None}
        d.update(extra or {})
        return d

    # the grid kernel executes FMAs on the records left after merging (exact by linearity): the fraction is claimed
    # on the FMAs it EXECUTED; the nominal rate (16 flop per visibility-tap gridded) is beside it
    merged = st.n_entries / st_exec.n_records_gridded if st_exec.n_records_gridded else None
    kernels["grid_kernel"] = alu("grid_kernel", stage["grid"], exec_flop, {
        "records_gridded": st_exec.n_records_gridded, "merge_factor": merged,
        "nominal": {"tflops": nominal_flop / (stage["grid"] * 1e-3) / 1e12 if stage["grid"] > 0 else None,
                    "flop_per_launch": nominal_flop,
                    "note": "16 (32) flop per visibility-tap gridded; not a roofline statement once visibilities are pre-summed"}})
    if stage.get("presum", 0.0) > 0:
        # SURVEY 8(d) algorithmic bytes of the kernel that streams the visibilities: 32 B + 4 B weight each
        ps_bytes = n * (32 + (4 if has_w else 0))
        io_bytes = n * (32 + (4 if has_w else 0) + 1) + st.n_presum_records * 32
        kernels["presum_kernel"] = hbm("presum_kernel", stage["presum"], ps_bytes, {
            "partial_records": st.n_presum_records, "vis_per_record": n / st.n_presum_records if st.n_presum_records else None,
            "frac_kernel_io": io_bytes / (stage["presum"] * 1e-3) / 1e9 / hbm_peak,
            "kernel_io_bytes": int(io_bytes), "note": "frac: 32 B + 4 B per visibility (SURVEY 8(d)); frac_kernel_io adds the "
                                                     "flag byte per visibility and the 32 B written per partial record"})
    longest = max(kernels.values(), key=lambda k: k["kernel_ms"])
    out = dict(longest)
    out["kernels"] = kernels
    out["step"] = {
        "algorithmic_bytes": int(alg_bytes), "ms_per_step": ms_per_step,
        "frac_of_hbm_peak": alg_bytes / (ms_per_step * 1e-3) / 1e9 / hbm_peak if ms_per_step else None,
        "executed_flop": exec_flop, "frac_of_fma_peak": exec_flop / (ms_per_step * 1e-3) / 1e12 / fma_peak_tf if ms_per_step else None,
        "nominal_flop": nominal_flop,
        "nominal_frac_of_fma_peak": nominal_flop / (ms_per_step * 1e-3) / 1e12 / fma_peak_tf if ms_per_step else None,
        "binding": "hbm" if alg_bytes / (hbm_peak * 1e9) > exec_flop / (fma_peak_tf * 1e12) else "alu",
        "floor_ms": {"hbm": alg_bytes / (hbm_peak * 1e9) * 1e3, "fma_executed": exec_flop / (fma_peak_tf * 1e12) * 1e3,
                     "fma_nominal": nominal_flop / (fma_peak_tf * 1e12) * 1e3},
        "note": "after pre-summation the binding roofline of the step is the slower of HBM (inputs once) and the FMAs "
                "actually executed; the nominal-FMA figure is kept for comparison with a gridder that may not merge"}
    return out


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

    shard = shard_plan(world, rank)
    L = Loaded(args.config, dev, band=shard["band"], n_bands=world)
    wl, g = L.wl, L.g
    nt, nb, nf, n = wl.n_time, wl.n_baseline, wl.n_chan, wl.n_vis
    mfs_on = bool(args.mfs and world > 1)
    if mfs_on:
        from paper_1003_5575_b200 import mfs

    def step():
        L.step()
        if mfs_on:
            mfs.reduce_grids(L.grid)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    st = g.stats()
    g.set_profiling(True)
    launches0 = g.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    per_step = timed_steps(step, args.steps, barrier)
    clocks = sampler.stop()
    ms_rank = float(sum(per_step))
    stage = g.stage_ms()
    st_exec = g.stats()                   # records gridded / FMAs executed by the last gridder_grid
    launches = g.launch_count() - launches0 + (args.steps if mfs_on else 0)      # + gridder_sum_parts per step
    g.set_profiling(False)
    checksum = float(L.grid[0, wl.grid_size // 2, wl.grid_size // 2, 0].item())

    def gather(x: float):
        if world == 1:
            return [x]
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        out = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(out, t)
        return [float(o.item()) for o in out]

    agg = aggregate(gather(ms_rank), gather(float(st.vis_taps)), args.steps)

    # ---- end to end: pinned host buffers through gridder_run_host, the same number of steps --------------
    e2e = None
    if not args.no_e2e:
        per_t = nb * nf * (32 + (4 if L.weight is not None else 0))
        nt_e = int(max(1, min(nt, _host_budget_bytes(world) // max(1, per_t))))
        h_vis = torch.empty((nt_e, nb, nf, 4, 2), dtype=torch.float32, pin_memory=True)
        h_vis.copy_(L.vis[:nt_e])
        h_w = None
        if L.weight is not None:
            h_w = torch.empty((nt_e, nb, nf), dtype=torch.float32, pin_memory=True)
            h_w.copy_(L.weight[:nt_e])
        h_uvw = torch.from_numpy(np.ascontiguousarray(wl.uvw[:nt_e])).pin_memory()
        h_freq = torch.from_numpy(wl.freq).pin_memory()
        h_grid = torch.empty(L.grid.shape, dtype=torch.float32, pin_memory=True)
        staging = {"uvw": L.uvw, "freq": L.freq, "vis": L.vis, "weight": L.weight, "grid": L.grid}
        g.run_host(h_uvw, h_freq, h_vis, h_w, h_grid, staging)            # warm-up
        taps_e = st.vis_taps * nt_e // nt        # (run_host grids in slices; the plan's stats are the last slice's)
        per_e = timed_steps(lambda: g.run_host(h_uvw, h_freq, h_vis, h_w, h_grid, staging), args.steps, barrier)
        agg_e = aggregate(gather(float(sum(per_e))), gather(float(taps_e)), args.steps)
        h2d = h_vis.numel() * 4 + (h_w.numel() * 4 if h_w is not None else 0) + h_uvw.numel() * 8 + h_freq.numel() * 8
        e2e = {"value": agg_e["value"], "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(h_grid.numel() * 4), "ms_per_step": agg_e["ms_per_step"],
               "ms_per_step_min": min(per_e), "ms_per_step_median": _median(per_e),
               "steps": args.steps, "n_time": nt_e, "result_checksum": float(h_grid[0, wl.grid_size // 2, wl.grid_size // 2, 0])}
        del h_vis, h_w, h_grid
    f1 = None
    if args.atomic:
        # row f1: per-visibility FP32 atomic scatter, same inputs, one warm-up and one timed pass
        g.scatter_atomic(L.uvw, L.freq, L.vis, L.weight, out=L.grid)
        ms_f1 = timed_steps(lambda: g.scatter_atomic(L.uvw, L.freq, L.vis, L.weight, out=L.grid), 1, barrier)[0]
        f1 = {"ms": ms_f1, "value": st.vis_taps / (ms_f1 * 1e-3), "unit": UNIT,
              "note": "gridder_scatter_atomic: no binning, red.global.add.v2.f32 per (tap, pol); not deterministic"}
    # the same workload with merging and pre-summation off: every visibility gridded on its own (what per-visibility
    # GCFs would need) -- the like-for-like FMA-bound number
    unmerged = None
    if world == 1 and not args.no_unmerged:
        L.close()
        torch.cuda.empty_cache()
        L.g = L.plan({"merge": 2})
        L.step()
        torch.cuda.synchronize()
        L.g.set_profiling(True)
        ms_u = timed_steps(L.step, 2, barrier)
        st2, stage2 = L.g.stats(), L.g.stage_ms()
        unmerged = {"grid_kernel_ms": stage2["grid"], "fma_executed": st2.fma_executed, "ms_per_step": min(ms_u),
                    "records_gridded": st2.n_records_gridded}
    L.close()
    shapes = {"nt": nt, "nb": nb, "nf": nf, "n": n}
    has_weight = L.weight is not None

    # ---- compact legs on the other configs (after the timed region; development figures for the driver record) --
    per_config = None
    if world == 1 and not args.no_per_config and rank == 0:
        del L
        torch.cuda.empty_cache()
        per_config = {}
        for c in (0, 1, 2, 3):
            if c == args.config:
                continue
            Lc = Loaded(c, dev)
            for _ in range(3):
                Lc.step()
            torch.cuda.synchronize()
            Lc.g.set_profiling(True)
            reps = 20 if c < 2 else 10
            ms_c = timed_steps(Lc.step, reps, barrier)
            sc, stc = Lc.g.stage_ms(), Lc.g.stats()
            per_config[f"config{c}"] = {"ms_per_step_min": min(ms_c), "ms_per_step_median": _median(ms_c), "steps": reps,
                                        "vis_taps": stc.vis_taps, "stage_ms": sc, "fma_executed": stc.fma_executed,
                                        "records_gridded": stc.n_records_gridded, "presum_records": stc.n_presum_records,
                                        "complex_table": bool(Lc.wl.kernel_is_complex)}
            Lc.close()
            del Lc
            torch.cuda.empty_cache()
    # ---- row f4: the paper's deployment shape, 12 consecutive channels of a GPU, one grid each (PAPER.md :108-120)
    f4 = None
    if world == 1 and not args.no_per_config:
        import synth
        wl12 = synth.make_workload(4, n_chan=12)
        v12 = torch.stack([wl12.vis_block(t, dev) for t in range(wl12.n_time)])
        w12 = torch.stack([wl12.weight_block(t, dev) for t in range(wl12.n_time)])
        u12, f12 = torch.from_numpy(wl12.uvw).to(dev), torch.from_numpy(wl12.freq).to(dev)
        tab = torch.from_numpy(wl12.kernel).to(dev)
        kw12 = dict(grid_size=wl12.grid_size, cell_size=wl12.cell_size, oversample=wl12.oversample, support=wl12.support, kernel=tab)
        gb = gridder.Gridder(max_vis=wl12.n_vis, max_grids=12, **kw12)
        grids = torch.empty((12, 4, wl12.grid_size, wl12.grid_size, 2), dtype=torch.float32, device=dev)

        def batched():
            gb.bin(u12, f12, chans_per_grid=1)
            gb.grid(v12, w12, out=grids)
        for _ in range(3):
            batched()
        ms_b = timed_steps(batched, 10, barrier)
        taps12 = gb.stats().vis_taps
        gb.destroy()
        g1 = gridder.Gridder(max_vis=wl12.n_vis // 12, **kw12)
        vc = [v12[:, :, c:c + 1].contiguous() for c in range(12)]
        wc = [w12[:, :, c:c + 1].contiguous() for c in range(12)]

        def one_by_one():
            for c in range(12):
                g1.bin(u12, f12[c:c + 1])
                g1.grid(vc[c], wc[c], out=grids[c])
        for _ in range(2):
            one_by_one()
        ms_1 = timed_steps(one_by_one, 5, barrier)
        g1.destroy()
        f4 = {"workload": "config 4 geometry, first 12 channels, 8 integrations, one 4096^2 grid per channel",
              "n_vis": wl12.n_vis, "n_grids": 12, "batched_ms_min": min(ms_b), "batched_ms_median": _median(ms_b),
              "twelve_bin_grid_rounds_ms_min": min(ms_1), "vis_taps_per_s": taps12 / (min(ms_b) * 1e-3),
              "note": "gridder_bin_channels + gridder_grid_channels: one map, one sort, one set of kernel launches for the "
                      "12 grids, against 12 gridder_bin + gridder_grid rounds on per-channel copies"}
        del v12, w12, grids, vc, wc
        torch.cuda.empty_cache()
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return None

    # ---- rooflines -------------------------------------------------------------------------
    peaks = measured_peaks()
    props = torch.cuda.get_device_properties(dev)
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    fma_peak_tf = props.multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    fma_source = (f"derived: {props.multi_processor_count} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x {sm_max_mhz:.0f} MHz "
                  "(clocks.max.sm); DESIGN.md section 7")
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_source = "MEASURED_PEAKS.json hbm_gbs (copy bandwidth)" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md)"
    flop_per_tap = FLOP_PER_VIS_TAP * (2 if wl.kernel_is_complex else 1)

    class _Shim:                      # (the Loaded object is gone: what kernel_rooflines needs of it)
        pass
    shim = _Shim()
    shim.wl, shim.weight = wl, (True if has_weight else None)
    roofline = kernel_rooflines(shim, stage, st, st_exec, agg["ms_per_step"], fma_peak_tf, hbm_peak, hbm_source, fma_source)
    roofline["frac_at_sampled_clock"] = (roofline["frac"] * sm_max_mhz / clocks["sm_mhz"]
                                         if roofline["bound"] == "alu" and clocks.get("sm_mhz") else None)
    if per_config:
        for name, pc in per_config.items():
            fpt = FLOP_PER_VIS_TAP * (2 if pc["complex_table"] else 1)
            t = pc["ms_per_step_min"] * 1e-3
            pc["vis_taps_per_s"] = pc["vis_taps"] / t
            pc["nominal_frac_of_fma_peak"] = fpt * pc["vis_taps"] / t / 1e12 / fma_peak_tf
            pc["executed_frac_of_fma_peak_grid_kernel"] = (2.0 * pc["fma_executed"] / (pc["stage_ms"]["grid"] * 1e-3) / 1e12 / fma_peak_tf
                                                          if pc["stage_ms"]["grid"] > 0 else None)
    out = {
        "metric": METRIC, "value": agg["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": warmup, "ms_per_step": agg["ms_per_step"], "ms_per_step_min": min(per_step),
        "ms_per_step_median": _median(per_step), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{wl.cfg}", "n_antennas": wl.n_ant, "n_baselines": nb, "n_chan": nf,
                   "n_time": nt, "n_vis_per_gpu": n, "grid": wl.grid_size, "support": max(wl.support),
                   "oversample": wl.oversample, "n_wplanes": wl.n_wplanes, "weights": has_weight,
                   "parallelism": (f"channel-block x{world} + grid sum (all-to-all, FP64 fixed-order sum, all-gather)"
                                   if mfs_on else f"channel-block x{world} (no collective)"),
                   "l2": "inputs per step exceed the 126 MB L2" if n * 32 > (126 << 20) else "L2-resident inputs",
                   "tile": st.tile_size, "chunk": st.chunk_size, "work_items": st.n_work_items,
                   "grid_warps_per_sm": st.grid_warps_per_sm, "presum_records": st.n_presum_records},
        "gflops_nominal": flop_per_tap * agg["value"] / 1e9,
        "stage_ms": stage, "grid_only_ms": stage["grid"] + stage["flush"] + stage.get("presum", 0.0),   # gridder_grid alone (a bin serves many)
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
        "cadence_budget_s": 8.0, "result_checksum": checksum,
    }
    if unmerged is not None and unmerged["grid_kernel_ms"] > 0:
        tf = 2.0 * unmerged["fma_executed"] / (unmerged["grid_kernel_ms"] * 1e-3) / 1e12
        unmerged.update({"achieved": tf, "frac": tf / fma_peak_tf, "unit": "TFLOP/s",
                         "step_frac_of_nominal_fma_roofline": (flop_per_tap * st.vis_taps / (fma_peak_tf * 1e12)) / (unmerged["ms_per_step"] * 1e-3),
                         "note": "tuning merge = off: every visibility gridded on its own, same grid kernel"})
        out["roofline"]["without_merging"] = unmerged
    if f1 is not None:
        out["f1_atomic_scatter"] = f1
    if e2e is not None:
        out["e2e"] = e2e
    if per_config is not None:
        out["per_config"] = per_config
    if f4 is not None:
        out["f4_channel_grids"] = f4
    if world == 1 and not args.no_cpu:
        import oracle
        oracle.build()
        out["cpu_baseline"] = cpu_baseline(args.config, args.cpu_seconds)
        # one oracle thread on the small configs, for comparison with the paper's single Nehalem core
        # (PAPER.md :216, Table 3: 13 285 ms for 12 channels ~ 68 M visibility-taps/s, derived in BASELINE.md)
        one = {}
        for c in (0, 1):
            s1 = OracleSample(c, 1 if c == 1 else synth_shape(c)["n_time"], min(4, synth_shape(c)["n_chan"]))
            s1.run(n_threads=1)
            taps, dt, _ = s1.run(n_threads=1)
            one[f"config{c}"] = {"value": taps / dt, "unit": UNIT, "cores": 1, "sample": s1.describe(), "seconds": dt}
        out["cpu_baseline"]["one_thread"] = one
    return out


def synth_shape(cfg: int) -> dict:
    import synth
    return synth.config_shape(cfg)


def main():
    args = parse_args()
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        print(json.dumps(run_reference(args)), flush=True)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(_self_spawn(args))
    if args.spawn_check:
        out = spawn_check(args)
        if out is not None:
            print(json.dumps(out), flush=True)
        return
    out = run_ours(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
