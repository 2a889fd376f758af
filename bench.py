#!/usr/bin/env python
"""EPIC hot-path benchmark (BASELINE.json metric: E-field frames/s and fraction of roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl epic|reference]

One step = one epic_image call over the whole workload (all channels x all time samples of the
configuration): unpack -> grid -> 2-D transform -> products -> accumulate.
N=1 times configs[1] (C2, the LWA-station-like case BASELINE.json's target is quoted on).
For N>1 (torchrun, one rank per GPU) every rank images its own copy of the workload -- channels
are independent, so the path shards with no collective ("weak" scaling).
Rank 0 prints ONE JSON line.  `--impl reference` times the float64 CPU oracle instead.

The line carries: `value` (device-resident inputs, CUDA events), `e2e` (one epic_image_host call per step: pinned host
voltages in, host images out, copies inside the timed region), `roofline` (algorithmic flops and bytes against the FP32
and HBM peaks, `bound` = the slower side, measured DRAM `traffic` and pipe-busy `executed` from the ncu captures under
profiles/), `clocks`, `cpu_baseline` (the oracle on one core and on all cores), and -- default C2 run only --
`other_configs` (C3, C4, C5, the streamed and tensor-core variants, the wide-support workloads).
`--sweep grid|gulp` prints the paper-figure analogues (Fig. 7, 8), one JSON line per point.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import make_config, make_custom, make_lwa55, make_per_channel  # noqa: E402

METRIC = "E-field frames/sec (chan x time gridded+FFT'd+accumulated)"
UNIT = "frames/s"
FP32_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12  # SMs x lanes x FMA x max clock
L2_FLUSH_BYTES = 256 << 20
PATH_NAMES = {1: "twopass", 2: "fused", 3: "tiled", 4: "tensor", 5: "stream"}
PATH_KERNELS = {1: "grid_rowfft+colfft_accum", 2: "epic_fused_kernel (+ epic_fused_fixup, <1 % of the step)", 3: "tiled_rows+tiled_cols",
                4: "epic_tc_kernel (column transform as BF16x3 tcgen05.mma; + epic_fused_fixup)",
                5: "tiled_stream (one persistent kernel: row CTAs -> L2 ring -> column CTAs)"}


def algorithmic_flops_per_frame(wl) -> float:
    """SURVEY.md §8(d) / DESIGN.md: row-pruned FFT 7.5 N^2 log2 N per pol (pad 2; 10 N^2 log2 N
    times (1+1/pad)/2 in general), gridding 2 (unit delta tap) or 8 flops per (antenna, tap, pol),
    4 flops/pixel per real product and 8 for XY (YX = conj, free)."""
    N, P = wl.N, wl.n_pol
    fft = 5.0 * N * N * np.log2(N) * (1.0 + 1.0 / wl.pad) * P
    grid = (2.0 if wl.taps is None else 8.0) * wl.n_ant * wl.kernel_k ** 2 * P
    prod = N * N * (4.0 * min(P, 2) + (8.0 if wl.n_products == 4 else 0.0))
    return fft + grid + prod


def algorithmic_bytes_per_frame(wl) -> float:
    """Voltages once + out_accum read and written once per call, spread over the call's frames."""
    v = wl.n_pol * wl.n_ant * (8 if wl.input_kind == "cf32" else 1)
    img = 2.0 * wl.n_planes * wl.N * wl.N * 4 / wl.n_t
    return v + img


def per_channel_variant(wl):
    """The same shape as BASELINE.json's config (antennas, grid, channels x samples, products) with
    one layout per channel: 25 kHz channels from 38 MHz, antennas uniform in a disc
    that fills the same fraction of the aperture grid, delta kernel where the config has one and
    the deployment's 3 m top-hat (3x3 cells at these wavelengths) where it has taps."""
    if wl.index not in (2, 3, 4):
        raise SystemExit("--per-channel-cells: configs 2, 3 and 4")
    diameter_m = 100.0 * wl.grid_n / 64.0
    pc = make_per_channel(grid_n=wl.grid_n, pad=wl.pad, n_ant=wl.n_ant, n_pol=wl.n_pol, kernel_k=min(wl.kernel_k, 3),
                          n_chan=wl.n_chan, n_t=wl.n_t, n_products=wl.n_products, f0_hz=38e6, df_hz=25e3,
                          diameter_m=diameter_m, layout_seed=wl.seed, seed=wl.index)
    pc.name = f"{wl.name}+per-channel-cells"
    pc.index = wl.index
    return pc


def make_wide_workload(kind: str, n_chan: int, n_t: int):
    """Workloads whose occupied cells need more than 32 x 32 (the wide fused kernel), C2's extent."""
    if kind == "lwa55-tophat":
        wl = make_lwa55(n_chan=n_chan, n_t=n_t, kernel="tophat", n_products=4)
    elif kind == "lwa55-delta":
        wl = make_lwa55(n_chan=n_chan, n_t=n_t, kernel="delta", n_products=2)
    else:
        uv = np.random.default_rng(64).uniform(-0.49, 63.49, (256, 2)).astype(np.float32)
        wl = make_custom(grid_n=64, pad=2, n_ant=256, n_pol=2, kernel_k=1, n_chan=n_chan, n_t=n_t, n_products=2, ant_uv=uv)
        wl.name = "fill64-256ant-128x128-delta-XXYY"
    wl.index = 2
    return wl


def max_over_ranks(values, device) -> list:
    """Element-wise MAX of a list of floats over all ranks (identity for a single process)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    tt = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return [float(v) for v in tt.cpu()]


def channel_shard(n_chan: int, rank: int, world: int):
    """Channels [lo, hi) of rank `rank` when ONE workload is split over ranks (channels are
    independent: no collective).  bench.py itself runs weak scaling (one full
    workload per GPU); this is the strong-scaling split a deployment would use."""
    return (n_chan * rank) // world, (n_chan * (rank + 1)) // world


class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.QUERY}",
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


HBM_FALLBACK_GBS = 6650.0  # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def measured_hbm_gbs():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except (OSError, ValueError, KeyError):
        return HBM_FALLBACK_GBS, "B200_PROFILING.md fallback"


def input_fingerprint(wl, volt) -> dict:
    """numpy version and SHA-256 of every generated buffer, so that a run can be tied to its inputs."""
    import hashlib
    h = lambda a: hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
    out = {"numpy": np.__version__, "seed": int(wl.seed), "sha256": {"voltages": h(volt), "ant_uv": h(wl.ant_uv)}}
    if wl.taps is not None:
        out["sha256"]["taps"] = h(wl.taps)
    return out


def measured_traffic(wl_name: str, path: int):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of this workload and kernel family
    from the ncu captures summarised in profiles/traffic.csv, or None."""
    row = _profile_row(wl_name, path)
    try:
        return int(row[1]) if row and row[1] else None
    except ValueError:
        return None


def _profile_row(wl_name: str, path: int):
    """Row of profiles/traffic.csv for this workload and kernel family: [key, dram bytes per launch, FMA-pipe busy %,
    issue slots busy %] from the ncu --set full capture named in profiles/traffic.md, or None."""
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(tpath) as fh:
            for ln in fh.read().splitlines()[1:]:
                f = [x.strip() for x in ln.split(",")]
                if f and f[0] == f"{wl_name}:{PATH_NAMES.get(path)}":
                    return f + [""] * (4 - len(f))
    except OSError:
        pass
    return None


def measured_pipe_busy(wl_name: str, path: int) -> dict:
    """What the dominant kernel EXECUTES, beside the algorithmic fraction: sm__pipe_fma_cycles_active and
    smsp__issue_active (% of peak) of the same ncu capture as `traffic`; None where no capture has them."""
    row = _profile_row(wl_name, path)
    def num(x):
        try:
            return float(x)
        except (TypeError, ValueError):
            return None
    return {"fma_pipe_busy_pct": num(row[2]) if row else None, "issue_slots_busy_pct": num(row[3]) if row else None,
            "source": "profiles/traffic.csv (ncu --set full capture, see profiles/traffic.md)"}


def roofline_of(wl, kernel_ms: float, path: int, probe_tflops=None) -> dict:
    """BASELINE.json north_star: the roofline is the SLOWER of (FFT + gridding + product flops at FP32 peak) and
    (voltage + image bytes at HBM bandwidth); both sides are computed and `bound` says which one binds."""
    flops = algorithmic_flops_per_frame(wl)
    bytes_f = algorithmic_bytes_per_frame(wl)
    hbm_gbs, hbm_kind = measured_hbm_gbs()
    t_alu = flops * wl.frames / (FP32_NOMINAL_TFLOPS * 1e12)
    t_hbm = bytes_f * wl.frames / (hbm_gbs * 1e9)
    achieved = flops * wl.frames / (kernel_ms * 1e-3) / 1e12
    r = {
        "bound": "alu" if t_alu >= t_hbm else "hbm", "achieved": achieved, "peak": FP32_NOMINAL_TFLOPS, "unit": "TFLOP/s",
        "frac": max(t_alu, t_hbm) / (kernel_ms * 1e-3), "traffic": measured_traffic(wl.name, path),
        "frac_kind": "algorithmic work (SURVEY.md 8(d)) / measured time; the kernels execute less than the algorithmic count where they prune",
        "peak_kind": "nominal FP32: 148 SM x 128 lanes x 2 x 1.965 GHz (DESIGN.md)",
        "t_alu_ms": t_alu * 1e3, "t_hbm_ms": t_hbm * 1e3, "hbm_peak_gbs": hbm_gbs, "hbm_peak_kind": hbm_kind,
        "algorithmic_flops_per_frame": flops, "algorithmic_bytes_per_frame": bytes_f,
        "algorithmic_bytes_per_launch": bytes_f * wl.frames,
        "hbm_achieved_gbs": bytes_f * wl.frames / (kernel_ms * 1e-3) / 1e9,
        "kernel_ms": kernel_ms, "kernel": PATH_KERNELS.get(path, str(path)),
        "executed": measured_pipe_busy(wl.name, path),
    }
    if probe_tflops:
        r["peak_measured_fma_probe"] = probe_tflops
        r["frac_of_measured_probe"] = achieved / probe_tflops
    return r


def time_other_config(label: str, wl, dev, steps: int, warmup: int, path=None, probe_tflops=None) -> dict:
    """Device-resident timing of another workload in the same process (same rules: L2 flushed between
    iterations, CUDA events on the launching stream); returns a compact record for `other_configs`."""
    import torch
    import paper_1904_11422_b200 as epic
    t0 = time.perf_counter()
    volt = wl.voltages()
    d_volt = torch.from_numpy(volt).to(dev)
    plan = epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k)
    try:
        plan.set_products(wl.n_products)
        if path is not None:
            plan.set_path(path)
        out = torch.zeros((wl.n_chan, plan.n_planes(wl.n_pol), wl.N, wl.N), dtype=torch.float32, device=dev)
        flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
        stream = torch.cuda.current_stream()
        ms = []
        for i in range(warmup + steps):
            out.zero_()
            flush.fill_(1)
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            plan.image(d_volt, wl.n_t, wl.n_chan, wl.n_pol, out, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            if i >= warmup:
                ms.append(e0.elapsed_time(e1))
        used = plan.path(wl.n_pol)
        launches = plan.last_launches()
        support = plan.support()
    finally:
        plan.destroy()
    mean_ms = float(np.mean(ms))
    roof = roofline_of(wl, mean_ms, used, probe_tflops)
    return {"label": label, "workload": wl.name, "kernel_path": PATH_NAMES.get(used, str(used)), "value": wl.frames / (mean_ms * 1e-3),
            "unit": UNIT, "ms_per_step": mean_ms, "ms_per_step_median": float(np.median(ms)), "ms_per_step_min": float(np.min(ms)),
            "steps": steps, "warmup": warmup, "launches_per_step": launches, "support_box": list(support),
            "frac": roof["frac"], "frac_of_measured_probe": roof.get("frac_of_measured_probe"), "bound": roof["bound"],
            "traffic": roof["traffic"], "algorithmic_bytes_per_launch": roof["algorithmic_bytes_per_launch"],
            "setup_s": round(time.perf_counter() - t0, 1)}


def run_sweep(args):
    """Paper-figure analogues, one JSON line per point, device-resident inputs:
    --sweep grid: image side N in {32, 64, 128, 256} with the SAME 256 dual-pol antennas (C2's disc layout scaled
                  to the same fraction of the aperture grid), delta kernel, XX and YY, 128 channels x 1000 samples
                  (Fig. 8: run time against grid size);
    --sweep gulp: C2 with n_t samples per epic_image call in {50, ..., 2500} (Fig. 7: gulp size)."""
    import torch
    import paper_1904_11422_b200 as epic
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    probe = epic.epic_fp32_peak_probe(20000)
    points = []
    if args.sweep == "grid":
        base = make_config(2, n_chan=1, n_t=1)
        for grid_n in (16, 32, 64, 128):
            uv = (grid_n / 2.0 + (base.ant_uv.astype(np.float64) - 32.0) * (grid_n / 64.0)).astype(np.float32)
            wl = make_custom(grid_n=grid_n, pad=2, n_ant=256, n_pol=2, kernel_k=1, n_chan=128, n_t=1000, n_products=2, ant_uv=uv)
            wl.name = f"sweep-grid-256ant-{2 * grid_n}x{2 * grid_n}-delta-XXYY"
            points.append((f"N = {2 * grid_n}", wl))
    else:
        for n_t in (50, 125, 250, 500, 1000, 2500):
            points.append((f"n_t = {n_t} per call", make_config(2, n_t=n_t)))
    for label, wl in points:
        rec = time_other_config(label, wl, dev, steps=args.steps, warmup=max(args.warmup, 3), probe_tflops=probe["tflops"])
        rec.update({"sweep": args.sweep, "metric": METRIC, "n_chan": wl.n_chan, "n_t": wl.n_t, "N": wl.N, "n_ant": wl.n_ant,
                    "flops_per_frame": algorithmic_flops_per_frame(wl)})
        print(json.dumps(rec))


def _cpu_worker(job):
    """One channel of the bounded sample in a worker process (all-cores leg of cpu_baseline)."""
    os.environ.setdefault("OMP_NUM_THREADS", "1")
    from oracle import epic_oracle as orc
    (volt_c, kind, ant_uv, taps, grid_n, pad, n_products, kernel_k, order) = job
    orc.epic_image(volt_c, kind, ant_uv, taps, grid_n, pad, n_products, kernel_k=kernel_k, mode="fast", order=order)
    return volt_c.shape[0]


def cpu_baseline_all_cores(wl, volt, order: str = "TCPA", seconds_hint: float = 10.0, single_fps: float = 1.0) -> dict:
    """the same oracle fanned over os.cpu_count() processes, one channel each (channels are
    independent); the time-sample count per channel is cut so that the leg stays near `seconds_hint`."""
    import multiprocessing as mp
    n_proc = os.cpu_count() or 1
    n_jobs = min(wl.n_chan, n_proc)
    n_t = int(max(1, min(volt.shape[0], single_fps * seconds_hint)))   # every process images n_t frames
    jobs = []
    for c in range(n_jobs):
        uv = wl.ant_uv[c] if wl.ant_uv.ndim == 3 else wl.ant_uv
        tp = None if wl.taps is None else (wl.taps[c] if wl.ant_uv.ndim == 3 else wl.taps)
        vc = np.ascontiguousarray(volt[:n_t, c:c + 1])
        jobs.append((vc, wl.input_kind, uv, tp, wl.grid_n, wl.pad, wl.n_products, wl.kernel_k, order))
    ctx = mp.get_context("fork")
    t0 = time.perf_counter()
    with ctx.Pool(n_jobs) as pool:
        done = pool.map(_cpu_worker, jobs)
    dt = time.perf_counter() - t0
    frames = int(sum(done))
    return {"value": frames / dt, "unit": UNIT, "cores": n_jobs, "kind": "oracle",
            "sample": f"{n_jobs} processes x 1 channel x {n_t} time samples of {wl.name} ({frames} frames, {dt:.1f} s, numpy float64, "
                      f"one thread per process, pool start-up included)"}


def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(wl, volt, n_chan_sample: int, order: str = "TCPA") -> dict:
    """The float64 oracle, as it stands, on a bounded sample of the same workload."""
    from oracle import epic_oracle as orc
    ch = list(range(min(n_chan_sample, wl.n_chan)))
    t0 = time.perf_counter()
    orc.epic_image(volt, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products,
                   kernel_k=wl.kernel_k, mode="fast", channels=ch, order=order)
    dt = time.perf_counter() - t0
    frames = len(ch) * volt.shape[0]
    return {"value": frames / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"channels 0..{len(ch) - 1} x all {volt.shape[0]} time samples of {wl.name} "
                      f"({frames} frames, {dt:.1f} s, numpy float64 single thread)"}


def run_reference(args, wl):
    """--impl reference: the oracle on the host cores, each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_t = min(wl.n_t, 250)
    small = make_config(wl.index, n_chan=2, n_t=n_t)
    if wl.ant_uv.ndim == 3:
        small = per_channel_variant(small)
    volt = small.voltages()
    times = []
    res = None
    for i in range(args.warmup + args.steps):
        res = cpu_baseline(small, volt, 2)
        if i >= args.warmup:
            times.append(2 * n_t / res["value"])
    ms = 1e3 * float(np.mean(times))
    value = 2 * n_t / (ms * 1e-3)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, **{k: v for k, v in wl.describe().items() if k != "workload"},
                   "step_sample": f"2 channels x {n_t} time samples per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": res["sample"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_epic(args, wl):
    import torch
    import torch.distributed as dist
    import paper_1904_11422_b200 as epic

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    volt = wl.voltages()                       # host, seeded synthetic (DESIGN.md input recipe)
    if args.input_order == "tcap":             # the untransposed F-engine order
        volt = np.ascontiguousarray(np.swapaxes(volt, 2, 3))
    h_volt = torch.from_numpy(volt).pin_memory()
    d_volt = h_volt.to(dev, non_blocking=True)
    plan = epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k)
    plan.set_products(wl.n_products)
    if args.path:
        plan.set_path({"auto": 0, "twopass": 1, "fused": 2, "tiled": 3, "tensor": 4, "stream": 5}[args.path])
    if args.scratch_mib:
        plan.set_scratch_limit(args.scratch_mib << 20)
    if args.input_order == "tcap":
        plan.set_input_order(epic.EPIC_ORDER_TCAP)
    if args.delay_phasors:                     # unit-modulus synthetic cable phases
        ph_rng = np.random.default_rng(wl.seed + 77)
        plan.set_delay_phasors(np.exp(2j * np.pi * ph_rng.random((wl.n_chan, wl.n_pol, wl.n_ant))).astype(np.complex64))
    planes = plan.n_planes(wl.n_pol)
    out = torch.zeros((wl.n_chan, planes, wl.N, wl.N), dtype=torch.float32, device=dev)
    h_out = torch.empty(out.shape, dtype=torch.float32).pin_memory()
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    call = plan.image_cf32 if wl.input_kind == "cf32" else plan.image

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        out.zero_()
        flush.fill_(1)                          # L2 flush between timed iterations
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        call(d_volt, wl.n_t, wl.n_chan, wl.n_pol, out, stream)
        e1.record(stream)
        return e0, e1

    # End to end through the C ABI with HOST buffers: epic_image_host (include/epic.h) takes the pinned host voltages
    # and a pinned host out_accum; inside it the gulp is cut into time chunks whose H2D copies (copy stream) overlap
    # the previous chunk's kernels (compute stream), and the accumulated images are copied back.  The call is
    # synchronous and runs on the library's own streams, so this leg is timed with the host clock around the call,
    # the device idle on both sides.
    n_chunks = max(0, min(args.e2e_chunks, wl.n_t))

    class _HostTimed:
        def __init__(self, ms):
            self.ms = ms

        def elapsed_time(self, other):
            return self.ms

    def step_e2e():
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        plan.image_host(h_volt, wl.n_t, wl.n_chan, wl.n_pol, h_out, accumulate=False, n_chunks=n_chunks)
        ms = (time.perf_counter() - t0) * 1e3
        ev = _HostTimed(ms)
        return ev, ev

    for _ in range(max(args.warmup, 3)):
        step_device()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    evs = [step_device() for _ in range(args.steps)]
    barrier()
    launches = plan.last_launches() * args.steps
    dev_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = float(sum(dev_ms))

    if wl.input_kind == "cf32":
        args.no_e2e = True   # epic_image_host takes 4+4-bit voltages (C1's cf32 gulp is 1 KiB: nothing to pipeline)
    run_e2e = step_device if args.no_e2e else step_e2e   # --no-e2e (profiling runs): the e2e object then repeats the device leg
    for _ in range(0 if args.no_e2e else 2):
        run_e2e()
    barrier()
    evs = [run_e2e() for _ in range(1 if args.no_e2e else args.steps)]
    barrier()
    clocks = sampler.stop() if rank == 0 else None  # sampled over both timed regions
    e2e_ms = float(sum(a.elapsed_time(b) for a, b in evs)) * (args.steps if args.no_e2e else 1)

    total_ms, e2e_ms = max_over_ranks([total_ms, e2e_ms], dev)
    path = plan.path(wl.n_pol)
    support = plan.support()
    probe = epic.epic_fp32_peak_probe(20000) if rank == 0 else None
    plan.destroy()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    frames_step = wl.frames * world
    ms_per_step = total_ms / args.steps
    value = frames_step / (ms_per_step * 1e-3)
    e2e_value = frames_step / (e2e_ms / args.steps * 1e-3)
    kernel_ms = float(np.mean(dev_ms))           # rank 0's own kernel time (one launch per step when fused)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step,
        "ms_per_step_median": float(np.median(dev_ms)), "ms_per_step_min": float(np.min(dev_ms)),
        "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": wl.name, **{k: v for k, v in wl.describe().items() if k != "workload"},
                   "kernel_path": PATH_NAMES.get(path, str(path)),
                   "input_order": args.input_order, "delay_phasors": bool(args.delay_phasors),
                   "layouts": int(wl.ant_uv.shape[0]) if wl.ant_uv.ndim == 3 else 1,
                   "support_box": list(support), "l2": f"flushed between iterations ({L2_FLUSH_BYTES >> 20} MiB write)",
                   "sharding": "independent replicas of the workload per GPU (channels are independent), no collective"},
        "roofline": roofline_of(wl, kernel_ms, path, probe["tflops"]),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(volt.nbytes),
                "d2h_bytes_per_step": int(out.numel() * 4), "measured": not args.no_e2e,
                "how": f"one epic_image_host call (C ABI, HOST pointers: pinned voltages in, pinned out_accum out) per step: inside "
                       f"the library {n_chunks if n_chunks else 'an automatic number of'} channel-range chunks (the first half as long as the others): H2D of chunk "
                       f"k+1 and D2H of chunk k's finished images each on their own stream, overlapped with the kernels in between; synchronous call "
                       f"timed with the host clock, device idle before and after"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "inputs": input_fingerprint(wl, volt),
    }
    if path == 4:
        # the tensor-core variant, reported beside the FP32 roofline above (same algorithmic flops, so the two
        # paths compare directly): what its MMAs execute, against the measured dense BF16 peak of this pool
        per_frame = 24 * 2.0 * 128 * 256 * 16 * (wl.N // 32) / 4   # 24 MMAs of 128x256x16 per (4 frames, one residue)
        exe = per_frame * wl.frames / (kernel_ms * 1e-3) / 1e12
        try:
            bf16_peak = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["bf16_tflops_sustained"])
            kind = "MEASURED_PEAKS.json bf16_tflops_sustained"
        except (OSError, ValueError, KeyError):
            bf16_peak, kind = 2250.0, "nominal dense BF16 (B200_PROFILING.md fallback)"
        line["roofline"]["tensor"] = {"executed_bf16_tflops": exe, "peak": bf16_peak, "frac": exe / bf16_peak,
                                      "peak_kind": kind, "executed_mma_flops_per_frame": per_frame,
                                      "note": "BF16 hi/lo split: 3 products per real product, 4 real per complex"}
    if world == 1 and args.other_configs and wl.index == 2 and not args.workload and not args.per_channel_cells \
            and args.n_chan is None and args.n_t is None:
        # the other BASELINE.json configurations and the variants DESIGN.md reports, device-resident, fewer steps
        # (C5 is 33 ms per step); the clocks line above does not cover them, so each run is bracketed by its own sample
        import paper_1904_11422_b200 as epic_mod
        others = [("C3", make_config(3), None), ("C4", make_config(4), None), ("C5", make_config(5), None),
                  ("C4 streamed kernel", make_config(4), epic_mod.EPIC_PATH_STREAM),
                  ("C5 streamed kernel", make_config(5), epic_mod.EPIC_PATH_STREAM),
                  ("C2 tensor-core column pass", make_config(2), epic_mod.EPIC_PATH_TENSOR),
                  ("LWA 55.25 MHz, 3 m top-hat, 4 products (wide fused kernel)", make_wide_workload("lwa55-tophat", 128, 1000), None),
                  ("LWA 55.25 MHz, delta, XX YY (wide fused kernel)", make_wide_workload("lwa55-delta", 128, 1000), None)]
        sampler2 = ClockSampler(local)
        sampler2.start()
        recs = []
        for label, w2, pth in others:
            try:
                recs.append(time_other_config(label, w2, dev, steps=5, warmup=3, path=pth, probe_tflops=probe["tflops"]))
            except Exception as exc:  # a failed extra must not cost the headline line
                recs.append({"label": label, "error": repr(exc)})
        line["other_configs"] = {"records": recs, "clocks": sampler2.stop(),
                                 "note": "device-resident inputs, 3 warm-up + 5 timed steps each, L2 flushed between iterations"}
    if world == 1 and not args.no_cpu_baseline:
        # bounded sample: the oracle's cost per frame grows with the plane (N^2 log N), so fewer channels of the big configs
        n_cpu = max(1, args.cpu_channels * (128 * 128) // max(128 * 128, wl.N * wl.N * wl.n_planes // 2))
        cb = cpu_baseline(wl, volt, n_cpu, args.input_order.upper())
        cb["cpu_model"] = cpu_model()
        cb["host_cores"] = os.cpu_count()
        try:
            cb["all_cores"] = cpu_baseline_all_cores(wl, volt, args.input_order.upper(), 8.0, cb["value"])
        except Exception as exc:
            cb["all_cores"] = {"error": repr(exc)}
        line["cpu_baseline"] = cb
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (1-based)")
    ap.add_argument("--impl", default="epic", choices=["epic", "reference"])
    ap.add_argument("--path", default=None, choices=[None, "auto", "twopass", "fused", "tiled", "tensor", "stream"])
    ap.add_argument("--n-chan", type=int, default=None)
    ap.add_argument("--n-t", type=int, default=None)
    ap.add_argument("--n-ant", type=int, default=None)
    ap.add_argument("--cpu-channels", type=int, default=16, help="channels of the workload the oracle images for cpu_baseline (~13 s on C2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="profiling runs only: skip the host-buffer leg (its object is then not a measurement)")
    ap.add_argument("--no-other-configs", dest="other_configs", action="store_false",
                    help="skip the other_configs block (C3, C4, C5, streamed, tensor, wide) of the default C2 run")
    ap.add_argument("--input-order", default="tcpa", choices=["tcpa", "tcap"], help="tcap = [T][C][A][Np], transposed in the load")
    ap.add_argument("--delay-phasors", action="store_true", help="apply per-(channel, pol, antenna) delay phasors")
    ap.add_argument("--e2e-chunks", type=int, default=0, help="time chunks of the end-to-end leg (H2D overlapped); 0 = the library's choice")
    ap.add_argument("--scratch-mib", type=int, default=0, help="cap the per-batch scratch (tiled / two-pass paths)")
    ap.add_argument("--per-channel-cells", action="store_true",
                    help="configs 2-4 with one antenna layout per 25 kHz channel (cell = lambda_c/2) and, for 3 and 4, "
                         "the 3 m top-hat kernel (PAPER.md:122, 162-168)")
    ap.add_argument("--workload", default=None, choices=[None, "lwa55-tophat", "lwa55-delta", "fill64"],
                    help="instead of --config: the paper's operating point (256 antennas, 110 m x 100 m, lambda/2 cells at "
                         "55.25 MHz, PAPER.md:148, 166-168) with the 3 m top-hat / four products or the delta kernel / XX, YY; "
                         "or 256 antennas uniformly filling all 64 x 64 cells (delta, XX, YY)")
    ap.add_argument("--sweep", default=None, choices=[None, "grid", "gulp"],
                    help="paper-figure analogues: image side at fixed antennas (Fig. 8) or samples per call (Fig. 7); one JSON line per point")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
        return
    if args.workload:
        wl = make_wide_workload(args.workload, args.n_chan or 128, args.n_t or 1000)
    else:
        wl = make_config(args.config, n_chan=args.n_chan, n_t=args.n_t, n_ant=args.n_ant)
    if args.per_channel_cells:
        wl = per_channel_variant(wl)
    if args.impl == "reference":
        run_reference(args, wl)
    else:
        run_epic(args, wl)


if __name__ == "__main__":
    main()
