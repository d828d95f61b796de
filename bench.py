#!/usr/bin/env python
"""bench.py - throughput of the gridding hot path on seeded synthetic input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C4] [--design auto]

A step = one mwa_grid_visibilities call (scale + binning + gridding + write-out) over one whole snapshot of
the named config.  `value` is whole-job vis*pol samples/s with the inputs resident in HBM; `e2e` is the same
metric through mwa_grid_visibilities_host with pinned HOST buffers (H2D of the inputs and D2H of the grid
inside the timed region).  With N > 1 (torchrun) every rank grids its own snapshot (channels / snapshots are
independent: no collective on the data path) and the time is the max over ranks: weak scaling.
`--impl reference` times the fp64 CPU oracle, as it stands, on the host cores.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from gen import CONFIGS, generate  # noqa: E402

METRIC = "gridded_vis_pol_samples_per_sec"
UNIT = "vis_pol/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines, self.thread = index, None, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
                power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "power_w_max": max(power) if power else None, "samples": len(sm)}


def _dist():
    ws = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    lr = int(os.environ.get("LOCAL_RANK", "0"))
    return ws, rank, lr


# --------------------------------------------------------------------------------------------- reference arm
def run_reference(args):
    ws, rank, _ = _dist()
    if rank != 0:
        return
    import oracle  # the one other place bench.py may execute oracle/
    from gen import scaled
    cfg = CONFIGS[args.config]
    cores = os.cpu_count() or 1
    n_ch = min(cfg.n_chan, max(cores, 8))
    # bounded sample of the workload: all rows, n_ch channels evenly spaced over the same band
    g = generate(scaled(cfg, n_chan=n_ch), device="cuda" if torch.cuda.is_available() else "cpu")
    uv, fr, vis, w = g.uv.cpu(), g.freqs.cpu(), g.vis.cpu(), g.weights.cpu()

    def step():
        oracle.grid(uv, fr, vis, w, cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O, g.kernel_table,
                    want_abs=False, n_threads=cores)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    val = cfg.n_vis * n_ch * 4 / dt
    sample = f"{n_ch} channels evenly spaced over the band of {cfg.name} (all {cfg.n_vis} rows each) per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{cfg.name} (bounded sample: {sample})"},
        "kernel_tap_updates_per_sec": val * cfg.support_W ** 2,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": min(cores, n_ch), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# --------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    ws, rank, lr = _dist()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(lr)
    dist = None
    if ws > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", lr))
    # importing the package builds the library when it is stale: rank 0 does that alone, the others import afterwards
    if rank == 0:
        import paper_0902_0915_b200 as lib
    if dist is not None:
        dist.barrier()
    import paper_0902_0915_b200 as lib
    cfg = CONFIGS[args.config]
    if args.n_chan:                               # profiling subset (ncu captures): same rows, the TOP n channels
        from gen import scaled                    # of the band at the config's own channel spacing (same du)
        step_hz = (cfg.f_hi_hz - cfg.f_lo_hz) / max(cfg.n_chan - 1, 1)
        cfg = scaled(cfg, n_chan=args.n_chan, f_lo_hz=cfg.f_hi_hz - step_hz * (args.n_chan - 1))
    dev = torch.device("cuda", lr)
    g = generate(cfg, device=dev)
    if args.row_order == "baseline-major":          # comparison runs of design 2 (K3b): [baseline][integration] rows
        from gen import baseline_major
        g = baseline_major(g)
    plan = lib.Plan(cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O, g.kernel_table, design=args.design)
    lib.mwa_grid_plan_set_profiling(plan.handle, True)        # the plan's stage timers (CUDA events on the call's stream); see below
    if args.mfs:                                  # comparison runs only: all channels onto one shared grid (f3)
        plan.set_mfs(True)
    grid = torch.empty((1 if args.mfs else cfg.n_chan, 4, cfg.grid_n, cfg.grid_n), dtype=torch.complex64, device=dev)
    alg_bytes = cfg.algorithmic_bytes()
    small = alg_bytes < 512e6                     # fits (mostly) in the 126 MB L2: flush between iterations
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if small else None

    # Stage timers: on during the timed steps (the roofline's kernel time then comes from the timed region itself), except on
    # the launch-bound configs (C1 - C3, a call of 0.02 - 0.4 ms): there the event records between the kernels cost
    # microseconds and keep the gridding kernel from being launched as a programmatic dependent of its pre-pass, so the
    # timed steps run without them and a second pass of the same steps measures the split.
    inline_timers = not small
    lib.mwa_grid_plan_set_profiling(plan.handle, inline_timers)

    def step():
        if flush is not None:
            flush.fill_(1)
        lib.mwa_grid_visibilities(plan.handle, g.uv, g.freqs, g.vis, g.weights, cfg.n_vis, cfg.n_chan, grid)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(lr)
    if rank == 0:
        sampler.start()
    stage = []
    tot_ms = 0.0
    launches = 0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(args.steps):
        if flush is not None:
            flush.fill_(1)
        ev0.record()
        lib.mwa_grid_visibilities(plan.handle, g.uv, g.freqs, g.vis, g.weights, cfg.n_vis, cfg.n_chan, grid)
        ev1.record()
        ev1.synchronize()
        tot_ms += ev0.elapsed_time(ev1)
        if inline_timers:
            stage.append(lib.mwa_grid_plan_stage_ms(plan.handle))
        launches += lib.mwa_grid_plan_last_launches(plan.handle)
    barrier()
    if not inline_timers:                         # second pass, same steps, stage timers on: the per-stage split and the roofline
        lib.mwa_grid_plan_set_profiling(plan.handle, True)
        for _ in range(args.steps):
            if flush is not None:
                flush.fill_(1)
            lib.mwa_grid_visibilities(plan.handle, g.uv, g.freqs, g.vis, g.weights, cfg.n_vis, cfg.n_chan, grid)
            torch.cuda.synchronize()
            stage.append(lib.mwa_grid_plan_stage_ms(plan.handle))
        lib.mwa_grid_plan_set_profiling(plan.handle, False)
        barrier()
    ran = lib.mwa_grid_plan_last_design(plan.handle)           # resolves AUTO (device-side choice)
    clocks = sampler.stop() if rank == 0 else None
    t = torch.tensor([tot_ms], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_per_step = float(t.item()) / args.steps
    value = ws * cfg.vis_pol() / (ms_per_step * 1e-3)
    grid_ms = sum(s[1] for s in stage) / len(stage)
    bin_ms = sum(s[0] for s in stage) / len(stage)

    # ---- end to end through the host entry point (pinned host buffers)
    e2e = None
    if not args.no_e2e:
        try:
            h_uv, h_fr = g.uv.cpu().pin_memory(), g.freqs.cpu().pin_memory()
            h_vis, h_w = g.vis.cpu().pin_memory(), g.weights.cpu().pin_memory()
            del grid
            torch.cuda.empty_cache()
            h_grid = torch.empty((cfg.n_chan, 4, cfg.grid_n, cfg.grid_n), dtype=torch.complex64).pin_memory()
            n_e2e = max(1, min(args.steps, 3))
            lib.mwa_grid_visibilities_host(plan.handle, h_uv, h_fr, h_vis, h_w, cfg.n_vis, cfg.n_chan, h_grid)
            barrier()
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                lib.mwa_grid_visibilities_host(plan.handle, h_uv, h_fr, h_vis, h_w, cfg.n_vis, cfg.n_chan, h_grid)
            torch.cuda.synchronize()
            dt = torch.tensor([(time.perf_counter() - t0) / n_e2e], dtype=torch.float64, device=dev)
            if dist is not None:
                dist.all_reduce(dt, op=dist.ReduceOp.MAX)
            h2d = h_uv.numel() * 8 + h_fr.numel() * 8 + h_vis.numel() * 8 + h_w.numel() * 4
            e2e = {"value": ws * cfg.vis_pol() / float(dt.item()), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                   "d2h_bytes_per_step": int(h_grid.numel() * 8), "ms_per_step": float(dt.item()) * 1e3,
                   "steps": n_e2e, "host_memory": "pinned"}
            del h_grid
        except Exception as ex:  # report, never fake
            e2e = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = _peaks()
    fp32_ffma, fp32_ffma2 = lib.mwa_grid_probe_fp32(plan.handle)   # register-only FMA loops, measured now
    fp32_peak = max(fp32_ffma, fp32_ffma2)
    achieved = alg_bytes / (grid_ms * 1e-3) / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ws, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: {cfg.n_ant} antennas, {cfg.n_vis} rows x {cfg.n_chan} channels x 4 pol, "
                               f"grid {cfg.grid_n}^2 per channel and pol, kernel {cfg.support_W}x{cfg.support_W} "
                               f"oversampling {cfg.oversample_O}",
                   "design": args.design, "design_ran": ran, "row_order": args.row_order, "mfs": bool(args.mfs), "per_gpu": "one full snapshot per rank",
                   "stage_split": "stage timers on during the timed steps" if inline_timers else
                                  "launch-bound config: timed steps without stage timers; stage_ms and roofline from a second pass of the same steps with them on",
                   "cache": "256 MB L2 flush before every step" if small else
                            f"inputs+outputs {alg_bytes / 1e9:.1f} GB >> 126 MB L2, no flush"},
        "kernel_tap_updates_per_sec": value * cfg.support_W ** 2,
        "stage_ms": {"scale_and_binning": bin_ms, "gridding": grid_ms},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": None, "peak_source": peak_src, "kernel": {"gather": "gather_kernel", "chan": "chan_kernel", "chanws": "chanws_kernel", "atomic": "atomic_grid_kernel",
                                "smem": "smem_kernel", "romein": "romein_kernel"}.get(ran, ran),
                     "frac_is": "algorithmic bytes / time of the gridding stage (index + list pre-passes and the gridding kernel; "
                                "CUDA events recorded by the library) / peak; whole_call_frac adds scale + binning",
                     "algorithmic_bytes_per_launch": alg_bytes,
                     "whole_call_frac": alg_bytes / (ms_per_step * 1e-3) / 1e9 / peak,
                     "fp32_peak_tflops_measured": {"fma.rn.f32": fp32_ffma, "fma.rn.f32x2": fp32_ffma2},
                     "smem_atomic_peak_lane_ops_per_s": lib.mwa_grid_probe_smem_atomics(plan.handle),
                     "fp32_time_ms_at_measured_peak": cfg.tap_updates() * 4 / (fp32_peak * 1e12) * 1e3,
                     "hbm_time_ms_at_peak": alg_bytes / (peak * 1e9) * 1e3},
        "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
    }
    tr = os.path.join(ROOT, "profiles", "traffic.csv")      # dram bytes per launch from the committed ncu captures
    if os.path.exists(tr):
        import csv
        with open(tr) as f:
            for row in csv.DictReader(f):
                if row["workload:kernel"] == f"{cfg.name}:{out['roofline']['kernel']}" and not args.n_chan:
                    out["roofline"]["traffic"] = float(row["dram_bytes_per_launch"])
                    out["roofline"]["traffic_source"] = row["source"]

    if ws == 1 and not args.no_cpu:
        import oracle  # cpu_baseline leg: the oracle as it stands, on the box's cores, on a bounded channel sample
        cores = os.cpu_count() or 1
        uv = g.uv.cpu()

        def run_channels(chans):
            fr = g.freqs.cpu()[chans]
            vis, w = g.vis[:, chans].cpu().contiguous(), g.weights[:, chans].cpu().contiguous()
            t0 = time.perf_counter()
            used = 0
            for c0 in range(0, len(chans), cores):        # bounded memory: `cores` channel grids at a time
                sl = slice(c0, c0 + cores)
                _, _, th = oracle.grid(uv, fr[sl], vis[:, sl].contiguous(), w[:, sl].contiguous(), cfg.grid_n, g.cell_du,
                                       cfg.support_W, cfg.oversample_O, g.kernel_table, want_abs=False, n_threads=cores)
                used = max(used, th)
            return time.perf_counter() - t0, used

        def spaced(n):
            return sorted({int(round(k * (cfg.n_chan - 1) / max(n - 1, 1))) for k in range(n)})

        probe = spaced(min(cfg.n_chan, cores))
        t_probe, _ = run_channels(probe)                  # calibration: how many channels make ~15 s of CPU work
        n_ch = int(min(cfg.n_chan, max(len(probe), 15.0 / max(t_probe / len(probe), 1e-6))))
        n_ch = max(cores, (n_ch // cores) * cores) if cfg.n_chan >= cores else cfg.n_chan
        chans = spaced(min(n_ch, cfg.n_chan))
        dt, used = run_channels(chans)
        out["cpu_baseline"] = {"value": cfg.n_vis * len(chans) * 4 / dt, "unit": UNIT, "cores": used, "kind": "oracle",
                               "sample": f"{len(chans)} of {cfg.n_chan} channels of {cfg.name} evenly spaced over the band, "
                                         f"all {cfg.n_vis} rows, fp64, {dt:.1f} s of wall time on {used} threads",
                               "host_cpus": cores}
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4", choices=sorted(CONFIGS))
    ap.add_argument("--design", default="auto")
    ap.add_argument("--n-chan", type=int, default=0, help="profiling only: cut the config down to this many channels")
    ap.add_argument("--row-order", default="generated", choices=["generated", "baseline-major"],
                    help="comparison runs only: reorder the rows of a multi-integration config [baseline][integration]")
    ap.add_argument("--mfs", action="store_true", help="comparison runs only: multi-frequency synthesis onto one shared grid (implies --no-e2e)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.mfs:
        args.no_e2e = True
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: launch the ranks the way the driver does and hand over
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
