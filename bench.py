#!/usr/bin/env python
"""bench.py -- headline measurement of the dedispersion hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config fast] [--kernel auto|direct|tiled]
    python bench.py --impl reference ...          # the CPU oracle on the host cores, same metric

A "step" is one pass of the whole hot path (ddsp_execute: stage, fused bin-sum, shifted accumulate,
write-out) over one synthetic observation.  At N = 1 the workload is BASELINE.json configs[1]
("FAST-like": 2048 channels, 150 s, 1001 DM trials).  With N > 1 (torchrun, one rank per GPU) every
rank dedisperses its own observation of that shape -- independent units, no collective on the data
path (weak scaling).  One JSON line is printed by rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "dedispersion_gadds_per_s"
UNIT = "Gadd/s (DM x chan x sample)"
SM_COUNT, SM_MAX_MHZ, ADDS_PER_CLK_SM = 148, 1965.0, 128   # P_add


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="fast", help="workload name (synth.CONFIG_NAMES); headline = fast")
    ap.add_argument("--kernel", default="auto", choices=["auto", "direct", "tiled"])
    ap.add_argument("--crop", type=int, default=0, help="debug: crop to this many output samples")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--traffic-bytes", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from an ncu capture (profiles/)")
    return ap.parse_args()


# ----------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region
# ----------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.proc, self.lines = None, []
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append((time.time(), ln.strip()))

    def window(self, t0, t1):
        rows = [ln for (t, ln) in self.lines if t0 <= t <= t1] or [ln for (_, ln) in self.lines[-3:]]
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in rows:
            f = [v.strip() for v in ln.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return None
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w": float(np.median(pw)),
                "reasons": sorted(reasons), "samples": len(sm)}

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except subprocess.TimeoutExpired:
                self.proc.kill()


# ----------------------------------------------------------------------------------------------
# workload helpers
# ----------------------------------------------------------------------------------------------
def library_native_delays(wl):
    """dm -> delays on the native grid, from the LIBRARY's own plan-time table (bench never asks the
    oracle for inputs of the CUDA path)."""
    from paper_2511_02328_b200 import binding

    def fn(dm):
        with binding.Plan(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, 1 << 40, [dm], 1, None,
                          binding.DDSP_IN_U8) as p:
            return p.get_delays()[0]
    return fn


def get_workload(args):
    from paper_2511_02328_b200 import synth
    wl = synth.config(args.config)
    return wl


def adds_per_execute(plan):
    return float(plan.ndm) * float(plan.nchan_unmasked) * float(plan.nsamp_out)


def oracle_sample(wl, x_dev_or_host, plan_geom, target_adds=1.6e10, ntrials=8):
    """Bounded sample of the same workload for the CPU oracle: all channels, `ntrials` evenly spaced
    trials, the first `ncol` output columns.  Returns (rows, ncol, host input window)."""
    nout, dmax, nch_un = plan_geom
    rows = np.unique(np.linspace(0, wl.ndm - 1, ntrials).round().astype(np.int64))
    ncol = int(min(nout, max(1024, target_adds / (len(rows) * max(1, nch_un)))))
    ncols_in = min(wl.nsamp, (ncol + dmax) * wl.downsample)
    xh = x_dev_or_host[:, :ncols_in]
    xh = xh.cpu().numpy() if hasattr(xh, "cpu") else np.ascontiguousarray(xh)
    return rows, ncol, np.ascontiguousarray(xh)


def time_oracle(wl, rows, ncol, xh, dmax):
    """Run the oracle (as it stands, single thread) on the sample; returns (seconds, output, adds)."""
    from oracle import oracle
    table, dmax_o = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    assert dmax_o == dmax
    nsamp_win = xh.shape[1]
    t0 = time.perf_counter()
    out = oracle.dedisperse_table(xh, table[rows], nsamp=nsamp_win, downsample=wl.downsample,
                                  mask=wl.mask, t_lo=0, t_hi=ncol)
    dt = time.perf_counter() - t0
    nch_un = wl.nchan - (0 if wl.mask is None else int(wl.mask.sum()))
    return dt, out, float(len(rows)) * nch_un * ncol


# ----------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2511_02328_b200 import binding, build, multi, synth

    rank, local_rank, world = multi.init()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if rank == 0:
        build.build()
    multi.barrier()
    binding.lib()

    wl = get_workload(args)
    if args.crop:
        with binding.plan_for(wl) as geom:
            wl = wl.cropped(wl.downsample * (geom.max_delay + args.crop))
    # every rank owns whole observations (units); rank r's observation uses seed + r
    unit = list(multi.shard_units(world, rank, world))[0]
    wl.seed = wl.seed + 1000 * unit

    plan = binding.plan_for(wl)
    in_pitch = synth.round_up(wl.nsamp, 128)
    out_pitch = synth.round_up(plan.nsamp_out, 32)
    plan.set_pitch(in_pitch, out_pitch)
    plan.set_kernel({"auto": 0, "direct": 1, "tiled": 2}[args.kernel])
    x = synth.make_input(wl, dev, pitch=in_pitch, native_delays=library_native_delays(wl),
                         nsamp_out=plan.nsamp_out)
    out = torch.empty((plan.ndm, out_pitch), dtype=torch.int32 if wl.dtype == "u8" else torch.float32,
                      device=dev)
    stream = torch.cuda.current_stream(dev)
    adds = adds_per_execute(plan)
    for _ in range(max(args.warmup, 0)):
        plan.execute(x, out, stream)
    torch.cuda.synchronize(dev)
    multi.barrier()

    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    t_wall0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        plan.execute(x, out, stream)
    ev1.record(stream)
    torch.cuda.synchronize(dev)
    t_wall1 = time.time()
    multi.barrier()
    secs = ev0.elapsed_time(ev1) * 1e-3
    clocks = sampler.window(t_wall0, t_wall1) if sampler else None
    if sampler:
        sampler.stop()

    total_rate, t_max = multi.job_throughput(adds * args.steps, secs)      # adds/s over all ranks
    ms_per_step = t_max / args.steps * 1e3

    # end to end through the public host-buffer call (H2D + kernels + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        e2e = measure_e2e(plan, wl, x, out, in_pitch, out_pitch, adds, min(args.steps, 3), multi)

    result = None
    if rank == 0:
        p_add = SM_COUNT * ADDS_PER_CLK_SM * SM_MAX_MHZ * 1e6                 # adds/s
        launch_s = secs / args.steps / plan.launches_per_execute
        achieved = adds / (secs / args.steps)
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except (OSError, ValueError):
            pass
        hbm = float(peaks.get("hbm_gbs", 6650.0)) * 1e9
        ideal_bytes = float(wl.nchan) * wl.nsamp * wl.elem_size + float(plan.ndm) * plan.nsamp_out * 4
        t_roof = max(ideal_bytes / hbm, adds / p_add)
        result = {
            "metric": METRIC, "value": total_rate / 1e9, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u32" if wl.dtype == "u8" else "f32", "data": "synthetic",
            "config": {"workload": "%s%s" % (wl.name, "" if not args.crop else "(cropped)"),
                       "nchan": wl.nchan, "nchan_unmasked": plan.nchan_unmasked, "ndm": plan.ndm,
                       "nsamp": wl.nsamp, "nsamp_out": plan.nsamp_out, "tsamp_s": wl.tsamp,
                       "downsample": wl.downsample, "in_dtype": wl.dtype,
                       "kernel": {1: "direct", 2: "tiled"}[plan.kernel],
                       "units": "one observation per GPU", "parallelism": "dp%d" % world,
                       "l2": "inputs (%.2f GB) larger than L2; no flush" % (x.numel() * x.element_size() / 1e9)},
            "x_realtime": plan.nsamp_out * wl.tsamp * wl.downsample / (t_max / args.steps),
            "gpu_launches": args.steps * plan.launches_per_execute,
            "clocks": clocks,
            "roofline": {"bound": "alu", "achieved": achieved / 1e9, "peak": p_add / 1e9, "unit": "Gadd/s",
                         "frac": achieved / p_add, "traffic": args.traffic_bytes,
                         "peak_source": "148 SM x 128 int32 adds/clk/SM (measured, profiles/ubench_r01_raw.txt) x 1965 MHz",
                         "kernel_ms": launch_s * 1e3,
                         "t_roof_ms": t_roof * 1e3, "frac_of_path_roofline": t_roof / (secs / args.steps),
                         "hbm_ideal_bytes": ideal_bytes, "hbm_peak_gbs": hbm / 1e9,
                         "hbm_peak_source": "measured" if peaks else "fallback"},
            "e2e": e2e,
        }
        if not args.no_cpu_baseline and world >= 1:
            rows, ncol, xh = oracle_sample(wl, x, (plan.nsamp_out, plan.max_delay, plan.nchan_unmasked))
            dt, oout, oadds = time_oracle(wl, rows, ncol, xh, plan.max_delay)
            got = out[torch.as_tensor(rows, device=dev), :ncol].cpu().numpy()
            if wl.dtype == "u8":
                ok = bool(np.array_equal(got.view(np.uint32), oout))
            else:
                ok = bool((np.abs(got.astype(np.float64) - oout) <= 1e-5 * np.abs(oout)).all())
            result["cpu_baseline"] = {"value": oadds / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
                                      "sample": "%d trials x %d channels x first %d output samples of the same "
                                                "input (%.1f s of CPU)" % (len(rows), plan.nchan_unmasked, ncol, dt),
                                      "parity_on_sample": "ok" if ok else "MISMATCH"}
        print(json.dumps(result))
        sys.stdout.flush()
    plan.destroy()
    multi.finalize()
    return result


def measure_e2e(plan, wl, x, out, in_pitch, out_pitch, adds, steps, multi):
    """Same metric through ddsp_execute_host: pinned host input -> device, kernels, result -> pinned host."""
    import psutil
    import torch
    in_bytes = x.numel() * x.element_size()
    out_bytes = out.numel() * 4
    valid_out_bytes = plan.ndm * plan.nsamp_out * 4
    if psutil.virtual_memory().available < 1.5 * (in_bytes + out_bytes):
        return {"value": None, "unit": UNIT, "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": valid_out_bytes,
                "note": "skipped: not enough host memory to pin the buffers"}
    # free the device-resident copies so that the plan's own staging buffers fit comfortably
    xh = torch.empty(x.shape, dtype=x.dtype, pin_memory=True)
    xh.copy_(x)
    oh = torch.empty(out.shape, dtype=out.dtype, pin_memory=True)
    call, how = plan.execute_host, "ddsp_execute_host (copy in, kernel, copy out in sequence)"
    call(xh, oh)                                   # warm-up: allocates the staging buffers
    torch.cuda.synchronize()
    multi.barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        call(xh, oh)                               # synchronises before returning
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    rate, t_max = multi.job_throughput(adds * steps, dt)
    same = bool(torch.equal(oh[:, :plan.nsamp_out], out[:, :plan.nsamp_out].cpu()))
    return {"value": rate / 1e9, "unit": UNIT, "h2d_bytes_per_step": in_bytes,
            "d2h_bytes_per_step": valid_out_bytes, "steps": steps, "ms_per_step": t_max / steps * 1e3,
            "x_realtime": plan.nsamp_out * wl.tsamp * wl.downsample / (t_max / steps),
            "matches_device_result": same, "call": how}


# ----------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on the host cores (rank 0 only)
# ----------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return None
    import torch
    from oracle import oracle
    from paper_2511_02328_b200 import synth
    oracle.build()
    wl = get_workload(args)
    table, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    nout = oracle.nsamp_ds(wl.nsamp, wl.downsample) - dmax
    nch_un = wl.nchan - (0 if wl.mask is None else int(wl.mask.sum()))
    # bounded sample per step: 8 evenly spaced trials, all channels, a window of the observation
    rows = np.unique(np.linspace(0, wl.ndm - 1, 8).round().astype(np.int64))
    ncol = int(min(nout, max(1024, 4e9 / (len(rows) * max(1, nch_un)))))
    win = wl.cropped(min(wl.nsamp, (ncol + dmax) * wl.downsample))
    xh = synth.make_input(win, "cpu", native_delays=lambda dm: oracle.delay_table(
        wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, [dm], 1)[0][0], nsamp_out=nout).numpy()
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.dedisperse_table(xh, table[rows], nsamp=win.nsamp, downsample=wl.downsample, mask=wl.mask,
                                t_lo=0, t_hi=ncol)
        if it >= args.warmup:
            times.append(time.perf_counter() - t0)
    adds = float(len(rows)) * nch_un * ncol
    secs = sum(times)
    value = adds * args.steps / secs / 1e9
    sample = "%d trials x %d channels x %d output samples per step" % (len(rows), nch_un, ncol)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u32" if wl.dtype == "u8" else "f32", "data": "synthetic",
            "config": {"workload": wl.name, "nchan": wl.nchan, "ndm": wl.ndm, "nsamp": wl.nsamp,
                       "sample": sample},
            "gpu_launches": 0,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return line


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
