#!/usr/bin/env python
"""bench.py -- headline measurement of the dedispersion hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config fast] [--kernel auto|direct|tiled|lanes]
    python bench.py --impl reference ...          # the CPU oracle on the host cores, same metric

A "step" is one pass of the whole hot path (ddsp_execute: stage, fused bin-sum, shifted accumulate,
write-out) over one synthetic observation.  At N = 1 the workload is BASELINE.json configs[1]
("FAST-like": 2048 channels, 150 s, 1001 DM trials).  With N > 1 (torchrun, one rank per GPU) every
rank dedisperses its own observation of that shape -- independent units, no collective on the data
path (weak scaling).  One JSON line is printed by rank 0.

The kernel that runs is the LIBRARY's choice (`--kernel auto` = ddsp's AUTO); bench.py never picks, races or
sweeps kernels.  A result that differs from the oracle on the compared sample, or an end-to-end result that
differs from the device result, prints an error line and exits non-zero: a wrong kernel publishes no number.
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
KERNEL_IDS = {"auto": 0, "direct": 1, "tiled": 2, "lanes": 3}
KERNEL_NAMES = {1: "direct", 2: "tiled", 3: "lanes"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="fast", help="workload name (synth.CONFIG_NAMES); headline = fast")
    ap.add_argument("--kernel", default="auto", choices=sorted(KERNEL_IDS))
    ap.add_argument("--split", default="obs", choices=["obs", "dm"],
                    help="N > 1: 'obs' = one whole observation per GPU (weak scaling, no exchange); 'dm' = ONE "
                         "observation, DM rows sharded over the GPUs after one NCCL broadcast of the input (strong)")
    ap.add_argument("--crop", type=int, default=0, help="debug: crop to this many output samples")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
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
    return synth.config(args.config)


def adds_per_execute(plan):
    return float(plan.ndm) * float(plan.nchan_unmasked) * float(plan.nsamp_out)


def cpu_model():
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_sample(wl, x, nout, dmax, nch_un, ntrials, target_adds, row_range=None):
    """Bounded sample of the same workload for the CPU oracle: all channels, `ntrials` evenly spaced trials (of
    this rank's row range), the first `ncol` output columns.  Returns (rows, ncol, host input window)."""
    lo, cnt = (0, wl.ndm) if row_range is None else row_range
    rows = np.unique(np.linspace(lo, lo + cnt - 1, ntrials).round().astype(np.int64))
    ncol = int(min(nout, max(1024, target_adds / (len(rows) * max(1, nch_un)))))
    ncols_in = min(wl.nsamp, (ncol + dmax) * wl.downsample)
    xh = x[:, :ncols_in]
    xh = xh.cpu().numpy() if hasattr(xh, "cpu") else np.ascontiguousarray(xh)
    return rows, ncol, np.ascontiguousarray(xh)


def run_oracle(wl, table, rows, ncol, xh, nthreads):
    """The oracle as it stands (a single-threaded C++ triple loop) on the sample.  nthreads > 1: the SAME
    function is called on disjoint DM-row ranges from one thread per host core (SURVEY.md 8(d) 'all-core
    figure'); ctypes releases the GIL.  Returns (seconds, output, adds, threads used)."""
    from oracle import oracle
    parts = [p for p in np.array_split(np.arange(len(rows)), nthreads) if len(p)]
    outs = [None] * len(parts)

    def work(k):
        outs[k] = oracle.dedisperse_table(xh, table[rows[parts[k]]], nsamp=xh.shape[1], downsample=wl.downsample,
                                          mask=wl.mask, t_lo=0, t_hi=ncol)
    threads = [threading.Thread(target=work, args=(k,)) for k in range(len(parts))]
    t0 = time.perf_counter()
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    dt = time.perf_counter() - t0
    nch_un = wl.nchan - (0 if wl.mask is None else int(wl.mask.sum()))
    return dt, np.concatenate(outs, axis=0), float(len(rows)) * nch_un * ncol, len(parts)


def profile_traffic(kernel, config):
    """dram bytes per launch of the dominant kernel from the committed ncu summary (profiles/traffic.json, written
    by paper_2511_02328_b200/ncu_summary.py from `ncu --page raw --csv`), or None if that kernel / config has no
    capture yet."""
    try:
        table = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    except (OSError, ValueError):
        return None, None
    e = table.get("%s/%s" % (kernel, config))
    return (float(e["dram_bytes_per_launch"]), e.get("source")) if e else (None, None)


def fail(what, **kw):
    print(json.dumps(dict({"metric": METRIC, "value": None, "unit": UNIT, "error": what}, **kw)))
    sys.stdout.flush()
    sys.exit(3)


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
    split_dm = args.split == "dm" and world > 1
    rows = None
    if split_dm:
        # ONE observation; rank r computes the contiguous DM-row range shard_rows(ndm, r, world)
        rows = multi.shard_rows(wl.ndm, rank, world)
        if rows[1] < 1:
            raise SystemExit("bench.py: more ranks than DM rows")
    else:
        # every rank owns whole observations (units); rank r's observation uses seed + 1000 r
        unit = list(multi.shard_units(world, rank, world))[0]
        wl.seed = wl.seed + 1000 * unit

    rows_of_rank, row0 = rows, (rows[0] if rows else 0)
    plan = binding.plan_for(wl, rows=rows)
    in_pitch = synth.round_up(wl.nsamp, 128)
    out_pitch = synth.round_up(plan.nsamp_out, 32)
    plan.set_pitch(in_pitch, out_pitch)
    plan.set_kernel(KERNEL_IDS[args.kernel])          # "auto": the library's AUTO, nothing else
    kernel = KERNEL_NAMES[plan.kernel]
    if split_dm and rank != 0:
        x = torch.empty((wl.nchan, in_pitch), dtype=wl.torch_dtype, device=dev)
    else:
        x = synth.make_input(wl, dev, pitch=in_pitch, native_delays=library_native_delays(wl),
                             nsamp_out=plan.nsamp_out)
    bcast_ms = None
    if split_dm:                                      # the path's only exchange step: one broadcast of the input
        torch.cuda.synchronize(dev)
        multi.barrier()
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b0.record()
        multi.broadcast_input(x, src=0)
        b1.record()
        torch.cuda.synchronize(dev)
        bcast_ms = multi.max_over_ranks(b0.elapsed_time(b1))
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
    status = plan.device_status()
    if status != 0:
        fail("device status %d after the timed region (1: a bounded barrier wait ran out, 2: table bounds check)"
             % status, kernel=kernel)

    total_rate, t_max = multi.job_throughput(adds * args.steps, secs)      # adds/s over all ranks
    ms_per_step = t_max / args.steps * 1e3

    # end to end through the public host-buffer call (H2D + kernels + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        e2e = measure_e2e(plan, wl, x, out, adds, min(args.steps, 3), multi)
        if e2e.get("matches_device_result") is False:
            fail("end-to-end result differs from the device result", kernel=kernel)

    result = None
    if rank == 0:
        p_add = SM_COUNT * ADDS_PER_CLK_SM * SM_MAX_MHZ * 1e6                 # adds/s
        achieved = adds / (secs / args.steps)
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except (OSError, ValueError):
            pass
        hbm = float(peaks.get("hbm_gbs", 6650.0)) * 1e9
        ideal_bytes = float(wl.nchan) * wl.nsamp * wl.elem_size + float(plan.ndm) * plan.nsamp_out * 4
        t_roof = max(ideal_bytes / hbm, adds / p_add)
        traffic, traffic_src = profile_traffic(kernel, wl.name)
        result = {
            "metric": METRIC, "value": total_rate / 1e9, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "strong" if split_dm else "weak", "vs_baseline": None,
            "dtype": "u32" if wl.dtype == "u8" else "f32", "data": "synthetic",
            "config": {"workload": "%s%s" % (wl.name, "" if not args.crop else "(cropped)"),
                       "nchan": wl.nchan, "nchan_unmasked": plan.nchan_unmasked, "ndm": plan.ndm,
                       "nsamp": wl.nsamp, "nsamp_out": plan.nsamp_out, "tsamp_s": wl.tsamp,
                       "downsample": wl.downsample, "in_dtype": wl.dtype, "kernel": kernel,
                       "launches_per_execute": plan.launches_per_execute,
                       "workspace_bytes": plan.workspace_bytes,
                       "units": "DM rows of one observation per GPU" if split_dm else "one observation per GPU",
                       "parallelism": ("dm-rows%d" if split_dm else "dp%d") % world,
                       "input_broadcast_ms": bcast_ms,
                       "l2": "inputs (%.2f GB) larger than L2; no flush" % (x.numel() * x.element_size() / 1e9)},
            "x_realtime": plan.nsamp_out * wl.tsamp * wl.downsample / (t_max / args.steps),
            "gpu_launches": args.steps * plan.launches_per_execute,
            "clocks": clocks,
            "roofline": {"bound": "alu", "achieved": achieved / 1e9, "peak": p_add / 1e9, "unit": "Gadd/s",
                         "frac": achieved / p_add, "traffic": traffic, "traffic_source": traffic_src,
                         "peak_source": "148 SM x 128 32-bit integer adds/clk/SM x 1965 MHz (DESIGN.md 6.6; issue "
                                        "rates: paper_2511_02328_b200/ubench.py, table in profiles/)",
                         "execute_ms": secs / args.steps * 1e3,
                         "t_roof_ms": t_roof * 1e3, "frac_of_path_roofline": t_roof / (secs / args.steps),
                         "hbm_ideal_bytes": ideal_bytes, "hbm_peak_gbs": hbm / 1e9,
                         "hbm_peak_source": "measured" if peaks else "fallback"},
            "e2e": e2e,
        }
        if not args.no_cpu_baseline:
            from oracle import oracle
            table, dmax_o = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
            assert dmax_o == plan.max_delay        # also in a DM-row split: d_max is the whole list's
            ncores = host_cores()
            # (i) one thread, 8 evenly spaced trials: also the parity sample of the timed launch configuration
            rows, ncol, xh = oracle_sample(wl, x, plan.nsamp_out, plan.max_delay, plan.nchan_unmasked, 8, 1.6e10, rows_of_rank)
            dt1, oout, oadds1, _ = run_oracle(wl, table, rows, ncol, xh, 1)
            got = out[torch.as_tensor(rows - row0, device=dev), :ncol].cpu().numpy()
            if wl.dtype == "u8":
                ok = bool(np.array_equal(got.view(np.uint32), oout))
            else:
                ok = bool((np.abs(got.astype(np.float64) - oout) <= 1e-5 * np.abs(oout)).all())
            if not ok:
                fail("the CUDA result differs from the oracle on the sample (%d trials x first %d columns)"
                     % (len(rows), ncol), kernel=kernel)
            # (ii) all cores: the same function on disjoint DM-row ranges, one thread per core
            rows_n, ncol_n, xh_n = oracle_sample(wl, x, plan.nsamp_out, plan.max_delay, plan.nchan_unmasked,
                                                 max(8, 4 * ncores), 1.2e10 * max(1, ncores) ** 0.5)
            dtn, _, oaddsn, used = run_oracle(wl, table, rows_n, ncol_n, xh_n, ncores)
            result["cpu_baseline"] = {
                "value": oaddsn / dtn / 1e9, "unit": UNIT, "cores": used, "kind": "oracle", "cpu": cpu_model(),
                "sample": "%d trials x %d channels x first %d output samples of the same input, the unchanged "
                          "single-threaded oracle on disjoint DM rows in %d threads (%.1f s)"
                          % (len(rows_n), plan.nchan_unmasked, ncol_n, used, dtn),
                "single_thread": {"value": oadds1 / dt1 / 1e9, "cores": 1,
                                  "sample": "%d trials x %d channels x first %d output samples (%.1f s)"
                                            % (len(rows), plan.nchan_unmasked, ncol, dt1)},
                "parity_on_sample": "ok"}
        print(json.dumps(result))
        sys.stdout.flush()
    plan.destroy()
    multi.finalize()
    return result


def measure_e2e(plan, wl, x, out, adds, steps, multi):
    """Same metric through ddsp_execute_host: pinned host input -> device, kernels, result -> pinned host."""
    import psutil
    import torch
    in_bytes = x.numel() * x.element_size()
    out_bytes = out.numel() * 4
    valid_out_bytes = plan.ndm * plan.nsamp_out * 4
    if psutil.virtual_memory().available < 1.5 * (in_bytes + out_bytes):
        return {"value": None, "unit": UNIT, "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": valid_out_bytes,
                "note": "skipped: not enough host memory to pin the buffers"}
    xh = torch.empty(x.shape, dtype=x.dtype, pin_memory=True)
    xh.copy_(x)
    oh = torch.empty(out.shape, dtype=out.dtype, pin_memory=True)
    call, how = plan.execute_host, "ddsp_execute_host (copy in, kernels, copy out in sequence)"
    if KERNEL_NAMES[plan.kernel] == "lanes":       # the kernels that can be launched on a run of output columns
        call = lambda a, b: plan.execute_host_pipelined(a, b, npieces=16)
        how = "ddsp_execute_host_pipelined (16 runs of output columns; copy in, kernels, copy out overlapped)"
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
    from oracle import oracle
    from paper_2511_02328_b200 import synth
    oracle.build()
    wl = get_workload(args)
    table, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    nout = oracle.nsamp_ds(wl.nsamp, wl.downsample) - dmax
    nch_un = wl.nchan - (0 if wl.mask is None else int(wl.mask.sum()))
    ncores = host_cores()
    # bounded sample per step: evenly spaced trials (4 per core), all channels, a window of the observation
    rows = np.unique(np.linspace(0, wl.ndm - 1, max(8, 4 * ncores)).round().astype(np.int64))
    ncol = int(min(nout, max(1024, 4e9 * max(1, ncores) ** 0.5 / (len(rows) * max(1, nch_un)))))
    win = wl.cropped(min(wl.nsamp, (ncol + dmax) * wl.downsample))
    xh = synth.make_input(win, "cpu", native_delays=lambda dm: oracle.delay_table(
        wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, [dm], 1)[0][0], nsamp_out=nout).numpy()
    times, used, adds = [], 1, 0.0
    for it in range(args.warmup + args.steps):
        dt, _, adds, used = run_oracle(wl, table, rows, ncol, xh, ncores)
        if it >= args.warmup:
            times.append(dt)
    secs = sum(times)
    value = adds * args.steps / secs / 1e9
    sample = "%d trials x %d channels x %d output samples per step, %d threads" % (len(rows), nch_un, ncol, used)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u32" if wl.dtype == "u8" else "f32", "data": "synthetic",
            "config": {"workload": wl.name, "nchan": wl.nchan, "ndm": wl.ndm, "nsamp": wl.nsamp,
                       "sample": sample},
            "gpu_launches": 0,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "cpu": cpu_model(),
                             "sample": sample},
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
