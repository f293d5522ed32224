"""Helpers shared by the test modules: seeded inputs, oracle row sampling, comparisons.

The oracle (oracle/) and the CUDA library (paper_2511_02328_b200/) never see each other; only this
test code talks to both.  Expected values always come from the oracle, never from the CUDA path.
"""
import numpy as np
import torch

from paper_2511_02328_b200 import synth


def native_delay_fn(oracle, wl):
    """dm -> int delays on the NATIVE grid (ds = 1), from the oracle's delay table (pulse injection)."""
    def fn(dm):
        return oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, [dm], 1)[0][0]
    return fn


def oracle_geometry(oracle, wl):
    """(delay table, d_max, nsamp_out) of a workload, from the oracle."""
    table, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    return table, dmax, oracle.nsamp_ds(wl.nsamp, wl.downsample) - dmax


def make_input(oracle, wl, device, pitch=None):
    _, _, nout = oracle_geometry(oracle, wl)
    return synth.make_input(wl, device, pitch=pitch, native_delays=native_delay_fn(oracle, wl),
                            nsamp_out=nout)


def crop(oracle, wl, extra_out):
    """Same channels / DM list, nsamp shortened so that nsamp_out == extra_out (exercises every
    (dm, c) delay and the tile edges at a size the oracle can follow)."""
    _, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    return wl.cropped(wl.downsample * (dmax + int(extra_out)))




def assert_u32_equal(got, want, what=""):
    got = np.asarray(got)
    want = np.asarray(want)
    assert got.shape == want.shape, (what, got.shape, want.shape)
    if not np.array_equal(got, want):
        bad = np.argwhere(got != want)
        i = tuple(bad[0])
        raise AssertionError("%s: %d of %d elements differ; first at %s: got %d want %d"
                             % (what, len(bad), got.size, i, got[i], want[i]))


F32_RTOL = 1e-5  # north_star: "within a relative tolerance of 1e-5 per output element for float32 input"


def assert_f32_close(got, want, want64=None, what=""):
    """|g - o| <= 1e-5 |o| against the fp32 sequential oracle (equality passes, so 0 vs 0 passes);
    optionally the order-independent check against the double-accumulated sum (R9)."""
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    assert got.shape == want.shape, (what, got.shape, want.shape)
    assert np.isfinite(got).all(), what + ": non-finite output"
    err = np.abs(got - want)
    bad = err > F32_RTOL * np.abs(want)
    if bad.any():
        i = tuple(np.argwhere(bad)[0])
        raise AssertionError("%s: %d of %d elements beyond rtol 1e-5; first at %s: got %r want %r"
                             % (what, int(bad.sum()), got.size, i, got[i], want[i]))
    if want64 is not None:
        w = np.asarray(want64, dtype=np.float64)
        rms = np.sqrt((w * w).mean(axis=1, keepdims=True))
        bad = np.abs(got - w) > F32_RTOL * np.maximum(np.abs(w), rms)
        assert not bad.any(), "%s: %d elements off the fp64-accumulated sum" % (what, int(bad.sum()))


def run_plan(plan, x, out_fill=None):
    """Execute on the current stream into a fresh (ndm, out_pitch) tensor; returns it (on device)."""
    dt = torch.int32 if plan.in_dtype == 0 else torch.float32   # int32 storage holds the uint32 sums
    out = torch.empty((plan.ndm, plan.out_pitch), dtype=dt, device=x.device)
    if out_fill is not None:
        out.view(torch.int32).fill_(out_fill)
    plan.execute(x, out)
    torch.cuda.synchronize()
    return out


def to_host(out, plan, rows=None, t_lo=0, t_hi=None):
    """Valid columns [t_lo, t_hi) of the selected rows as numpy (uint32 for the u8 path)."""
    t_hi = plan.nsamp_out if t_hi is None else t_hi
    sel = out if rows is None else out[torch.as_tensor(rows, device=out.device)]
    a = sel[:, t_lo:t_hi].contiguous().cpu().numpy()
    return a.view(np.uint32) if plan.in_dtype == 0 else a
