"""TEST INFRASTRUCTURE -- ctypes front end of the CPU oracle (oracle_ddsp.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It never imports the CUDA package and the CUDA package never
imports it.  All arithmetic of the method lives in oracle_ddsp.cpp, which follows
PAPER.md:95-99, 111, 121, 158 (Eq. 4, Eq. 5, the shifted sum over frequency); this
file only marshals numpy arrays.

Parity status: pinned (see tests/test_oracle_pins.py).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_ddsp.cpp")
_LIB = os.path.join(_HERE, "liboracle_ddsp.so")
_lib = None

CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]


def build(force=False):
    """Compile the oracle with g++ (plain C++, single thread, no intrinsics)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["g++"] + CXXFLAGS + ["-o", tmp, _SRC])
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    i32, i64, f64, vp = ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
    lib.oracle_nsamp_ds.restype = i64
    lib.oracle_nsamp_ds.argtypes = [i64, i32]
    lib.oracle_delay_table.restype = i64
    lib.oracle_delay_table.argtypes = [i32, f64, f64, f64, i32, vp, i32, vp]
    for name in ("oracle_dedisperse_u8", "oracle_dedisperse_f32", "oracle_dedisperse_f32_acc64"):
        fn = getattr(lib, name)
        fn.restype = i32
        fn.argtypes = [vp, i32, i64, i64, i32, vp, vp, i32, i64, i64, vp, i64]
    _lib = lib
    return lib


def nsamp_ds(nsamp, downsample=1):
    return int(_load().oracle_nsamp_ds(int(nsamp), int(downsample)))


def delay_table(nchan, f_top, chan_bw, tsamp, dm_list, downsample=1):
    """int32 [ndm][nchan] delay table and d_max (over all channels)."""
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    out = np.empty((dm.size, nchan), dtype=np.int32)
    dmax = _load().oracle_delay_table(int(nchan), float(f_top), float(chan_bw), float(tsamp),
                                      int(downsample), dm.ctypes.data, int(dm.size), out.ctypes.data)
    if dmax < 0:
        raise ValueError("oracle_delay_table: invalid arguments")
    return out, int(dmax)


def dedisperse_table(x, delays, nsamp=None, downsample=1, mask=None, t_lo=0, t_hi=None,
                     acc64=False):
    """Shifted sum for an explicit delay table (rows of `delays`), columns [t_lo, t_hi).

    x: (nchan, pitch) uint8 or float32, C-contiguous rows; nsamp valid samples per row.
    `t_hi` must satisfy t_hi + max(delays) <= ceil(nsamp/downsample).
    Returns uint32 (uint8 in), float32 (float32 in) or float64 (float32 in, acc64=True).
    """
    lib = _load()
    x = np.asarray(x)
    assert x.ndim == 2 and x.flags.c_contiguous
    nchan, pitch = x.shape
    nsamp = pitch if nsamp is None else int(nsamp)
    delays = np.ascontiguousarray(delays, dtype=np.int32)
    assert delays.ndim == 2 and delays.shape[1] == nchan
    ndm = delays.shape[0]
    nds = nsamp_ds(nsamp, downsample)
    if t_hi is None:
        raise ValueError("t_hi required")
    if t_hi + int(delays.max(initial=0)) > nds or t_lo < 0 or t_hi < t_lo:
        raise ValueError("window reaches outside the downsampled series")
    m = None
    if mask is not None:
        m = np.ascontiguousarray(mask, dtype=np.uint8)
        assert m.shape == (nchan,)
    n = t_hi - t_lo
    if x.dtype == np.uint8:
        out = np.empty((ndm, n), dtype=np.uint32)
        fn = lib.oracle_dedisperse_u8
    elif x.dtype == np.float32:
        out = np.empty((ndm, n), dtype=np.float64 if acc64 else np.float32)
        fn = lib.oracle_dedisperse_f32_acc64 if acc64 else lib.oracle_dedisperse_f32
    else:
        raise TypeError("oracle supports uint8 and float32 input")
    rc = fn(x.ctypes.data, nchan, nsamp, pitch, int(downsample),
            m.ctypes.data if m is not None else None, delays.ctypes.data, ndm,
            int(t_lo), int(t_hi), out.ctypes.data, n)
    if rc != 0:
        raise ValueError("oracle dedisperse: invalid arguments")
    return out


def dedisperse(x, f_top, chan_bw, tsamp, dm_list, nsamp=None, downsample=1, mask=None,
               acc64=False, rows=None, t_lo=0, t_hi=None):
    """Full definition: delay table from (f_top, chan_bw, tsamp, dm_list), d_max over the
    WHOLE dm_list, nsamp_out = ceil(nsamp/ds) - d_max, then the shifted sum.  `rows`
    optionally selects a subset of DM rows (indices into dm_list) and [t_lo, t_hi) a column
    window, so that full-size outputs can be sampled.  Returns (out, nsamp_out, d_max)."""
    x = np.asarray(x)
    nchan = x.shape[0]
    nsamp = x.shape[1] if nsamp is None else int(nsamp)
    table, dmax = delay_table(nchan, f_top, chan_bw, tsamp, dm_list, downsample)
    nout = nsamp_ds(nsamp, downsample) - dmax
    if nout <= 0:
        raise ValueError("no output: ceil(nsamp/ds) <= d_max")
    if rows is not None:
        table = table[np.asarray(rows, dtype=np.int64)]
    if t_hi is None:
        t_hi = nout
    if t_hi > nout:
        raise ValueError("t_hi beyond nsamp_out")
    out = dedisperse_table(x, table, nsamp=nsamp, downsample=downsample, mask=mask,
                           t_lo=t_lo, t_hi=t_hi, acc64=acc64)
    return out, nout, dmax
