"""Plan-time tables of the tiled kernel at the full size of the uint8
ds = 1 configs, replayed on the CPU against the oracle's delay table: every (channel, trial) offset decodes to the
oracle's delay, every read of the hot loop lies inside the staged units of its phase copy, and the stages fit in
shared memory.  Tables from the test build of the library (tests/emu, -DDDSP_TESTING)."""
import ctypes
import importlib.util
import os

import numpy as np
import pytest

from paper_2511_02328_b200 import binding, synth

HERE = os.path.dirname(os.path.abspath(__file__))
_spec = importlib.util.spec_from_file_location("build_emu", os.path.join(HERE, "emu", "build_emu.py"))
build_emu = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(build_emu)


@pytest.fixture(scope="module")
def emu():
    lib = ctypes.CDLL(build_emu.build())
    for name, (res, args) in binding.SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    vp = ctypes.c_void_p
    lib.ddsp_testing_tiled_geometry.argtypes = [vp, vp]
    lib.ddsp_testing_tiled_tables.argtypes = [vp] * 6
    return lib


@pytest.mark.parametrize("name", ["tiny", "fast", "wide"])
def test_tiled_tables_replay(emu, oracle, name):
    wl = synth.config(name)
    dm = np.ascontiguousarray(wl.dm_list, dtype=np.float64)
    h = ctypes.c_void_p()
    assert emu.ddsp_plan_create(ctypes.byref(h), wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp, dm.ctypes.data,
                                dm.size, 1, None, binding.DDSP_IN_U8) == 0
    try:
        geom = np.zeros(10, dtype=np.int64)
        assert emu.ddsp_testing_tiled_geometry(h, geom.ctypes.data) == 0
        bdm, T, nblk, ntile, cc, nstage, rs, smem, nchunk, npad = (int(v) for v in geom)
        base = np.zeros((nblk, npad), dtype=np.int32)
        nunit = np.zeros((nblk, npad), dtype=np.int32)
        chan = np.zeros(npad, dtype=np.int32)
        off = np.zeros((nblk, npad, bdm), dtype=np.uint32)
        rows = np.zeros((nblk, bdm), dtype=np.int32)
        assert emu.ddsp_testing_tiled_tables(h, base.ctypes.data, nunit.ctypes.data, chan.ctypes.data, off.ctypes.data,
                                             rows.ctypes.data) == 0
    finally:
        emu.ddsp_plan_destroy(h)
    table, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, 1)
    nout = wl.nsamp - dmax
    assert (bdm, T, nstage) == (32, 2048, 2) and nblk == -(-wl.ndm // bdm) and ntile == -(-nout // T)
    assert smem == nstage * cc * (4 * rs + bdm * 4) <= 232448 - 1024 and rs % 16 == 0
    assert nchunk == -(-wl.nchan // cc) and npad == (nchunk + 2) * cc
    assert np.array_equal(chan[:wl.nchan], np.arange(wl.nchan)) and (chan[wl.nchan:] == wl.nchan - 1).all()
    order = np.argsort(np.asarray(wl.dm_list), kind="stable")
    want_rows = np.full(nblk * bdm, -1, dtype=np.int64)
    want_rows[:wl.ndm] = order
    assert np.array_equal(rows.reshape(-1), want_rows)
    for b in range(nblk):
        tr = want_rows[b * bdm:(b + 1) * bdm].copy()
        tr[tr < 0] = order[wl.ndm - 1]
        d = table[tr].astype(np.int64)                       # [bdm][nchan]
        lo = d[0] & ~15                                      # trials are DM-sorted: the first has the smallest delay
        assert (d >= d[0][None, :]).all()
        assert np.array_equal(base[b, :wl.nchan], lo)
        q = d - lo[None, :]
        slot = np.arange(wl.nchan) % cc
        want = (slot[None, :] * 4 + (q & 3)) * rs + (q >> 2) * 4
        assert np.array_equal(off[b, :wl.nchan].T.astype(np.int64), want), b
        # the hot loop reads words (q >> 2) .. (q >> 2) + T/4 - 1 of phase copy q & 3; copy p, unit u is staged from
        # bytes 16 u + p .. 16 u + p + 15 of the window, so the staged units must cover byte q + T - 1 (+ phase)
        need = (q.max(axis=0) + T + 3 + 15) // 16
        assert (nunit[b, :wl.nchan] >= np.minimum(need, rs // 16)).all()
        assert ((q >> 2) * 4 + T <= rs).all()
        assert not nunit[b, wl.nchan:].any()
