"""Plan-time tables of the lanes kernels at the FULL size of every
BASELINE.json config, checked on the CPU against the oracle's delay table.

The emulation (tests/test_emulated_cpu.py) runs the kernels on cropped problems; what it cannot run is the real
problem size.  Everything that decides whether a full-size launch stays inside its buffers is decided on the
host at plan time, so it is checked here, entry for entry:

  * every staged row window lies inside its interleaved row for every time tile, is no longer than a stage row,
    starts and ends on 16 bytes (the copy engine's rule);
  * every (row, trial) offset is exactly (delay - window start) words into its stage row, and the furthest
    shared-memory read of any thread (offset + 512 words) ends inside the staged window;
  * the ring fits in shared memory with at least 3 stages;
  * segments cover the output, the workspace size is the one the library reports.

The tables come from the test build of the library (tests/emu, -DDDSP_TESTING: include/ddsp_testing.h); expected
values from oracle/ only.
"""
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

GEOM = ("kind", "W", "WB", "bdm", "TW", "C", "nblk", "nchunk", "RS", "NS", "stage_bytes", "smem_bytes", "flush_rows",
        "NT", "Q", "M")


@pytest.fixture(scope="module")
def emu():
    lib = ctypes.CDLL(build_emu.build())
    for name, (res, args) in binding.SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    vp = ctypes.c_void_p
    lib.ddsp_testing_lanes_geometry.argtypes = [vp, vp]
    lib.ddsp_testing_lanes_tables.argtypes = [vp, vp, vp, vp]
    return lib


def lanes_tables(emu, wl):
    dm = np.ascontiguousarray(wl.dm_list, dtype=np.float64)
    mask = None if wl.mask is None else np.ascontiguousarray(wl.mask, dtype=np.uint8)
    h = ctypes.c_void_p()
    rc = emu.ddsp_plan_create(ctypes.byref(h), wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp, dm.ctypes.data,
                              dm.size, wl.downsample, mask.ctypes.data if mask is not None else None,
                              binding.DDSP_IN_U8 if wl.dtype == "u8" else binding.DDSP_IN_F32)
    assert rc == 0, rc
    try:
        geom = np.zeros(16, dtype=np.int64)
        assert emu.ddsp_testing_lanes_geometry(h, geom.ctypes.data) == 0
        g = dict(zip(GEOM, (int(v) for v in geom)))
        win = np.zeros((g["nblk"], g["nchunk"] * g["C"], 2), dtype=np.int32)
        off = np.zeros((g["nblk"], g["nchunk"], g["C"], g["bdm"]), dtype=np.uint32)
        rows = np.zeros((g["nblk"], g["bdm"]), dtype=np.int32)
        assert emu.ddsp_testing_lanes_tables(h, win.ctypes.data, off.ctypes.data, rows.ctypes.data) == 0
        assert emu.ddsp_plan_set_kernel(h, binding.DDSP_KERNEL_LANES) == 0
        g["ws_bytes"] = int(emu.ddsp_plan_workspace_bytes(h))
        g["nsamp_out"] = int(emu.ddsp_plan_nsamp_out(h))
        g["dmax"] = int(emu.ddsp_plan_max_delay(h))
        return g, win, off, rows
    finally:
        emu.ddsp_plan_destroy(h)


def check_tables(oracle, wl, g, win, off, rows):
    table, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    nout = oracle.nsamp_ds(wl.nsamp, wl.downsample) - dmax
    chans = np.arange(wl.nchan) if wl.mask is None else np.flatnonzero(np.asarray(wl.mask) == 0)
    nlist, ndm = len(chans), wl.ndm
    W, WB, B, TW, C, RS = g["W"], g["WB"], g["bdm"], g["TW"], g["C"], g["RS"]
    kind = 2 if wl.dtype == "f32" else (0 if wl.downsample == 1 else 1)
    assert (g["kind"], W, WB) == [(0, 8, 8), (1, 8, 16), (2, 4, 16)][kind]
    assert (B, TW, C) == (16, 512, 4)

    # geometry: segments cover the output; the ring fits
    assert g["nsamp_out"] == nout and g["dmax"] == dmax
    assert g["nblk"] == -(-ndm // B) and g["nchunk"] == -(-nlist // C)
    assert g["Q"] == g["NT"] * TW and g["Q"] * W >= nout and (g["NT"] - 1) * TW * W < max(nout, 1)
    assert g["M"] >= g["Q"] + dmax and (g["M"] * WB) % 16 == 0
    assert g["ws_bytes"] == max(nlist, 1) * g["M"] * WB
    assert RS % 16 == 0 and g["stage_bytes"] == C * RS + C * B * 4 and g["stage_bytes"] % 16 == 0
    assert 3 <= g["NS"] <= 8 and g["smem_bytes"] == 1024 + g["NS"] * g["stage_bytes"] <= 232448
    assert g["flush_rows"] >= C
    if kind == 0:
        assert g["flush_rows"] * 255 <= 65535
    if kind == 1:
        assert g["flush_rows"] * 255 * wl.downsample <= 65535 < (g["flush_rows"] + 1) * 255 * wl.downsample

    # rows: trials sorted by DM (stable), -1 padding
    order = np.argsort(np.asarray(wl.dm_list), kind="stable")
    want_rows = np.full(g["nblk"] * B, -1, dtype=np.int64)
    want_rows[:ndm] = order
    assert np.array_equal(rows.reshape(-1), want_rows)

    # windows and offsets, block by block (vectorised over channels)
    lpad = g["nchunk"] * C
    for b in range(g["nblk"]):
        tr = want_rows[b * B:(b + 1) * B].copy()
        tr[tr < 0] = order[ndm - 1]                       # padding trials repeat the last one
        d = table[tr][:, chans].astype(np.int64)          # [B][nlist]
        lo = d.min(axis=0)
        hi = d.max(axis=0)
        if WB == 8:
            lo = lo & ~1
        words = TW + (hi - lo)
        if WB == 8:
            words = (words + 1) & ~1
        assert np.array_equal(win[b, :nlist, 0], lo), b
        assert np.array_equal(win[b, :nlist, 1], words), b
        assert not win[b, nlist:].any()
        assert (lo >= 0).all() and (words * WB <= RS).all()
        assert ((lo * WB) % 16 == 0).all() and ((words * WB) % 16 == 0).all()
        assert ((g["NT"] - 1) * TW + lo + words <= g["M"]).all()            # last tile's window inside the row
        slot = (np.arange(nlist) % C) * RS
        want_off = slot[None, :] + (d - lo[None, :]) * WB                     # [B][nlist]
        got_off = off[b].reshape(lpad, B)[:nlist].T.astype(np.int64)          # [B][nlist]
        assert np.array_equal(got_off, want_off), b
        # furthest read of any thread of the tile: word (TW - 1) of the trial's shifted row
        assert (got_off + TW * WB <= slot[None, :] + words[None, :] * WB).all()
    return RS


@pytest.mark.parametrize("name", synth.CONFIG_NAMES)
def test_lanes_tables_full_size(emu, oracle, name):
    wl = synth.config(name)
    g, win, off, rows = lanes_tables(emu, wl)
    check_tables(oracle, wl, g, win, off, rows)


def test_lanes_tables_unsorted_duplicates_and_mask(emu, oracle):
    wl = synth.Workload("t", 1, 37, 1500.0, -4.0, 1e-3, 5003, np.linspace(0.0, 60.0, 23))
    rng = np.random.default_rng(5)
    wl.dm_list = np.concatenate([rng.permutation(wl.dm_list), [wl.dm_list[7], wl.dm_list[7], 0.0]])
    wl.mask = (rng.random(37) < 0.3).astype(np.uint8)
    g, win, off, rows = lanes_tables(emu, wl)
    check_tables(oracle, wl, g, win, off, rows)


def test_lanes_stage_sizes_of_the_configs(emu, oracle):
    """The ring depth DESIGN.md section 6 quotes for each config follows from the delay spread of 16 trials."""
    depth = {}
    for name in ("fast", "wide", "lowfreq", "rfids"):
        g, _, _, _ = lanes_tables(emu, synth.config(name))
        depth[name] = (g["RS"], g["NS"])
    assert depth["fast"][1] >= 5 and depth["wide"][1] == 8 and depth["lowfreq"][1] >= 4 and depth["rfids"][1] >= 4, depth
