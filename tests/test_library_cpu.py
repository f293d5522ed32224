"""CPU-side checks of libddsp (no kernel launches): the library builds and loads, exports every symbol
include/ddsp.h declares, validates arguments, and its plan-time delay table (computed by the library's
own host code) equals the oracle's table entry for entry on all five BASELINE.json configs."""
import os
import re

import numpy as np
import pytest

from paper_2511_02328_b200 import binding, build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def test_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "ddsp.h")).read()
    declared = set(re.findall(r"DDSP_API[^;(]*?\b(ddsp_\w+)\s*\(", header))
    assert len(declared) >= 15
    assert declared == set(binding.SIGNATURES), declared ^ set(binding.SIGNATURES)
    for name in declared:
        assert hasattr(lib, name), name
    assert binding.version().startswith("ddsp")


def test_strerror_codes(lib):
    msgs = {lib.ddsp_strerror(c).decode() for c in range(6)}
    assert len(msgs) == 6 and "ok" in msgs
    assert lib.ddsp_strerror(99).decode().startswith("unknown")


@pytest.mark.parametrize("name", synth.CONFIG_NAMES)
def test_plan_delay_table_equals_oracle(lib, oracle, name):
    wl = synth.config(name)
    want, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    with binding.plan_for(wl) as plan:
        got = plan.get_delays()
        assert np.array_equal(got, want)
        assert plan.max_delay == dmax
        assert plan.nsamp_out == oracle.nsamp_ds(wl.nsamp, wl.downsample) - dmax
        assert plan.nchan_unmasked == wl.nchan - (0 if wl.mask is None else int(wl.mask.sum()))
        assert plan.launches_per_execute >= 1


def test_dm_list_order_is_preserved_in_table(lib, oracle):
    dms = np.array([30.0, 0.0, 12.5, 30.0, 7.0])
    want, _ = oracle.delay_table(64, 1500.0, -2.0, 1e-3, dms, 1)
    with binding.Plan(64, 1500.0, -2.0, 1e-3, 4096, dms) as plan:
        assert np.array_equal(plan.get_delays(), want)


def _create(lib, **kw):
    import ctypes
    a = dict(nchan=8, f_top=1500.0, chan_bw=-10.0, tsamp=1e-3, nsamp=1000, dm=[0.0, 1.0], ds=1,
             mask=None, dtype=0)
    a.update(kw)
    dm = np.asarray(a["dm"], dtype=np.float64)
    h = ctypes.c_void_p()
    mask = None if a["mask"] is None else np.asarray(a["mask"], dtype=np.uint8)
    code = lib.ddsp_plan_create(ctypes.byref(h), a["nchan"], a["f_top"], a["chan_bw"], a["tsamp"], a["nsamp"],
                                dm.ctypes.data if dm.size else None, int(dm.size), a["ds"],
                                mask.ctypes.data if mask is not None else None, a["dtype"])
    if code == 0:
        lib.ddsp_plan_destroy(h)
    else:
        assert not h.value
    return code


def test_invalid_arguments(lib):
    E = binding.DDSP_ERR_INVALID_ARG
    assert _create(lib) == 0
    assert _create(lib, nchan=0) == E
    assert _create(lib, dm=[]) == E
    assert _create(lib, ds=0) == E
    assert _create(lib, chan_bw=0.0) == E
    assert _create(lib, chan_bw=2.0) == E          # ascending band rejected (R12)
    assert _create(lib, tsamp=0.0) == E
    assert _create(lib, tsamp=float("nan")) == E
    assert _create(lib, dm=[0.0, -1.0]) == E
    assert _create(lib, dm=[0.0, float("inf")]) == E
    assert _create(lib, dtype=7) == E
    assert _create(lib, nsamp=0) == E
    assert _create(lib, nchan=200, chan_bw=-10.0) == E   # lowest channel frequency <= 0
    assert lib.ddsp_plan_create(None, 8, 1500.0, -1.0, 1e-3, 100, None, 1, 1, None, 0) == E
    assert lib.ddsp_plan_destroy(None) == 0
    assert lib.ddsp_plan_nsamp_out(None) == -1
    assert lib.ddsp_execute(None, None, None, None) == E


def test_no_output_error(lib):
    # DM 1000 across 1000..1500 MHz at 1 ms is ~2300 samples of delay: nsamp = 1000 leaves nothing
    assert _create(lib, nchan=64, chan_bw=-7.8125, dm=[1000.0], nsamp=1000) == binding.DDSP_ERR_NO_OUTPUT
    assert _create(lib, nchan=64, chan_bw=-7.8125, dm=[1000.0], nsamp=10000) == 0


def test_pitch_validation(lib):
    with binding.Plan(8, 1500.0, -10.0, 1e-3, 1000, [0.0, 5.0]) as plan:
        nout = plan.nsamp_out
        plan.set_pitch(1024, nout + 3)
        with pytest.raises(binding.DdspError):
            plan.set_pitch(999, nout)
        with pytest.raises(binding.DdspError):
            plan.set_pitch(1000, nout - 1)
        with pytest.raises(binding.DdspError):
            plan.set_kernel(42)


def test_execute_without_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with binding.Plan(8, 1500.0, -10.0, 1e-3, 1000, [0.0, 5.0]) as plan:
        x = np.zeros((8, 1000), dtype=np.uint8)
        out = np.zeros((2, plan.nsamp_out), dtype=np.uint32)
        with pytest.raises(binding.DdspError) as ei:
            plan.execute_ptr(x.ctypes.data, out.ctypes.data, 0)
        assert ei.value.code == binding.DDSP_ERR_CUDA
        assert not out.any()          # nothing was computed on the CPU


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2511_02328_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "oracle_ddsp" not in text and "liboracle" not in text, f


def test_plan_rows_is_a_row_range_of_the_whole_plan(lib, oracle):
    """ddsp_plan_create_rows: the delay table is the row range, d_max and nsamp_out are the whole
    list's (invariant I7), whatever the range."""
    wl = synth.config("tiny")
    want, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, 1)
    for begin, count in ((0, 201), (0, 50), (50, 100), (200, 1), (13, 16)):
        with binding.plan_for(wl, rows=(begin, count)) as plan:
            assert plan.ndm == count
            assert np.array_equal(plan.get_delays(), want[begin:begin + count])
            assert plan.max_delay == dmax and plan.nsamp_out == wl.nsamp - dmax
    for bad in ((-1, 5), (0, 0), (200, 2), (201, 1)):
        with pytest.raises(binding.DdspError):
            binding.plan_for(wl, rows=bad)


def test_lanes_declines_what_its_32_bit_counters_cannot_hold(lib):
    """More than 2**31 output columns: the lanes kernels say UNSUPPORTED at plan time (AUTO falls back), they do not
    fail at launch."""
    with binding.Plan(2, 1500.0, -10.0, 1e-3, 3 * 2 ** 30, [0.0, 1.0]) as plan:
        with pytest.raises(binding.DdspError) as ei:
            plan.set_kernel(binding.DDSP_KERNEL_LANES)
        assert ei.value.code == binding.DDSP_ERR_UNSUPPORTED
        assert plan.kernel in (binding.DDSP_KERNEL_DIRECT, binding.DDSP_KERNEL_TILED)
    with binding.Plan(2, 1500.0, -10.0, 1e-3, 2 ** 20, [0.0, 1.0]) as plan:
        plan.set_kernel(binding.DDSP_KERNEL_LANES)          # host-only plan: geometry exists, nothing is allocated
        assert plan.kernel == binding.DDSP_KERNEL_LANES and plan.workspace_bytes > 0
        assert plan.launches_per_execute == 2
