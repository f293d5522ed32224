"""The library's kernels executed on the CPU, thread for thread, through the same C ABI.

tests/emu compiles the kernels' own source with g++ (three textual substitutions, see build_emu.py) against
host stand-ins of the device helpers (csrc/ddsp_dev.cuh -> tests/emu/emu_common.h): one std::thread per CUDA
thread, mbarriers with the PTX counting rules, a copy-engine thread for cp.async.bulk.  What this checks
without a GPU:

  * the result equals the oracle bit for bit (uint8) / in the same fp32 order (float32);
  * the pipeline protocol terminates: no deadlock, no over-arrival, no copy in flight at exit, no bounded wait
    that runs out;
  * EVERY memory access is in range: shared-memory accesses against the CTA's dynamic shared memory, global
    loads / stores / reductions and the SOURCE of every bulk copy against the exact extents of the device
    buffers (the plan's tables and workspace, and the caller's input and output, which are registered at their
    exact size) -- the class of bug that faults a GPU (Xid 13) -- plus the 16-byte rules of cp.async.bulk and the
    alignment of vector accesses.

What it cannot check: the PTX spellings themselves and the speed; the -m gpu tests and bench.py do.
"""
import ctypes
import importlib.util
import os
import subprocess

import numpy as np
import pytest

from paper_2511_02328_b200 import binding, synth

HERE = os.path.dirname(os.path.abspath(__file__))
_spec = importlib.util.spec_from_file_location("build_emu", os.path.join(HERE, "emu", "build_emu.py"))
build_emu = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(build_emu)

LANES, TILED, DIRECT = binding.DDSP_KERNEL_LANES, binding.DDSP_KERNEL_TILED, binding.DDSP_KERNEL_DIRECT


@pytest.fixture(scope="module")
def emu():
    lib = ctypes.CDLL(build_emu.build())
    for name, (res, args) in binding.SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    lib.ddsp_emu_faults.restype = ctypes.c_long
    lib.ddsp_emu_register.argtypes = [ctypes.c_void_p, ctypes.c_size_t]
    lib.ddsp_emu_unregister.argtypes = [ctypes.c_void_p]
    return lib


class DeviceArray:
    """A numpy array registered with the emulator as a device buffer of EXACTLY its size (16-byte aligned
    start unless `misalign`), so that an access one byte outside it is a reported fault."""

    def __init__(self, emu, shape, dtype, fill=None, misalign=0):
        n = int(np.prod(shape)) * np.dtype(dtype).itemsize
        self._raw = np.zeros(n + 320, dtype=np.uint8)
        off = (-self._raw.ctypes.data) % 256 + misalign
        self.a = self._raw[off:off + n].view(dtype).reshape(shape)
        if fill is not None:
            self.a[...] = fill
        self._emu = emu
        emu.ddsp_emu_register(self.a.ctypes.data, n)

    def release(self):
        self._emu.ddsp_emu_unregister(self.a.ctypes.data)


def run_emulated(emu, wl, x, in_pitch, kernel, out_extra=3, misalign=0, expect_faults=False, host_pieces=0):
    dm = np.ascontiguousarray(wl.dm_list, dtype=np.float64)
    mask = None if wl.mask is None else np.ascontiguousarray(wl.mask, dtype=np.uint8)
    h = ctypes.c_void_p()
    rc = emu.ddsp_plan_create(ctypes.byref(h), wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp, dm.ctypes.data,
                              dm.size, wl.downsample, mask.ctypes.data if mask is not None else None,
                              binding.DDSP_IN_U8 if wl.dtype == "u8" else binding.DDSP_IN_F32)
    assert rc == 0, rc
    xin = out = None
    try:
        nout = emu.ddsp_plan_nsamp_out(h)
        out_pitch = nout + out_extra
        assert emu.ddsp_plan_set_pitch(h, in_pitch, out_pitch) == 0
        rc = emu.ddsp_plan_set_kernel(h, kernel)
        if rc == binding.DDSP_ERR_UNSUPPORTED:
            pytest.skip("kernel does not support this plan")
        assert rc == 0, rc
        xin = DeviceArray(emu, x.shape, x.dtype, misalign=misalign)
        xin.a[...] = x
        out = DeviceArray(emu, (wl.ndm, out_pitch), np.uint32 if wl.dtype == "u8" else np.float32, fill=7)
        f0 = emu.ddsp_emu_faults()
        if host_pieces:     # overlapped host-buffer path: the plan's own staging buffers, runs of output columns
            rc = emu.ddsp_execute_host_pipelined(h, xin.a.ctypes.data, out.a.ctypes.data, None, host_pieces)
        else:
            rc = emu.ddsp_execute(h, xin.a.ctypes.data, out.a.ctypes.data, None)
        assert rc == 0, rc
        st = ctypes.c_int(-1)
        assert emu.ddsp_plan_device_status(h, ctypes.byref(st)) == 0
        faults = emu.ddsp_emu_faults() - f0
        if expect_faults:
            return faults, st.value
        assert faults == 0, "the emulator flagged %d fault(s) (see stderr)" % faults
        assert st.value == 0, "device status %d" % st.value
        if out_extra:
            assert (out.a[:, nout:] == 7).all(), "pitch padding was written"
        assert np.array_equal(xin.a, x), "the input was written"
        return out.a[:, :nout].copy(), nout
    finally:
        for d in (xin, out):
            if d is not None:
                d.release()
        emu.ddsp_plan_destroy(h)


def host_input(wl, pitch=None):
    return synth.make_input(wl, "cpu", pitch=pitch).numpy()


def check(emu, oracle, wl, kernel, pitch=None, misalign=0, host_pieces=0):
    pitch = wl.nsamp if pitch is None else pitch
    x = host_input(wl, pitch)
    got, nout = run_emulated(emu, wl, x, pitch, kernel, misalign=misalign, host_pieces=host_pieces)
    want, nout_o, _ = oracle.dedisperse(x, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, nsamp=wl.nsamp,
                                        downsample=wl.downsample, mask=wl.mask)
    assert nout == nout_o
    if wl.dtype == "u8":
        assert np.array_equal(got, want), "%d elements differ" % int((got != want).sum())
    else:   # same order of fp32 additions: bit-identical values (-0.0 == +0.0 numerically)
        assert np.array_equal(got, want), "max abs diff %g" % float(np.abs(got - want).max())


def small(dtype="u8", nchan=21, nsamp=1500, ndm=19, ds=1, seed=3, dm_max=40.0, mask_frac=0.0, tsamp=1e-3):
    wl = synth.Workload("emu", seed, nchan, 1500.0, -6.0, tsamp, nsamp, np.linspace(0.0, dm_max, ndm),
                        downsample=ds, dtype=dtype, mean=128.0 if dtype == "u8" else 0.0,
                        std=40.0 if dtype == "u8" else 1.0)
    if mask_frac > 0:
        wl.mask = (np.random.default_rng(seed).random(nchan) < mask_frac).astype(np.uint8)
    return wl


# ---- every kernel reproduces the oracle ----------------------------------------------------------------------
@pytest.mark.parametrize("kernel", [LANES, TILED, DIRECT], ids=["lanes", "tiled", "direct"])
def test_u8_small(emu, oracle, kernel):
    check(emu, oracle, small(mask_frac=0.2), kernel)


@pytest.mark.parametrize("ds", [2, 3, 4, 8])
@pytest.mark.parametrize("kernel", [LANES, DIRECT], ids=["lanes", "direct"])
def test_u8_downsampled(emu, oracle, kernel, ds):
    """A6: fused bin sum, partial last bin (nsamp mod ds != 0), mask."""
    check(emu, oracle, small(ds=ds, nsamp=1500 * ds + ds - 1, mask_frac=0.2, dm_max=40.0 * ds), kernel)


@pytest.mark.parametrize("ds", [1, 3])
@pytest.mark.parametrize("kernel", [LANES, DIRECT], ids=["lanes", "direct"])
def test_f32(emu, oracle, kernel, ds):
    check(emu, oracle, small(dtype="f32", ds=ds, nsamp=1300 * ds + 1, mask_frac=0.2, dm_max=30.0 * ds), kernel)


# ---- lanes kernel: protocol and geometry corner cases ----------------------------------------------------------
def test_lanes_ring_wraps_and_flushes(emu, oracle):
    """More chunks than ring stages, more than 256 channels (several flushes of the 16-bit lanes: store first,
    reduction afterwards), an odd channel count (last chunk of 1 row)."""
    wl = small(nchan=261, nsamp=900, ndm=5, dm_max=6.0, seed=5)
    wl.chan_bw = -0.5
    check(emu, oracle, wl, LANES)


def test_lanes_all_255_headroom(emu, oracle):
    """I10: x = 255 everywhere over 600 channels, ds = 4: 16-bit lanes would overflow without the flushes."""
    wl = synth.Workload("sat", 0, 600, 1500.0, -0.25, 64e-6, 4 * 700, np.arange(0, 3, dtype=np.float64) * 4.0,
                        downsample=4)
    x = np.full((wl.nchan, wl.nsamp), 255, dtype=np.uint8)
    got, _ = run_emulated(emu, wl, x, wl.nsamp, LANES)
    assert got.min() == got.max() == 600 * 4 * 255
    wl1 = synth.Workload("sat1", 0, 600, 1500.0, -0.25, 64e-6, 700, np.arange(0, 3, dtype=np.float64) * 4.0)
    got, _ = run_emulated(emu, wl1, x[:, :700].copy(), 700, LANES)
    assert got.min() == got.max() == 600 * 255


@pytest.mark.parametrize("case", ["ndm1", "nchan1", "nout1", "allmasked", "onechan", "ndm17", "unsorted"])
def test_lanes_degenerate(emu, oracle, case):
    kw = dict(ndm1=dict(ndm=1), nchan1=dict(nchan=1), nout1=dict(), allmasked=dict(), onechan=dict(),
              ndm17=dict(ndm=17), unsorted=dict(ndm=40, dm_max=70.0))[case]
    wl = small(**kw)
    if case == "nout1":
        _, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, 1)
        wl = wl.cropped(dmax + 1)
    if case == "allmasked":
        wl.mask = np.ones(wl.nchan, dtype=np.uint8)
    if case == "onechan":
        wl.mask = np.ones(wl.nchan, dtype=np.uint8)
        wl.mask[wl.nchan - 1] = 0
    if case == "unsorted":
        rng = np.random.default_rng(5)
        wl.dm_list = np.concatenate([rng.permutation(wl.dm_list), [wl.dm_list[7], wl.dm_list[7], 0.0]])
    check(emu, oracle, wl, LANES)


@pytest.mark.parametrize("dtype,ds", [("u8", 1), ("u8", 4), ("f32", 1)])
def test_lanes_unaligned_dense_input(emu, oracle, dtype, ds):
    """Dense rows whose pitch is no multiple of 16 and an input base that is not 16-byte aligned: the interleave
    pass reads single elements, so any pitch / alignment is in range and correct."""
    wl = small(dtype=dtype, ds=ds, nsamp=1237 * ds + 1, dm_max=30.0 * ds)
    check(emu, oracle, wl, LANES, misalign=4 if dtype == "f32" else 3)


@pytest.mark.parametrize("kernel", [LANES, TILED, DIRECT], ids=["lanes", "tiled", "direct"])
@pytest.mark.parametrize("name,extra", [("fast", 700), ("wide", 600), ("lowfreq", 500), ("rfids", 650)])
def test_real_geometries_cropped(emu, oracle, name, extra, kernel):
    """The real configs' channel grids and DM steps (so the real window lengths, ring depth and stage sizes),
    cropped in time and thinned in DM blocks: first, middle and last block of 32 trials."""
    full = synth.config(name)
    nblk = (full.ndm + 31) // 32                      # blocks of 32: whole blocks for the tiled kernel, pairs for lanes
    blocks = sorted({0, nblk // 2, nblk - 1})
    dms = np.concatenate([full.dm_list[32 * b:32 * b + 32] for b in blocks])
    # every 16th channel keeps the band, the delay spread per trial and the run time of the emulation small
    sub = slice(None, None, 16)
    wl = synth.Workload(name + "-emu", full.seed, len(np.arange(full.nchan)[sub]), full.f_top, full.chan_bw * 16,
                        full.tsamp, 1, dms, downsample=full.downsample, dtype=full.dtype, mean=full.mean,
                        std=full.std)
    _, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    wl = wl.cropped(wl.downsample * (dmax + extra) - (1 if wl.downsample > 1 else 0))
    if kernel == TILED:      # 2048 outputs per tile: a full tile plus a ragged one, dense rows of odd pitch as well
        wl = wl.cropped(wl.nsamp + 2048 + 37)
    check(emu, oracle, wl, kernel)


@pytest.mark.parametrize("kind,pieces", [("u8", 3), ("u8", 7), ("bins4", 3), ("f32", 2)])
def test_lanes_host_pipelined_runs(emu, oracle, kind, pieces):
    """ddsp_execute_host_pipelined: each run of output columns is its own interleave + accumulate launch pair (own
    segment length Q, own tiles) after only the input columns it needs (< (end + d_max) * ds) were copied; the
    runs do not divide the output evenly; the result equals the oracle."""
    if kind == "u8":
        wl = small(nsamp=2600, dm_max=50.0, mask_frac=0.1)
    elif kind == "bins4":
        wl = small(ds=4, nsamp=4 * 2100 + 2, dm_max=120.0)
    else:
        wl = small(dtype="f32", nsamp=1900, dm_max=40.0)
    check(emu, oracle, wl, LANES, host_pieces=pieces)


# ---- the checks can fail: negative controls -------------------------------------------------------------------
def test_negative_control_output_too_small(emu, oracle):
    """An output buffer registered 16 bytes short must be reported (the emulator sees global writes)."""
    wl = small()
    x = host_input(wl)
    dm = np.ascontiguousarray(wl.dm_list, dtype=np.float64)
    h = ctypes.c_void_p()
    assert emu.ddsp_plan_create(ctypes.byref(h), wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp, dm.ctypes.data,
                                dm.size, 1, None, binding.DDSP_IN_U8) == 0
    try:
        nout = emu.ddsp_plan_nsamp_out(h)
        assert emu.ddsp_plan_set_kernel(h, LANES) == 0
        xin = DeviceArray(emu, x.shape, x.dtype)
        xin.a[...] = x
        out = np.zeros((wl.ndm, nout), dtype=np.uint32)
        emu.ddsp_emu_register(out.ctypes.data, out.nbytes - 16)
        f0 = emu.ddsp_emu_faults()
        assert emu.ddsp_execute(h, xin.a.ctypes.data, out.ctypes.data, None) == 0
        assert emu.ddsp_emu_faults() - f0 == 4
        emu.ddsp_emu_unregister(out.ctypes.data)
        xin.release()
    finally:
        emu.ddsp_plan_destroy(h)


@pytest.mark.parametrize("kernel", [TILED, DIRECT], ids=["tiled", "direct"])
def test_negative_control_output_too_small_other_kernels(emu, oracle, kernel):
    """The same for the kernels with a hardware history: their output stores and read-modify-write flushes go
    through range-checked helpers too."""
    wl = small()
    x = host_input(wl)
    dm = np.ascontiguousarray(wl.dm_list, dtype=np.float64)
    h = ctypes.c_void_p()
    assert emu.ddsp_plan_create(ctypes.byref(h), wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp, dm.ctypes.data,
                                dm.size, 1, None, binding.DDSP_IN_U8) == 0
    try:
        nout = emu.ddsp_plan_nsamp_out(h)
        assert emu.ddsp_plan_set_kernel(h, kernel) == 0
        xin = DeviceArray(emu, x.shape, x.dtype)
        xin.a[...] = x
        out = np.zeros((wl.ndm, nout), dtype=np.uint32)
        emu.ddsp_emu_register(out.ctypes.data, out.nbytes - 16)
        f0 = emu.ddsp_emu_faults()
        assert emu.ddsp_execute(h, xin.a.ctypes.data, out.ctypes.data, None) == 0
        assert emu.ddsp_emu_faults() - f0 >= 1
        emu.ddsp_emu_unregister(out.ctypes.data)
        xin.release()
    finally:
        emu.ddsp_plan_destroy(h)


def test_negative_control_input_too_small(emu, oracle):
    """An input buffer registered one byte short must be reported (the emulator sees global reads)."""
    wl = small()
    x = host_input(wl)
    dm = np.ascontiguousarray(wl.dm_list, dtype=np.float64)
    h = ctypes.c_void_p()
    assert emu.ddsp_plan_create(ctypes.byref(h), wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp, dm.ctypes.data,
                                dm.size, 1, None, binding.DDSP_IN_U8) == 0
    try:
        nout = emu.ddsp_plan_nsamp_out(h)
        assert emu.ddsp_plan_set_kernel(h, LANES) == 0
        emu.ddsp_emu_register(x.ctypes.data, x.nbytes - 1)
        out = DeviceArray(emu, (wl.ndm, nout), np.uint32)
        f0 = emu.ddsp_emu_faults()
        assert emu.ddsp_execute(h, x.ctypes.data, out.a.ctypes.data, None) == 0
        assert emu.ddsp_emu_faults() - f0 >= 1
        emu.ddsp_emu_unregister(x.ctypes.data)
        out.release()
    finally:
        emu.ddsp_plan_destroy(h)


# ---- race check of the shared-memory protocol under ThreadSanitizer (tests/emu/emu_tsan_main.cpp) -------------
def _run_tsan(exe, case, halt=0, timeout=900):
    """Returns (returncode or None if it had to be killed, stdout, stderr)."""
    env = dict(os.environ, TSAN_OPTIONS="halt_on_error=%d report_signal_unsafe=0" % halt)
    p = subprocess.Popen([exe, case], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, env=env)
    try:
        out, err = p.communicate(timeout=timeout)
        rc = p.returncode
    except subprocess.TimeoutExpired:
        p.kill()
        out, err = p.communicate()
        rc = None
    if "FATAL: ThreadSanitizer" in err:        # e.g. an address-space layout the sanitizer runtime rejects
        pytest.skip("ThreadSanitizer cannot run here: " + err.strip().splitlines()[0])
    return rc, out, err


@pytest.mark.parametrize("case", ["u8", "bins2", "bins4", "f32"])
def test_lanes_protocol_is_race_free(case):
    """More chunks than ring stages and several work items per CTA, so every stage is refilled by the copy engine
    while other warps are still at work on its neighbours: no shared-memory access may be unordered with
    respect to the copy engine."""
    rc, out, err = _run_tsan(build_emu.build(tsan=True), case)
    assert "ThreadSanitizer" not in err, err[-3000:]
    assert rc == 0, (rc, out, err[-2000:])
    assert "faults=0" in out and "status=0" in out


def test_lanes_race_check_can_fail():
    """Negative control: a producer that refills a stage WITHOUT waiting for the consumers' `empty` barrier must be
    reported as a data race -- otherwise the clean runs above would prove nothing."""
    exe = build_emu.build(tsan=True, mutate=("early", "if (p_issued >= a.NS) ok = mbar_wait(", "if (false) ok = mbar_wait(",
                                              "ddsp_lanes.cu"))
    # The broken protocol may also lose a barrier phase and sit in its bounded waits; all that matters here is
    # that the unordered access is reported, so the run is cut short.
    for attempt in range(3):                  # thread interleavings differ from run to run
        rc, out, err = _run_tsan(exe, "u8", halt=1, timeout=240)
        if "ThreadSanitizer: data race" in err:
            break
    assert "ThreadSanitizer: data race" in err, (rc, out, err[-1500:])


# ---- seeded random plans: whatever the shape, the lanes kernels equal the oracle and stay inside their buffers -----
def test_lanes_random_plans(emu, oracle):
    rng = np.random.default_rng(20261105)
    done = 0
    for trial in range(40):
        dtype = "f32" if rng.random() < 0.3 else "u8"
        ds = int(rng.choice([1, 1, 2, 3, 4, 5, 7, 16]))
        nchan = int(rng.integers(1, 34))
        ndm = int(rng.integers(1, 40))
        f_top = float(rng.choice([1500.0, 800.0, 400.0]))
        wl = synth.Workload("rnd", int(rng.integers(0, 1000)), nchan, f_top, -float(rng.uniform(0.5, 8.0)),
                            float(rng.choice([1e-3, 2.5e-4])), 1, np.sort(rng.uniform(0.0, 40.0 * ds, ndm)),
                            downsample=ds, dtype=dtype, mean=128.0 if dtype == "u8" else 0.0,
                            std=50.0 if dtype == "u8" else 1.0)
        if rng.random() < 0.5:
            wl.mask = (rng.random(nchan) < 0.3).astype(np.uint8)
        if rng.random() < 0.3:
            wl.dm_list = rng.permutation(wl.dm_list)
        _, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, ds)
        if dmax > 3000:
            continue
        nout = int(rng.integers(1, 1400))
        wl = wl.cropped(ds * (dmax + nout) - int(rng.integers(0, ds)))
        pitch = wl.nsamp + int(rng.integers(0, 20))
        check(emu, oracle, wl, LANES, pitch=pitch, misalign=int(rng.integers(0, 4)) * (4 if dtype == "f32" else 1))
        done += 1
        if done == 12:
            break
    assert done == 12


@pytest.mark.parametrize("name", ["fast", "wide", "lowfreq", "rfids"])
def test_lanes_all_channels_last_dm_block(emu, oracle, name):
    """The big configs with ALL their channels (e.g. `fast`: 512 chunks through a ring of 5 stages, 8 flushes of
    the 16-bit lanes; `rfids`: mask, x4 bins, 29 flushes; the longest windows of each plan) for the last, ragged
    block of DM trials, cropped to one time tile."""
    full = synth.config(name)
    dms = full.dm_list[-9:]
    wl = synth.Workload(name + "-allchan", full.seed, full.nchan, full.f_top, full.chan_bw, full.tsamp, 1, dms,
                        downsample=full.downsample, dtype=full.dtype, mean=full.mean, std=full.std)
    wl.mask = full.mask
    _, dmax = oracle.delay_table(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, wl.downsample)
    wl = wl.cropped(wl.downsample * (dmax + 333) - (2 if wl.downsample > 1 else 0))
    check(emu, oracle, wl, LANES)


# ---- compile-time tuning knobs (csrc/ddsp_lanes.cu): the alternative geometries are correct too ------------------
@pytest.mark.parametrize("defines", [("DDSP_LANES_SLABS=2", "DDSP_LANES_GROUPS=8"), ("DDSP_LANES_FMA_E=0",),
                                     ("DDSP_LANES_SLABS=8", "DDSP_LANES_GROUPS=2"), ("DDSP_LANES_ROWS=6",),
                                     ("DDSP_LANES_ROWS=8", "DDSP_LANES_FLUSH_RMW=1")])
def test_lanes_tuning_knobs(oracle, defines):
    """32 trials x 256 words per item (and 8 x 1024), and the all-ALU accumulate: same results, same range checks."""
    lib = ctypes.CDLL(build_emu.build(defines=defines))
    for name, (res, args) in binding.SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    lib.ddsp_emu_faults.restype = ctypes.c_long
    lib.ddsp_emu_register.argtypes = [ctypes.c_void_p, ctypes.c_size_t]
    lib.ddsp_emu_unregister.argtypes = [ctypes.c_void_p]
    check(lib, oracle, small(mask_frac=0.2, ndm=37, nsamp=2100), LANES)
    check(lib, oracle, small(ds=4, nsamp=4 * 1500 + 3, dm_max=160.0, ndm=33), LANES)
    check(lib, oracle, small(dtype="f32", nsamp=1300, dm_max=30.0, ndm=33), LANES)
    wl = small(nchan=261, nsamp=900, ndm=35, dm_max=6.0, seed=5)      # several flushes, ragged last DM block
    wl.chan_bw = -0.5
    check(lib, oracle, wl, LANES)
