"""The library's kernels executed on the CPU, thread for thread: the ring kernels (ddsp_ring.cu, ddsp_ringx.cu),
which have not run on hardware yet, and -- as calibration of the harness -- the two that have (tiled, direct).

tests/emu compiles the kernels' own source with g++ (three textual substitutions, see build_emu.py) against
host stand-ins of the PTX helpers: one std::thread per CUDA thread, mbarriers with the PTX counting rules, a
copy-engine thread for cp.async.bulk.  What this checks without a GPU: the pipeline protocol terminates (no
deadlock, no over-arrival, no copies in flight at exit), every copy is 16-byte aligned and inside shared
memory, and the result equals the oracle bit for bit through the same C ABI (plan create -> execute).
What it cannot check: the PTX spellings themselves and performance -- those need the -m gpu tests.
"""
import ctypes
import importlib.util
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2511_02328_b200 import binding, synth

HERE = os.path.dirname(os.path.abspath(__file__))
_spec = importlib.util.spec_from_file_location("build_emu", os.path.join(HERE, "emu", "build_emu.py"))
build_emu = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(build_emu)


@pytest.fixture(scope="module")
def emu(request):
    os.environ["DDSP_ENABLE_RING"] = "1"
    request.addfinalizer(lambda: os.environ.pop("DDSP_ENABLE_RING", None))
    lib = ctypes.CDLL(build_emu.build())
    for name, (res, args) in binding.SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    lib.ddsp_emu_faults.restype = ctypes.c_long
    return lib


def aligned(shape, dtype, fill=None):
    """numpy array whose data pointer is 16-byte aligned (the ring kernels' requirement on the input base)."""
    n = int(np.prod(shape)) * np.dtype(dtype).itemsize
    raw = np.zeros(n + 64, dtype=np.uint8)
    off = (-raw.ctypes.data) % 64
    a = raw[off:off + n].view(dtype).reshape(shape)
    if fill is not None:
        a[...] = fill
    return a


def run_emulated(emu, wl, x, in_pitch, kernel=binding.DDSP_KERNEL_RING, host_chunks=0):
    dm = np.ascontiguousarray(wl.dm_list, dtype=np.float64)
    mask = None if wl.mask is None else np.ascontiguousarray(wl.mask, dtype=np.uint8)
    h = ctypes.c_void_p()
    rc = emu.ddsp_plan_create(ctypes.byref(h), wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp, dm.ctypes.data,
                              dm.size, wl.downsample, mask.ctypes.data if mask is not None else None,
                              binding.DDSP_IN_U8 if wl.dtype == "u8" else binding.DDSP_IN_F32)
    assert rc == 0, rc
    try:
        nout = emu.ddsp_plan_nsamp_out(h)
        out_pitch = nout + 3
        assert emu.ddsp_plan_set_pitch(h, in_pitch, out_pitch) == 0
        assert emu.ddsp_plan_set_kernel(h, kernel) == 0, "ring kernel does not support this plan"
        xin = aligned(x.shape, x.dtype)
        xin[...] = x
        out = aligned((wl.ndm, out_pitch), np.uint32 if wl.dtype == "u8" else np.float32, fill=7)
        f0 = emu.ddsp_emu_faults()
        if host_chunks:      # the overlapped host-buffer path: device staging buffers, pieces of the output columns
            rc = emu.ddsp_execute_host_pipelined(h, xin.ctypes.data, out.ctypes.data, None, host_chunks)
        else:
            rc = emu.ddsp_execute(h, xin.ctypes.data, out.ctypes.data, None)
        assert rc == 0, rc
        assert emu.ddsp_emu_faults() == f0, "the emulator flagged a fault (see stderr)"
        assert (out[:, nout:] == 7).all(), "pitch padding was written"
        return out[:, :nout].copy(), nout
    finally:
        emu.ddsp_plan_destroy(h)


def check(emu, oracle, wl, pitch=None, host_chunks=0):
    from _util import make_input
    x = make_input(oracle, wl, "cpu", pitch=pitch).numpy()
    got, nout = run_emulated(emu, wl, x, x.shape[1], host_chunks=host_chunks)
    want, nout_o, _ = oracle.dedisperse(x, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, nsamp=wl.nsamp,
                                        downsample=wl.downsample, mask=wl.mask)
    assert nout == nout_o
    if wl.dtype == "u8":
        assert np.array_equal(got, want)
    else:
        assert np.array_equal(got.astype(np.float64), want)       # same order, no FMA: bit-identical


@pytest.mark.timeout(600)
@pytest.mark.parametrize("pitch", [None, 2400])
def test_u8_ring_small(emu, oracle, pitch):
    """Two DM blocks (the second ragged), two time tiles with a ragged tail, 21 channels (last chunk has one
    row), a mask, an unsorted DM list; dense odd pitch and an aligned one."""
    rng = np.random.default_rng(3)
    dms = rng.permutation(np.linspace(0, 250, 40))
    wl = synth.Workload("emu-u8", 21, 21, 1400.0, -5.0, 2e-4, 2333, dms, dtype="u8", mean=128.0, std=60.0)
    wl.mask = (np.arange(21) % 7 == 2).astype(np.uint8)
    check(emu, oracle, wl, pitch)


@pytest.mark.timeout(900)
@pytest.mark.parametrize("pitch", [None, 2112])
def test_calibration_tiled_kernel(emu, oracle, pitch):
    """Calibration of the emulation: DDSP_KERNEL_TILED, whose parity is green on a B200, gives the oracle's result
    here as well (dense odd pitch = its byte-gather staging path, aligned pitch = its vector path; 300 channels
    = two flushes)."""
    wl = synth.Workload("emu-tiled", 26, 300, 1400.0, -0.5, 5e-4, 2100, np.linspace(0, 60, 40), dtype="u8",
                        mean=128.0, std=60.0)
    wl.mask = (np.arange(300) % 9 == 5).astype(np.uint8)
    from _util import make_input
    x = make_input(oracle, wl, "cpu", pitch=pitch).numpy()
    got, nout = run_emulated(emu, wl, x, x.shape[1], kernel=binding.DDSP_KERNEL_TILED)
    want, _, _ = oracle.dedisperse(x, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, nsamp=wl.nsamp, mask=wl.mask)
    assert np.array_equal(got, want)


@pytest.mark.timeout(900)
@pytest.mark.parametrize("dtype,ds", [("u8", 1), ("u8", 3), ("f32", 2)])
def test_calibration_direct_kernel(emu, oracle, dtype, ds):
    """The other hardware-verified kernel, DDSP_KERNEL_DIRECT (2-D grid), in the same harness."""
    wl = synth.Workload("emu-direct", 27, 11, 1400.0, -6.0, 2e-4, 1500 * ds + 1, np.linspace(0, 80, 7), downsample=ds,
                        dtype=dtype, mean=128.0 if dtype == "u8" else 0.0, std=50.0 if dtype == "u8" else 1.0)
    wl.mask = (np.arange(11) % 4 == 1).astype(np.uint8)
    from _util import make_input
    x = make_input(oracle, wl, "cpu").numpy()
    got, nout = run_emulated(emu, wl, x, x.shape[1], kernel=binding.DDSP_KERNEL_DIRECT)
    want, _, _ = oracle.dedisperse(x, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, nsamp=wl.nsamp, downsample=ds,
                                   mask=wl.mask)
    assert np.array_equal(got if dtype == "u8" else got.astype(np.float64), want)


@pytest.mark.timeout(900)
@pytest.mark.parametrize("variant", range(1, 8))
def test_u8_ring_variants(emu, oracle, variant, monkeypatch):
    """Every compiled instantiation (odd-byte adds on the ALU / FMA pipe, 8 x 4 or 4 x 8 words per thread, 2 or 4
    rows per stage) computes the same result; 300 channels so that the ring wraps and the lanes are flushed."""
    monkeypatch.setenv("DDSP_RING_VARIANT", str(variant))
    wl = synth.Workload("emu-var", 25, 300, 1400.0, -0.5, 5e-4, 2100, np.linspace(0, 60, 9), dtype="u8",
                        mean=200.0, std=60.0)
    wl.mask = (np.arange(300) % 11 == 4).astype(np.uint8)
    check(emu, oracle, wl, 2112)


@pytest.mark.timeout(900)
def test_u8_ring_flush(emu, oracle):
    """More than 256 channels of value 255: the 16-bit lanes are flushed and must not overflow (I10)."""
    wl = synth.Workload("emu-flush", 22, 300, 1400.0, -0.5, 5e-4, 2100, np.linspace(0, 60, 9), dtype="u8",
                        mean=255.0, std=0.0)
    check(emu, oracle, wl, 2112)


@pytest.mark.timeout(900)
@pytest.mark.parametrize("ds,nchan", [(2, 13), (3, 10), (4, 70)])
def test_bins_ring(emu, oracle, ds, nchan):
    """uint8 with ds > 1: partial last bin, mask; 70 channels at ds = 4 cross the 64-channel flush."""
    nsamp = ds * 2300 + 1
    wl = synth.Workload("emu-bins", 23, nchan, 1400.0, -20.0 / nchan * 5, 1e-4, nsamp, np.linspace(0, 120, 36),
                        downsample=ds, dtype="u8", mean=200.0, std=60.0)
    wl.mask = (np.arange(nchan) % 6 == 1).astype(np.uint8)
    check(emu, oracle, wl, synth.round_up(nsamp, 16))


@pytest.mark.timeout(900)
@pytest.mark.parametrize("pitch", [None, 1404])
def test_f32_ring(emu, oracle, pitch):
    wl = synth.Workload("emu-f32", 24, 19, 800.0, -6.0, 5e-4, 1401, np.linspace(0, 150, 37), dtype="f32",
                        mean=0.0, std=1.0)
    wl.mask = (np.arange(19) % 5 == 3).astype(np.uint8)
    check(emu, oracle, wl, pitch)


@pytest.mark.timeout(1200)
@pytest.mark.parametrize("kind", ["u8", "bins4", "f32"])
def test_host_pipelined_pieces(emu, oracle, kind):
    """ddsp_execute_host_pipelined: three pieces of the output columns, each launched on its own range of time
    tiles after only the input columns it needs (< (end + d_max) * ds) were copied; result equals the oracle."""
    if kind == "u8":
        wl = synth.Workload("emu-pipe-u8", 31, 9, 1400.0, -8.0, 2e-4, 6000, np.linspace(0, 200, 33), dtype="u8",
                            mean=128.0, std=60.0)
        pitch = 6016
    elif kind == "bins4":
        wl = synth.Workload("emu-pipe-b4", 32, 9, 1400.0, -8.0, 1e-4, 4 * 6000 + 2, np.linspace(0, 100, 20),
                            downsample=4, dtype="u8", mean=200.0, std=50.0)
        pitch = synth.round_up(wl.nsamp, 16)
    else:
        wl = synth.Workload("emu-pipe-f32", 33, 9, 800.0, -8.0, 5e-4, 5000, np.linspace(0, 100, 20), dtype="f32",
                            mean=0.0, std=1.0)
        pitch = None
    check(emu, oracle, wl, pitch, host_chunks=3)


# ------------------------------------------------------------------------------------------------
# race check of the shared-memory protocol under ThreadSanitizer (tests/emu/emu_tsan_main.cpp)
# ------------------------------------------------------------------------------------------------
def _run_tsan(exe, case):
    env = dict(os.environ, TSAN_OPTIONS="halt_on_error=0 report_signal_unsafe=0")
    r = subprocess.run([exe, case], capture_output=True, text=True, timeout=900, env=env)
    if "FATAL: ThreadSanitizer" in r.stderr:        # e.g. an address-space layout the sanitizer runtime rejects
        pytest.skip("ThreadSanitizer cannot run here: " + r.stderr.strip().splitlines()[0])
    return r


@pytest.mark.timeout(1200)
@pytest.mark.parametrize("case", ["u8", "bins2", "bins4", "f32"])
def test_protocol_is_race_free(case):
    """More chunks than ring stages, so every stage is refilled while other warps are still at work on its
    neighbours: no access to shared memory may be unordered with respect to the copy engine or the expansion."""
    r = _run_tsan(build_emu.build(tsan=True), case)
    assert "ThreadSanitizer" not in r.stderr, r.stderr[-3000:]
    assert r.returncode == 0, (r.stdout, r.stderr[-2000:])
    assert "faults=0" in r.stdout


@pytest.mark.timeout(1200)
def test_race_check_can_fail():
    """Negative control: refilling a stage one chunk too early (NS - 1 instead of NS - 2 chunks ahead) must be
    reported as a data race -- otherwise the clean runs above would prove nothing."""
    exe = build_emu.build(tsan=True, mutate=("early", "const int ahead = NS - 2; ", "const int ahead = NS - 1; ",
                                              "ddsp_ring.cu"))
    r = _run_tsan(exe, "u8")
    assert "ThreadSanitizer: data race" in r.stderr
