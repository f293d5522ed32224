"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

uint8 input: bit-exact uint32 sums.  float32 input: |g - o| <= 1e-5 |o| per element against the
fp32 sequential oracle (north_star tolerance; R9), plus the order-independent check against
the double-accumulated sum.  Expected values come from oracle/ only.
"""
import os

import numpy as np
import pytest
import torch

from paper_2511_02328_b200 import binding, build, synth

from _util import assert_f32_close, assert_u32_equal, crop, make_input, oracle_geometry, run_plan, to_host

pytestmark = pytest.mark.gpu

KERNELS = [binding.DDSP_KERNEL_DIRECT, binding.DDSP_KERNEL_TILED, binding.DDSP_KERNEL_LANES]
KNAME = {binding.DDSP_KERNEL_DIRECT: "direct", binding.DDSP_KERNEL_TILED: "tiled", binding.DDSP_KERNEL_LANES: "lanes"}
# Kernels without a hardware history are launched only when the bring-up protocol asks for them
# (DDSP_TEST_UNPROVEN=1, smallest case first, under compute-sanitizer); the default
# `pytest -m gpu` run touches only kernels that have already run green on a B200.  Promotion = removing the
# kernel from this set in the commit that cites the green log.
UNPROVEN = {binding.DDSP_KERNEL_LANES}
RUN_UNPROVEN = os.environ.get("DDSP_TEST_UNPROVEN", "") == "1"


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    binding.lib()


def _set_kernel(plan, kernel):
    if kernel in UNPROVEN and not RUN_UNPROVEN:
        pytest.skip("kernel %s has no hardware history yet: set DDSP_TEST_UNPROVEN=1 (bring-up protocol)" % KNAME[kernel])
    try:
        plan.set_kernel(kernel)
    except binding.DdspError as e:
        if e.code == binding.DDSP_ERR_UNSUPPORTED:
            pytest.skip("kernel %s does not support this plan" % KNAME[kernel])
        raise
    assert plan.kernel == kernel


def _compare(oracle, wl, plan, x, out, rows=None, t_lo=0, t_hi=None, what=""):
    assert plan.device_status() == 0, what + ": device status"
    xh = x.cpu().numpy()
    t_hi = plan.nsamp_out if t_hi is None else t_hi
    got = to_host(out, plan, rows, t_lo, t_hi)
    want, nout, dmax = oracle.dedisperse(xh, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, nsamp=wl.nsamp,
                                         downsample=wl.downsample, mask=wl.mask, rows=rows,
                                         t_lo=t_lo, t_hi=t_hi)
    assert nout == plan.nsamp_out and dmax == plan.max_delay
    if wl.dtype == "u8":
        assert_u32_equal(got, want, what)
    else:
        want64, _, _ = oracle.dedisperse(xh, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, nsamp=wl.nsamp,
                                         downsample=wl.downsample, mask=wl.mask, rows=rows,
                                         t_lo=t_lo, t_hi=t_hi, acc64=True)
        assert_f32_close(got, want, want64, what)


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
def test_tiny_full(oracle, kernel):
    """BASELINE.json configs[0], every output element."""
    wl = synth.config("tiny")
    x = make_input(oracle, wl, "cuda")
    with binding.plan_for(wl) as plan:
        _set_kernel(plan, kernel)
        out = run_plan(plan, x)
        _compare(oracle, wl, plan, x, out, what="tiny/" + KNAME[kernel])
        # the injected pulse (DM 100, t_p = 4096, width 3, amp 40) peaks in row 100 at its arrival time
        row = to_host(out, plan, [100])[0].astype(np.int64)
        assert 4096 <= int(row.argmax()) < 4099


def block_rows(ndm, seed):
    """At least one row of EVERY block of 16 trials (so also of every block of 32): a seeded position inside each
    block, plus both edges of the first, a middle and the last block."""
    rng = np.random.default_rng(seed)
    rows = {0, ndm - 1}
    for b0 in range(0, ndm, 16):
        rows.add(min(ndm - 1, b0 + int(rng.integers(0, 16))))
    for b0 in (0, (ndm // 32) * 16, ((ndm - 1) // 16) * 16):
        rows.update(r for r in (b0, b0 + 15, b0 + 16, b0 + 31) if 0 <= r < ndm)
    return np.array(sorted(rows), dtype=np.int64)


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
@pytest.mark.parametrize("name,extra", [("fast", 9000), ("wide", 5000), ("lowfreq", 6000), ("rfids", 7001)])
def test_cropped_configs(oracle, name, extra, kernel):
    """configs[1..4] with the full channel count and DM list, cropped in time: all columns of at least one row
    of every DM block (every block has its own window and offset tables) -- several time tiles and a ragged
    tail."""
    wl = crop(oracle, synth.config(name), extra)
    pitch = synth.round_up(wl.nsamp, 128)
    x = make_input(oracle, wl, "cuda", pitch=pitch)
    with binding.plan_for(wl) as plan:
        plan.set_pitch(pitch, synth.round_up(plan.nsamp_out, 32))
        _set_kernel(plan, kernel)
        out = run_plan(plan, x)
        rows = block_rows(wl.ndm, wl.seed)
        _compare(oracle, wl, plan, x[:, :].contiguous(), out, rows=rows, what="%s-crop/%s" % (name, KNAME[kernel]))


def _small(dtype="u8", nchan=37, nsamp=5003, ndm=23, ds=1, seed=11, dm_max=60.0, mask_frac=0.0,
           f_top=1500.0, chan_bw=-4.0, tsamp=1e-3):
    wl = synth.Workload("small", seed, nchan, f_top, chan_bw, tsamp, nsamp,
                        np.linspace(0.0, dm_max, ndm), downsample=ds, dtype=dtype,
                        mean=128.0 if dtype == "u8" else 0.0, std=30.0 if dtype == "u8" else 1.0)
    if mask_frac > 0:
        m = np.random.default_rng(seed).random(nchan) < mask_frac
        wl.mask = m.astype(np.uint8)
    return wl


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
@pytest.mark.parametrize("dtype", ["u8", "f32"])
@pytest.mark.parametrize("ds", [1, 2, 3, 4, 8])
def test_small_ragged(oracle, kernel, dtype, ds):
    """Odd sizes everywhere: unaligned dense pitch, partial last bin, mask, every element compared."""
    wl = _small(dtype=dtype, ds=ds, mask_frac=0.2, nsamp=5003 + ds)
    x = make_input(oracle, wl, "cuda")
    with binding.plan_for(wl) as plan:
        _set_kernel(plan, kernel)
        out = run_plan(plan, x)
        _compare(oracle, wl, plan, x, out, what="small ds=%d %s" % (ds, dtype))


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
def test_pitch_padding_untouched_and_input_unchanged(oracle, kernel):
    wl = _small(nsamp=4100)
    pitch = 4224
    x = make_input(oracle, wl, "cuda", pitch=pitch)
    x[:, wl.nsamp:] = 77                       # garbage in the input padding must never be read as data
    x0 = x.clone()
    with binding.plan_for(wl) as plan:
        plan.set_pitch(pitch, plan.nsamp_out + 13)
        _set_kernel(plan, kernel)
        out = run_plan(plan, x, out_fill=-1234567)
        assert torch.equal(x, x0)
        assert bool((out[:, plan.nsamp_out:] == -1234567).all())
        xv = x.clone()
        xv[:, wl.nsamp:] = 0
        got = to_host(out, plan)
        want, _, _ = oracle.dedisperse(x.cpu().numpy(), wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list,
                                       nsamp=wl.nsamp)
        assert_u32_equal(got, want, "pitched")


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
def test_unsorted_duplicate_dm_list(oracle, kernel):
    """Rows follow dm_list order whatever the order (R10); duplicates give identical rows."""
    wl = _small(ndm=40, dm_max=90.0)
    rng = np.random.default_rng(5)
    dms = np.concatenate([rng.permutation(wl.dm_list), [wl.dm_list[7], wl.dm_list[7], 0.0]])
    wl.dm_list = dms
    x = make_input(oracle, wl, "cuda")
    with binding.plan_for(wl) as plan:
        _set_kernel(plan, kernel)
        out = run_plan(plan, x)
        _compare(oracle, wl, plan, x, out, what="unsorted")


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
@pytest.mark.parametrize("case", ["ndm1", "nchan1", "nout1", "allmasked", "onechan", "dm0only"])
def test_degenerate(oracle, kernel, case):
    kw = dict(ndm1=dict(ndm=1, dm_max=0.0), nchan1=dict(nchan=1), nout1=dict(), allmasked=dict(),
              onechan=dict(), dm0only=dict(ndm=3, dm_max=0.0))[case]
    wl = _small(**kw)
    if case == "ndm1":
        wl.dm_list = np.array([33.0])
    if case == "nout1":
        _, dmax, _ = oracle_geometry(oracle, wl)
        wl = wl.cropped(dmax + 1)
    if case == "allmasked":
        wl.mask = np.ones(wl.nchan, dtype=np.uint8)
    if case == "onechan":
        wl.mask = np.ones(wl.nchan, dtype=np.uint8)
        wl.mask[wl.nchan - 1] = 0
    x = make_input(oracle, wl, "cuda")
    with binding.plan_for(wl) as plan:
        _set_kernel(plan, kernel)
        out = run_plan(plan, x, out_fill=-1)
        _compare(oracle, wl, plan, x, out, what=case)
        if case == "allmasked":
            assert not to_host(out, plan).any()


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
def test_I10_saturation_headroom(oracle, kernel):
    """x = 255 everywhere, downsample 4, 4096 channels: every output is 4 177 920 (16-bit lanes of a
    packed accumulator would overflow 64 times over)."""
    wl = synth.Workload("sat", 0, 4096, 1500.0, -0.1220703125, 64e-6, 4 * 3000,
                        np.arange(0, 41, dtype=np.float64) * 2.0, downsample=4)
    x = torch.full((wl.nchan, wl.nsamp), 255, dtype=torch.uint8, device="cuda")
    with binding.plan_for(wl) as plan:
        _set_kernel(plan, kernel)
        out = run_plan(plan, x)
        got = to_host(out, plan)
        assert got.min() == got.max() == 4177920
        # and ds = 1 with the full 8-bit range: 4096 * 255
        wl1 = synth.Workload("sat1", 0, 4096, 1500.0, -0.1220703125, 64e-6, 9000,
                             np.arange(0, 41, dtype=np.float64) * 2.0)
    with binding.plan_for(wl1) as plan:
        _set_kernel(plan, kernel)
        out = run_plan(plan, x[:, :9000].contiguous())
        got = to_host(out, plan)
        assert got.min() == got.max() == 4096 * 255


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
def test_I5_masked_channels_never_read(oracle, kernel):
    """NaN / Inf in zapped fp32 channels and 255 in zapped u8 channels cannot reach the output."""
    for dtype in ("f32", "u8"):
        wl = _small(dtype=dtype, mask_frac=0.3, seed=3)
        x = make_input(oracle, wl, "cuda")
        with binding.plan_for(wl) as plan:
            _set_kernel(plan, kernel)
            out = run_plan(plan, x)
            ref = to_host(out, plan)
            _compare(oracle, wl, plan, x, out, what="I5 reference " + dtype)      # the reference itself is the oracle's
            x2 = x.clone()
            zap = torch.as_tensor(np.flatnonzero(wl.mask), device="cuda")
            x2[zap] = float("nan") if dtype == "f32" else 255
            got = to_host(run_plan(plan, x2), plan)
            assert np.array_equal(got, ref)


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
def test_I2_impulse_and_I3_shift(oracle, kernel):
    wl = _small(nchan=64, nsamp=9000, ndm=33, dm_max=128.0)
    table, dmax, nout = oracle_geometry(oracle, wl)
    k, t0, amp = 20, 3000, 7
    x = torch.zeros((wl.nchan, wl.nsamp), dtype=torch.uint8, device="cuda")
    for c in range(wl.nchan):
        x[c, t0 + int(table[k, c])] = amp
    with binding.plan_for(wl) as plan:
        _set_kernel(plan, kernel)
        got = to_host(run_plan(plan, x), plan)
        assert got[k, t0] == wl.nchan * amp and got.max() == wl.nchan * amp
        shift = 129
        xs = torch.zeros_like(x)
        xs[:, shift:] = x[:, :-shift]
        gs = to_host(run_plan(plan, xs), plan)
        assert np.array_equal(gs[:, shift:], got[:, :-shift])


def test_execute_host_matches_device(oracle):
    wl = _small(nsamp=6000)
    x = make_input(oracle, wl, "cuda")
    with binding.plan_for(wl) as plan:
        dev = to_host(run_plan(plan, x), plan)
        xh = x.cpu().pin_memory()
        oh = torch.empty((plan.ndm, plan.out_pitch), dtype=torch.int32).pin_memory()
        plan.execute_host(xh, oh)
        assert np.array_equal(oh.numpy().view(np.uint32), dev)


@pytest.mark.parametrize("npieces", [1, 3, 8])
def test_execute_host_pipelined_lanes(oracle, npieces):
    """Overlapped host-buffer execute (lanes kernels): same result as the oracle, whatever the number of runs."""
    wl = _small(nsamp=9000)
    x = make_input(oracle, wl, "cuda")
    with binding.plan_for(wl) as plan:
        _set_kernel(plan, binding.DDSP_KERNEL_LANES)
        xh = x.cpu().pin_memory()
        oh = torch.full((plan.ndm, plan.out_pitch), -5, dtype=torch.int32).pin_memory()
        plan.execute_host_pipelined(xh, oh, npieces=npieces)
        assert plan.device_status() == 0
        want, _, _ = oracle.dedisperse(xh.numpy(), wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list)
        assert_u32_equal(oh.numpy().view(np.uint32)[:, :plan.nsamp_out], want, "pipelined")


def test_lanes_two_streams_own_workspaces(oracle):
    """Two executes of ONE lanes plan that overlap in time: each brings its own workspace (ddsp_execute_ws)."""
    wl = _small(nsamp=7000)
    x1 = make_input(oracle, wl, "cuda")
    x2 = torch.flip(x1, dims=[1]).contiguous()
    with binding.plan_for(wl) as plan:
        _set_kernel(plan, binding.DDSP_KERNEL_LANES)
        ws = [torch.empty(plan.workspace_bytes, dtype=torch.uint8, device="cuda") for _ in range(2)]
        o1 = torch.empty((plan.ndm, plan.out_pitch), dtype=torch.int32, device="cuda")
        o2 = torch.empty_like(o1)
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        torch.cuda.synchronize()
        plan.execute(x1, o1, stream=s1, workspace=ws[0])
        plan.execute(x2, o2, stream=s2, workspace=ws[1])
        torch.cuda.synchronize()
        assert plan.device_status() == 0
        for xx, oo in ((x1, o1), (x2, o2)):
            want, _, _ = oracle.dedisperse(xx.cpu().numpy(), wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list)
            assert_u32_equal(to_host(oo, plan), want, "stream")


def test_two_streams_concurrent(oracle):
    wl = _small(nsamp=7000)
    x1 = make_input(oracle, wl, "cuda")
    x2 = torch.flip(x1, dims=[1]).contiguous()
    with binding.plan_for(wl) as plan:
        o1 = torch.empty((plan.ndm, plan.out_pitch), dtype=torch.int32, device="cuda")
        o2 = torch.empty_like(o1)
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        torch.cuda.synchronize()
        plan.execute(x1, o1, stream=s1)
        plan.execute(x2, o2, stream=s2)
        torch.cuda.synchronize()
        for xx, oo in ((x1, o1), (x2, o2)):
            want, _, _ = oracle.dedisperse(xx.cpu().numpy(), wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list)
            assert_u32_equal(to_host(oo, plan), want, "stream")


@pytest.mark.parametrize("kernel", [binding.DDSP_KERNEL_TILED, binding.DDSP_KERNEL_LANES], ids=KNAME.get)
def test_full_size_fast_first_and_last_columns(oracle, kernel):
    """BASELINE.json configs[1] at FULL size, in the launch configuration bench.py times (pitches included):
    rows {0, 500, 1000} x the first and the last 4096 output columns against the oracle.  Input element offsets
    reach 6.2e9 and output byte offsets 1.2e10 -- beyond 2**32 -- so 32-bit index arithmetic anywhere in the
    path fails here (SURVEY.md 8(c) 'large-index check')."""
    free, _ = torch.cuda.mem_get_info()
    if free < 40e9:
        pytest.skip("needs 40 GB of free device memory")
    wl = synth.config("fast")
    in_pitch = synth.round_up(wl.nsamp, 128)
    x = make_input(oracle, wl, "cuda", pitch=in_pitch)
    table, dmax, nout = oracle_geometry(oracle, wl)
    with binding.plan_for(wl) as plan:
        out_pitch = synth.round_up(plan.nsamp_out, 32)
        plan.set_pitch(in_pitch, out_pitch)
        _set_kernel(plan, kernel)
        out = run_plan(plan, x, out_fill=-7)
        assert plan.device_status() == 0
        assert plan.nsamp_out == nout and plan.max_delay == dmax
        rows = np.array([0, 500, 1000])
        ncol = 4096
        assert (rows[-1] * out_pitch + nout) * 4 > 2 ** 32 and (wl.nchan - 1) * in_pitch + wl.nsamp > 2 ** 32
        for c0 in (0, nout - ncol):
            xw = x[:, c0:c0 + ncol + dmax].cpu().numpy()            # the shifted sum is translation invariant
            want = oracle.dedisperse_table(np.ascontiguousarray(xw), table[rows], nsamp=xw.shape[1], t_lo=0, t_hi=ncol)
            got = to_host(out, plan, rows, c0, c0 + ncol)
            assert_u32_equal(got, want, "fast full size, columns from %d" % c0)
        assert bool((out[:, nout:] == -7).all()), "pitch padding was written"


@pytest.mark.parametrize("kernel", KERNELS, ids=KNAME.get)
def test_dm_row_split_is_a_row_range(oracle, kernel):
    """ddsp_plan_create_rows: the outputs of plans that split one DM list are the row ranges of
    the whole list's output, with the whole list's nsamp_out (invariant I7)."""
    wl = _small(ndm=45, dm_max=80.0, nsamp=6000)
    x = make_input(oracle, wl, "cuda")
    want, nout, _ = oracle.dedisperse(x.cpu().numpy(), wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list)
    for begin, count in ((0, 23), (23, 22), (40, 5)):
        with binding.plan_for(wl, rows=(begin, count)) as plan:
            _set_kernel(plan, kernel)
            assert plan.nsamp_out == nout and plan.ndm == count
            out = run_plan(plan, x)
            assert plan.device_status() == 0
            assert_u32_equal(to_host(out, plan), want[begin:begin + count], "rows %d+%d" % (begin, count))
