"""Host logic of the ring kernel (tile geometry) without a GPU.

The plan-time tables of ddsp_ring.cu -- row-window offsets, unit counts, per-(channel, trial) shared
memory offsets, the DM-sorted row map -- are read back through ddsp_plan_ring_tables and replayed here
step by step the way the kernel consumes them (stage a window, form the four phase copies, read word
(q >> 2) of copy (q & 3)).  The replayed result must equal the oracle bit for bit.  This pins every
table entry that the kernel's addressing depends on; the kernel's own arithmetic is covered by the
-m gpu parity tests.
"""
import numpy as np
import pytest

from paper_2511_02328_b200 import binding, build, synth

T = 2048


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    binding.lib()


@pytest.fixture()
def ring_enabled(monkeypatch):
    monkeypatch.setenv("DDSP_ENABLE_RING", "1")


def replay(plan, x, in_pitch, blocks=None):
    """Replay the ring kernel's data flow on the host from the plan's tables.  x: uint8 [nchan, in_pitch]."""
    g = plan.ring_geometry()
    meta, tbl, rows = plan.ring_tables()
    assert g["tile_t"] == T
    C, S = g["c_rows"], g["row_stride"]
    nout = plan.nsamp_out
    flat = x.reshape(-1)
    in_valid = (plan.nchan - 1) * in_pitch + plan.nsamp
    out = np.zeros((plan.ndm, nout), dtype=np.uint32)
    done = np.zeros(plan.ndm, dtype=bool)
    ntile = (nout + T - 1) // T
    nlist = plan.nchan_unmasked
    for b in (range(g["nblk"]) if blocks is None else blocks):
        for tile in range(ntile):
            t0 = tile * T
            acc = np.zeros((32, T), dtype=np.uint32)
            for l in range(nlist):
                chunk, slot = divmod(l, C)
                m = int(meta[b, l])
                so, units = (m & ((1 << 48) - 1)) + t0, m >> 48
                assert so % 16 == 0, "copy-engine source must be 16-byte aligned"
                assert units == int(tbl[b, chunk, C * 32 + slot])
                assert (units + 1) * 16 <= S
                raw = np.zeros(units * 16 + 16, dtype=np.uint8)      # what is not copied is never needed
                n = max(0, min(units * 16, in_valid - so))
                raw[:n] = flat[so:so + n]
                for j in range(32):
                    off = int(tbl[b, chunk, slot * 32 + j])
                    copy, w = divmod(off, S)
                    assert copy // 4 == slot and w % 4 == 0
                    q = w + copy % 4                                 # byte offset of this trial in the window
                    assert q + T <= units * 16
                    acc[j] += raw[q:q + T]
            for j in range(32):
                r = int(rows[b, j])
                if r >= 0:
                    ncol = min(T, nout - t0)
                    out[r, t0:t0 + ncol] = acc[j, :ncol]
                    done[r] = True
    return out, done


def _case(oracle, wl, pitch=None, blocks=None):
    from _util import make_input
    x = make_input(oracle, wl, "cpu", pitch=pitch).numpy()
    with binding.plan_for(wl) as plan:
        if pitch is not None:
            plan.set_pitch(pitch, plan.nsamp_out)
        got, done = replay(plan, x, x.shape[1], blocks)
        want, nout, _ = oracle.dedisperse(x, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, nsamp=wl.nsamp,
                                          mask=wl.mask)
        assert nout == plan.nsamp_out
        assert done.any()
        assert np.array_equal(got[done], want[done])
        return done


def test_tiny_all_blocks(oracle, ring_enabled):
    done = _case(oracle, synth.config("tiny"))
    assert done.all()


@pytest.mark.parametrize("pitch", [None, 5003 + 61, 5120])
def test_odd_pitch_mask_unsorted(oracle, ring_enabled, pitch):
    """Dense and odd pitches (row windows start in the previous row), a mask, an unsorted DM list with
    duplicates, a channel count that is not a multiple of the rows per stage."""
    rng = np.random.default_rng(5)
    dms = rng.permutation(np.concatenate([np.linspace(0, 300, 70), [17.0, 17.0]]))
    wl = synth.Workload("ring-small", 11, 37, 1400.0, -3.0, 2.5e-4, 5003, dms, dtype="u8", mean=120.0, std=40.0)
    wl.mask = (np.arange(37) % 5 == 2).astype(np.uint8)
    done = _case(oracle, wl, pitch=pitch)
    assert done.all()


def test_fast_cropped_block_sample(oracle, ring_enabled):
    """BASELINE.json configs[1] geometry (2048 channels, 1001 trials), cropped in time; first, middle and
    last DM block (the last one is ragged: 1001 = 31 * 32 + 9)."""
    from _util import crop
    wl = crop(oracle, synth.config("fast"), 2500)
    with binding.plan_for(wl) as plan:
        g = plan.ring_geometry()
        assert g["nblk"] == 32 and g["c_rows"] in (2, 4) and g["nstage"] >= 4
        assert g["smem_bytes"] <= 232448
    _case(oracle, wl, pitch=synth.round_up(wl.nsamp, 128), blocks=[0, 15, 31])


def test_disabled_by_default(monkeypatch):
    monkeypatch.delenv("DDSP_ENABLE_RING", raising=False)
    with binding.plan_for(synth.config("tiny")) as plan:
        with pytest.raises(binding.DdspError) as e:
            plan.ring_geometry()
        assert e.value.code == binding.DDSP_ERR_UNSUPPORTED


# ------------------------------------------------------------------------------------------------
# float32 (ds = 1) and uint8 with ds > 1: tables of ddsp_ringx.cu
# ------------------------------------------------------------------------------------------------
def replay_x(plan, x, in_pitch, wl, blocks=None):
    g = plan.ringx_geometry()
    meta, tbl, rows = plan.ringx_tables()
    kind, C, T = g["kind"], g["c_rows"], g["tile_t"]
    ds = wl.downsample
    esize = 4 if kind == 2 else 1
    nout = plan.nsamp_out
    flat = x.reshape(-1).view(np.uint8)
    in_valid = ((plan.nchan - 1) * in_pitch + plan.nsamp) * esize
    chans = [c for c in range(plan.nchan) if wl.mask is None or not wl.mask[c]]
    out = np.zeros((plan.ndm, nout), dtype=np.float32 if kind == 2 else np.uint32)
    done = np.zeros(plan.ndm, dtype=bool)
    if kind == 1:
        assert g["flush_every"] * 255 * ds <= 65535 and g["flush_every"] >= 2 * C
        assert g["nraw"] >= 2 and g["nbins"] >= 3
    else:
        assert g["nraw"] >= 4
    assert g["smem_bytes"] <= 232448
    for b in (range(g["nblk"]) if blocks is None else blocks):
        for tile in range((nout + T - 1) // T):
            t0 = tile * T
            acc = np.zeros((32, T), dtype=out.dtype)
            for l, c in enumerate(chans):
                chunk, slot = divmod(l, C)
                m = int(meta[b, l])
                so, units = (m & ((1 << 48) - 1)) + t0 * (4 if kind == 2 else ds), m >> 48
                assert so % 16 == 0
                n = max(0, min(units * 16, in_valid - so))
                raw = np.zeros(units * 16, dtype=np.uint8)
                raw[:n] = flat[so:so + n]
                if kind == 2:
                    assert units == int(tbl[b, chunk, C * 32 + slot]) and units * 16 <= g["raw_stride"]
                    win = raw.view(np.float32)
                else:
                    nb = int(tbl[b, chunk, C * 32 + slot])
                    jstart = int(tbl[b, chunk, C * 32 + C + slot])
                    assert so == c * in_pitch + jstart + t0 * ds
                    assert units * 16 >= 8 * nb * ds and (8 * nb + 1) * ds <= g["raw_stride"] and nb * 16 <= g["bins_stride"]
                    limit = plan.nsamp - (jstart + t0 * ds)
                    if limit < raw.size:
                        raw[max(limit, 0):] = 0
                    win = raw[:8 * nb * ds].reshape(-1, ds).astype(np.uint32).sum(axis=1)
                for j in range(32):
                    off = int(tbl[b, chunk, slot * 32 + j])
                    if kind == 2:
                        s_, w = divmod(off, g["raw_stride"])
                        assert s_ == slot and w % 4 == 0
                        q = w // 4
                    else:
                        copy, w = divmod(off, g["bins_stride"])
                        assert copy // 2 == slot and w % 4 == 0
                        q = w // 2 + copy % 2
                    assert q + T <= win.size
                    acc[j] = acc[j] + win[q:q + T]          # float32: one IEEE add per channel, ascending
            for j in range(32):
                r = int(rows[b, j])
                if r >= 0:
                    ncol = min(T, nout - t0)
                    out[r, t0:t0 + ncol] = acc[j, :ncol]
                    done[r] = True
    return out, done


def _case_x(oracle, wl, pitch=None, blocks=None):
    from _util import make_input
    x = make_input(oracle, wl, "cpu", pitch=pitch).numpy()
    with binding.plan_for(wl) as plan:
        if pitch is not None:
            plan.set_pitch(pitch, plan.nsamp_out)
        got, done = replay_x(plan, x, x.shape[1], wl, blocks)
        want, nout, _ = oracle.dedisperse(x, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list, nsamp=wl.nsamp,
                                          downsample=wl.downsample, mask=wl.mask)
        assert nout == plan.nsamp_out and done.any()
        if wl.dtype == "u8":
            assert np.array_equal(got[done], want[done])
        else:       # the oracle returns float64 holding the fp32 sequential sums: equal bit for bit
            assert np.array_equal(got[done].astype(np.float64), want[done])
        return done


@pytest.mark.parametrize("ds,pitch", [(2, 5024), (3, 5024), (4, 5024), (4, 5040), (8, 5056)])
def test_bins_tables(oracle, ring_enabled, ds, pitch):
    """uint8 with ds > 1: partial last bin (nsamp % ds != 0), mask, odd channel count."""
    wl = synth.Workload("ringb-small", 12, 27, 1400.0, -4.0, 1e-4, 5003 + ds, np.linspace(0, 400, 45), downsample=ds,
                        dtype="u8", mean=128.0, std=50.0)
    wl.mask = (np.arange(27) % 6 == 1).astype(np.uint8)
    assert _case_x(oracle, wl, pitch=pitch).all()


def test_bins_need_aligned_rows(oracle, ring_enabled):
    wl = synth.Workload("ringb-pitch", 13, 8, 1400.0, -4.0, 1e-4, 5003, np.linspace(0, 100, 5), downsample=4, dtype="u8")
    with binding.plan_for(wl) as plan:           # dense pitch 5003: not a multiple of 16
        with pytest.raises(binding.DdspError):
            plan.ringx_geometry()
        plan.set_pitch(5008, plan.nsamp_out)
        assert plan.ringx_geometry()["kind"] == 1


@pytest.mark.parametrize("pitch", [None, 5003 + 2, 5008])
def test_f32_tables(oracle, ring_enabled, pitch):
    wl = synth.Workload("ringf-small", 14, 21, 800.0, -3.0, 5e-4, 5003, np.linspace(0, 300, 40), dtype="f32",
                        mean=0.0, std=1.0)
    wl.mask = (np.arange(21) % 5 == 3).astype(np.uint8)
    assert _case_x(oracle, wl, pitch=pitch).all()


def test_rfids_and_lowfreq_geometry(oracle, ring_enabled):
    """BASELINE.json configs[4] (ds = 4, mask) and configs[3] (float32): the geometry fits one SM's shared memory."""
    for name, kind in (("rfids", 1), ("lowfreq", 2)):
        wl = synth.config(name)
        with binding.plan_for(wl) as plan:
            plan.set_pitch(synth.round_up(wl.nsamp, 128), synth.round_up(plan.nsamp_out, 32))
            g = plan.ringx_geometry()
            assert g["kind"] == kind and g["c_rows"] in (2, 4)
            print(name, g)
