"""Pins of the CPU oracle (oracle/) against what the paper and the mathematics fix.

None of these compare the oracle with itself: the delay table is checked against exact
rational arithmetic and printed pins, the shifted sum against a hand-worked example, a
pure-Python per-output gather written independently, closed forms and invariants
(SURVEY.md section 8(c) I1-I12).  CPU only.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- helpers
def exact_delay(dm, c, f_top, chan_bw, tsamp, ds):
    """Eq. 4 / Eq. 5 in exact rational arithmetic, round half up."""
    K = Fraction("4148.808")
    f0 = Fraction(f_top)
    f = f0 + c * Fraction(chan_bw)
    v = K * Fraction(dm) * (1 / (f * f) - 1 / (f0 * f0)) / (Fraction(tsamp) * ds)
    return int((v + Fraction(1, 2)).__floor__())


def gather_brute(x, delays, mask, ds, nsamp, nout):
    """Independent formulation (I12): one output element at a time, pure Python ints."""
    nchan = len(x)
    out = []
    for drow in delays:
        row = []
        for t in range(nout):
            s = 0
            for c in range(nchan):
                if mask is not None and mask[c]:
                    continue
                u = t + int(drow[c])
                for k in range(ds):
                    j = ds * u + k
                    if j < nsamp:
                        s += int(x[c][j])
            row.append(s)
        out.append(row)
    return np.array(out, dtype=np.int64)


def read_golden(path):
    rows = {}
    with open(path) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            key, vals = line.split(":")
            rows[tuple(key.split())] = [int(v) for v in vals.split()]
    return rows


def golden_x():
    return np.array([[(3 * c + 5 * t + ((c * t) % 7)) % 11 for t in range(16)] for c in range(4)],
                    dtype=np.uint8)


# ----------------------------------------------------------------------------- delay table
def _pin_rows():
    with open(os.path.join(GOLD, "delay_pins.txt")) as fh:
        for line in fh:
            if line.startswith("#") or "|" not in line:
                continue
            left, right = line.split("|")
            yield left.split(), [int(v) for v in right.split()]


@pytest.mark.parametrize("left,right", list(_pin_rows()), ids=lambda v: v[0] if isinstance(v[0], str) else None)
def test_delay_table_printed_pins(oracle, left, right):
    name, nchan, f_top, bw, tsamp, ds, step, ndm = left
    nchan, ds, ndm = int(nchan), int(ds), int(ndm)
    dms = float(step) * np.arange(ndm, dtype=np.float64)
    tab, dmax = oracle.delay_table(nchan, float(f_top), float(bw), float(tsamp), dms, ds)
    total, p_dmax, d1last, imid, cmid, dmid, dlast1, dlastq = right
    assert int(tab.sum(dtype=np.int64)) == total
    assert dmax == p_dmax == int(tab[-1, -1]) == int(tab.max())
    assert int(tab[1, -1]) == d1last
    assert int(tab[imid, cmid]) == dmid
    assert int(tab[-1, 1]) == dlast1
    assert int(tab[-1, nchan // 4]) == dlastq
    assert (tab[:, 0] == 0).all()                      # reference = top of band
    assert (np.diff(tab.astype(np.int64), axis=1) >= 0).all()
    assert (np.diff(tab.astype(np.int64), axis=0) >= 0).all()


@pytest.mark.parametrize("left,right", list(_pin_rows()), ids=lambda v: v[0] if isinstance(v[0], str) else None)
def test_delay_table_exact_rational(oracle, left, right):
    """Every entry of tiny, a strided + random sample of the big tables, vs Fraction."""
    name, nchan, f_top, bw, tsamp, ds, step, ndm = left
    nchan, ds, ndm = int(nchan), int(ds), int(ndm)
    dms = float(step) * np.arange(ndm, dtype=np.float64)
    tab, _ = oracle.delay_table(nchan, float(f_top), float(bw), float(tsamp), dms, ds)
    if name == "tiny":
        pairs = [(i, c) for i in range(ndm) for c in range(nchan)]
    else:
        rng = np.random.default_rng(7)
        pairs = [(int(i), int(c)) for i, c in zip(rng.integers(0, ndm, 3000), rng.integers(0, nchan, 3000))]
        pairs += [(ndm - 1, c) for c in range(0, nchan, 37)] + [(i, nchan - 1) for i in range(0, ndm, 41)]
    for i, c in pairs:
        want = exact_delay(Fraction(step) * i, c, f_top, bw, tsamp, ds)
        assert int(tab[i, c]) == want, (name, i, c)


def test_delay_hand_check_and_row(oracle):
    # PAPER.md Eq. 4 by hand: 4148.808*2*(1400^-2 - 1500^-2)/1e-3 = 0.5456 -> 1
    v = 4148.808 * 2 * (1400.0 ** -2 - 1500.0 ** -2) / 1e-3
    assert abs(v - 0.5456) < 1e-3
    tab, _ = oracle.delay_table(2, 1500.0, -100.0, 1e-3, [2.0])
    assert tab.tolist() == [[0, 1]]
    with open(os.path.join(GOLD, "delay_pins.txt")) as fh:
        row = [l for l in fh if l.startswith("tiny_row100")][0].split(":")[1].split()
    tab, _ = oracle.delay_table(64, 1500.0, -2.0, 1e-3, np.arange(201.0))
    assert tab[100].tolist() == [int(v) for v in row]


def test_delay_units_reading_R1(oracle):
    """K in s*MHz^2: DM 1024 sweep over 1000-1500 MHz is 2.36 s (PAPER.md:236-248 use a 22 s
    file for a 20 s span), not 2.36 ms."""
    tab, dmax = oracle.delay_table(2, 1500.0, -500.0, 1.0, [1024.0])
    assert dmax == 2                      # 2.36 s -> rounds to 2 samples of 1 s
    tab, dmax = oracle.delay_table(2, 1500.0, -500.0, 1e-3, [1024.0])
    assert dmax == 2360


def test_downsample_scales_tsamp(oracle):
    # tsamp_ds = D * tsamp: table(ds=4, tsamp) == table(ds=1, 4*tsamp)
    dms = np.arange(0, 300, 7.0)
    a, _ = oracle.delay_table(128, 1500.0, -1.0, 64e-6, dms, 4)
    b, _ = oracle.delay_table(128, 1500.0, -1.0, 256e-6, dms, 1)
    assert (a == b).all()


# ----------------------------------------------------------------------------- golden example
def test_golden_example(oracle):
    g = read_golden(os.path.join(GOLD, "golden_4x16.txt"))
    x = golden_x()
    dms = [0.0, 2.0, 5.0]
    tab, dmax = oracle.delay_table(4, 1500.0, -100.0, 1e-3, dms)
    assert tab.tolist() == [g[("delays_ds1", str(i))] for i in range(3)] and dmax == 5
    out, nout, _ = oracle.dedisperse(x, 1500.0, -100.0, 1e-3, dms)
    assert nout == 11
    assert out.tolist() == [g[("plain", str(i))] for i in range(3)]
    out, _, _ = oracle.dedisperse(x, 1500.0, -100.0, 1e-3, dms, mask=[0, 0, 1, 0])
    assert out.tolist() == [g[("mask0010", str(i))] for i in range(3)]
    tab2, dmax2 = oracle.delay_table(4, 1500.0, -100.0, 1e-3, dms, 2)
    assert tab2.tolist() == [g[("delays_ds2", str(i))] for i in range(3)] and dmax2 == 3
    out, nout, _ = oracle.dedisperse(x, 1500.0, -100.0, 1e-3, dms, downsample=2)
    assert nout == 5
    assert out.tolist() == [g[("ds2", str(i))] for i in range(3)]


def test_golden_three_entries_by_hand():
    """x[c][t] = (3c + 5t + (ct mod 7)) mod 11, delays for DM 5 = [0,1,3,5]."""
    g = read_golden(os.path.join(GOLD, "golden_4x16.txt"))
    x = lambda c, t: (3 * c + 5 * t + ((c * t) % 7)) % 11
    # D[2][0] = x0[0] + x1[1] + x2[3] + x3[5] = 0 + 9 + 5 + 2
    assert (x(0, 0), x(1, 1), x(2, 3), x(3, 5)) == (0, 9, 5, 2)
    assert g[("plain", "2")][0] == 16
    # D[0][5] = x0[5]+x1[5]+x2[5]+x3[5] = 3 + 0 + 1 + 2
    assert (x(0, 5), x(1, 5), x(2, 5), x(3, 5)) == (3, 0, 1, 2)
    assert g[("plain", "0")][5] == 6
    # D[1][10] (DM 2, delays 0,1,1,2) = x0[10]+x1[11]+x2[11]+x3[12] = 6 + 7 + 7 + 4
    assert (x(0, 10), x(1, 11), x(2, 11), x(3, 12)) == (6, 7, 7, 4)
    assert g[("plain", "1")][10] == 24
    # ds=2, D[2][4] with delays [0,1,2,3]: bins x_ds[c][u] = x[c][2u]+x[c][2u+1]
    b = lambda c, u: x(c, 2 * u) + x(c, 2 * u + 1)
    assert b(0, 4) + b(1, 5) + b(2, 6) + b(3, 7) == g[("ds2", "2")][4] == 41


def test_golden_by_gather():
    g = read_golden(os.path.join(GOLD, "golden_4x16.txt"))
    x = golden_x().tolist()
    d1 = [g[("delays_ds1", str(i))] for i in range(3)]
    assert gather_brute(x, d1, None, 1, 16, 11).tolist() == [g[("plain", str(i))] for i in range(3)]
    assert gather_brute(x, d1, [0, 0, 1, 0], 1, 16, 11).tolist() == [g[("mask0010", str(i))] for i in range(3)]
    d2 = [g[("delays_ds2", str(i))] for i in range(3)]
    assert gather_brute(x, d2, None, 2, 16, 5).tolist() == [g[("ds2", str(i))] for i in range(3)]


# ----------------------------------------------------------------------------- invariants
P = dict(f_top=1500.0, chan_bw=-12.5, tsamp=2.5e-4)     # 8..40 channels, delays up to ~100s of samples


def _rand_u8(nchan, nsamp, seed):
    return np.random.default_rng(seed).integers(0, 256, (nchan, nsamp), dtype=np.uint8)


def test_I12_brute_force_8_channels(oracle):
    x = _rand_u8(8, 300, 1)
    dms = [0.0, 3.0, 11.5, 40.0, 40.0, 7.25]
    for ds, mask in ((1, None), (1, [0, 1, 0, 0, 0, 0, 1, 0]), (3, None), (4, [1, 0, 0, 0, 0, 0, 0, 1])):
        tab, dmax = oracle.delay_table(8, 1500.0, -50.0, 1e-3, dms, ds)
        out, nout, dm2 = oracle.dedisperse(x, 1500.0, -50.0, 1e-3, dms, downsample=ds, mask=mask)
        assert dm2 == dmax and nout == -(-300 // ds) - dmax and dmax > 3
        want = gather_brute(x.tolist(), tab.tolist(), mask, ds, 300, nout)
        assert (out.astype(np.int64) == want).all()


def test_I1_dm0_is_channel_sum(oracle):
    x = _rand_u8(24, 2000, 2)
    mask = np.zeros(24, np.uint8)
    mask[[3, 17]] = 1
    out, nout, _ = oracle.dedisperse(x, dm_list=[0.0, 30.0], **P)
    assert (out[0] == x[:, :nout].sum(axis=0, dtype=np.uint32)).all()
    out, nout, _ = oracle.dedisperse(x, dm_list=[0.0, 30.0], mask=mask, **P)
    assert (out[0] == x[mask == 0][:, :nout].sum(axis=0, dtype=np.uint32)).all()


def test_I2_impulse(oracle):
    nchan, nsamp, amp, t0 = 32, 4000, 40, 1234
    dms = np.arange(0, 60, 1.0)
    tab, dmax = oracle.delay_table(nchan, dm_list=dms, **P)
    mask = np.zeros(nchan, np.uint8)
    mask[[5, 6, 30]] = 1
    k = 37
    x = np.zeros((nchan, nsamp), np.uint8)
    for c in range(nchan):
        x[c, t0 + tab[k, c]] = amp
    out, nout, _ = oracle.dedisperse(x, dm_list=dms, mask=mask, **P)
    nun = int((mask == 0).sum())
    assert out[k, t0] == nun * amp
    assert out.max() == nun * amp
    for i in range(len(dms)):
        cnt = sum(1 for c in range(nchan) if not mask[c] and 0 <= t0 + tab[k, c] - tab[i, c] < nout)
        assert int(out[i].sum()) == amp * cnt


def test_I3_shift_and_I8_prefix(oracle):
    x = _rand_u8(16, 3000, 3)
    dms = [0.0, 5.0, 21.0]
    out, nout, _ = oracle.dedisperse(x, dm_list=dms, **P)
    k = 17
    xs = np.zeros_like(x)
    xs[:, k:] = x[:, :-k]
    outs, _, _ = oracle.dedisperse(xs, dm_list=dms, **P)
    assert (outs[:, k:] == out[:, : nout - k]).all()
    outp, noutp, _ = oracle.dedisperse(x[:, :2000].copy(), dm_list=dms, **P)
    assert noutp == nout - 1000 and (outp == out[:, :noutp]).all()


def test_I4_linearity_and_constant(oracle):
    a = np.random.default_rng(4).integers(0, 100, (16, 1500), dtype=np.uint8)
    b = np.random.default_rng(5).integers(0, 100, (16, 1500), dtype=np.uint8)
    dms = [0.0, 9.0, 33.0]
    oa, _, _ = oracle.dedisperse(a, dm_list=dms, **P)
    ob, _, _ = oracle.dedisperse(b, dm_list=dms, **P)
    oab, _, _ = oracle.dedisperse(a + b, dm_list=dms, **P)
    assert (oab == oa + ob).all()
    mask = np.zeros(16, np.uint8)
    mask[2] = 1
    c = np.full((16, 1600), 7, np.uint8)
    oc, _, _ = oracle.dedisperse(c, dm_list=dms, downsample=4, mask=mask, **P)
    assert (oc == 7 * 4 * 15).all()


def test_I5_mask_irrelevance_and_all_masked(oracle):
    x = _rand_u8(16, 1200, 6)
    mask = np.zeros(16, np.uint8)
    mask[[0, 9, 15]] = 1
    dms = [0.0, 14.0]
    o1, _, _ = oracle.dedisperse(x, dm_list=dms, mask=mask, **P)
    x2 = x.copy()
    x2[mask == 1] = 255
    o2, _, _ = oracle.dedisperse(x2, dm_list=dms, mask=mask, **P)
    assert (o1 == o2).all()
    xf = np.random.default_rng(1).standard_normal((16, 1200)).astype(np.float32)
    f1, _, _ = oracle.dedisperse(xf, dm_list=dms, mask=mask, **P)
    xf[mask == 1] = np.nan
    f2, _, _ = oracle.dedisperse(xf, dm_list=dms, mask=mask, **P)
    assert np.array_equal(f1, f2) and np.isfinite(f2).all()
    o3, nout, dmax = oracle.dedisperse(x, dm_list=dms, mask=np.ones(16, np.uint8), **P)
    assert (o3 == 0).all() and dmax > 0            # d_max ignores the mask (R6)


def test_I6_I7_dm_list_independence(oracle):
    x = _rand_u8(16, 2500, 7)
    dms = np.array([0.0, 2.0, 2.0, 10.0, 25.0, 3.0])
    out, nout, _ = oracle.dedisperse(x, dm_list=dms, **P)
    assert (out[1] == out[2]).all()
    perm = [4, 0, 5, 2]
    outp, noutp, _ = oracle.dedisperse(x, dm_list=dms[perm], **P)
    assert noutp == nout and (outp == out[perm]).all()
    outs, nouts, _ = oracle.dedisperse(x, dm_list=dms[[0, 1, 5]], **P)
    assert nouts > nout and (outs[:, :nout] == out[[0, 1, 5]]).all()


def test_I9_fused_equals_unfused(oracle):
    for nsamp in (2400, 2402):                       # second: partial last bin (R8)
        x = _rand_u8(16, nsamp, 8)
        dms = [0.0, 6.0, 31.0]
        k = 4
        fused, nout, _ = oracle.dedisperse(x, dm_list=dms, downsample=k, **P)
        nds = -(-nsamp // k)
        xp = np.zeros((16, nds * k), np.uint32)
        xp[:, :nsamp] = x
        binned = xp.reshape(16, nds, k).sum(axis=2)
        assert nout == nds - oracle.delay_table(16, P["f_top"], P["chan_bw"], P["tsamp"] * k, dms)[1]
        tab, _ = oracle.delay_table(16, P["f_top"], P["chan_bw"], P["tsamp"] * k, dms)
        want = np.stack([sum(binned[c, tab[i, c]: tab[i, c] + nout] for c in range(16)) for i in range(3)])
        assert (fused == want).all()


def test_I10_saturation_headroom(oracle):
    x = np.full((4096, 64), 255, np.uint8)
    out, nout, _ = oracle.dedisperse(x, 1500.0, -0.1, 1e-3, [0.0], downsample=4)
    assert nout == 16 and (out == 4177920).all()


def test_I11_subband_reduction(oracle):
    """Eq. 7 + Eq. 9 with N0 = 1 (coarse grid = fine grid, residual DM 0 so
    every R_{m,s} = 0) and one channel per subband is the brute-force definition verbatim."""
    x = _rand_u8(12, 1800, 9)
    dms = np.arange(0, 40, 4.0)
    tab, dmax = oracle.delay_table(12, dm_list=dms, **P)
    out, nout, _ = oracle.dedisperse(x, dm_list=dms, **P)
    L = nout
    Y = np.zeros((len(dms), L), np.int64)
    for m in range(len(dms)):
        j = m                                      # j(m) = floor(m / N0), N0 = 1
        I = np.zeros((12, L), np.int64)            # Eq. 7, C_s = {s}, tau0 = 0
        for s in range(12):
            I[s] = x[s, tab[j, s]: tab[j, s] + L]
        R = np.zeros(12, np.int64)                 # Eq. 8 with Delta DM_m = 0
        for s in range(12):
            Y[m] += I[s, R[s]: R[s] + L]           # Eq. 9
    assert (Y == out).all()


def test_window_and_rows(oracle):
    x = _rand_u8(16, 3000, 10)
    dms = np.arange(0, 30, 1.5)
    full, nout, _ = oracle.dedisperse(x, dm_list=dms, downsample=2, **P)
    sub, _, _ = oracle.dedisperse(x, dm_list=dms, downsample=2, rows=[3, 19, 7], t_lo=100, t_hi=nout - 3, **P)
    assert (sub == full[[3, 19, 7], 100: nout - 3]).all()


def test_pitch_and_partial_bin(oracle):
    x = _rand_u8(8, 1003, 11)
    xp = np.full((8, 1100), 99, np.uint8)          # padding must never be read
    xp[:, :1003] = x
    a, na, _ = oracle.dedisperse(x, dm_list=[0.0, 8.0], downsample=4, **P)
    b, nb, _ = oracle.dedisperse(xp, dm_list=[0.0, 8.0], downsample=4, nsamp=1003, **P)
    assert na == nb and (a == b).all()


# ----------------------------------------------------------------------------- float32 path
def test_f32_sequential_order_and_acc64(oracle):
    rng = np.random.default_rng(12)
    x = rng.standard_normal((24, 900)).astype(np.float32)
    dms = [0.0, 5.0, 17.0]
    tab, dmax = oracle.delay_table(24, dm_list=dms, **P)
    out, nout, _ = oracle.dedisperse(x, dm_list=dms, **P)
    o64, _, _ = oracle.dedisperse(x, dm_list=dms, acc64=True, **P)
    assert out.dtype == np.float32 and o64.dtype == np.float64
    # one fp32 accumulator from +0.0f, ascending channels (R9) -- numpy scalar fp32 adds
    for i in range(3):
        acc = np.zeros(nout, np.float32)
        for c in range(24):
            acc = (acc + x[c, tab[i, c]: tab[i, c] + nout]).astype(np.float32)
        assert np.array_equal(acc, out[i])
        want64 = sum(x[c, tab[i, c]: tab[i, c] + nout].astype(np.float64) for c in range(24))
        assert np.allclose(o64[i], want64, rtol=0, atol=1e-12)
    rms = np.sqrt((o64 ** 2).mean(axis=1, keepdims=True))
    assert (np.abs(out - o64) <= 1e-5 * np.maximum(np.abs(o64), rms)).all()


def test_f32_downsample_bins(oracle):
    x = np.random.default_rng(13).standard_normal((6, 403)).astype(np.float32)
    out, nout, _ = oracle.dedisperse(x, dm_list=[0.0], downsample=3, **P)
    xp = np.zeros((6, 405), np.float32)
    xp[:, :403] = x
    b = xp.reshape(6, 135, 3)
    bins = ((b[:, :, 0] + b[:, :, 1]).astype(np.float32) + b[:, :, 2]).astype(np.float32)
    acc = np.zeros(135, np.float32)
    for c in range(6):
        acc = (acc + bins[c]).astype(np.float32)
    assert nout == 135 and np.array_equal(out[0], acc)


def test_errors(oracle):
    x = _rand_u8(4, 10, 0)
    with pytest.raises(ValueError):
        oracle.dedisperse(x, 1500.0, -100.0, 1e-3, [50.0])     # d_max >= nsamp: no output
