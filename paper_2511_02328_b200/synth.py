"""Seeded synthetic filterbanks shaped like the paper's workloads (BASELINE.json configs).

This module holds NONE of the method's arithmetic: no delay formula, no shifted sum.
Where a recipe needs dispersion delays (pulse injection) or nsamp_out (pulse times), the
caller passes them in -- the tests take them from oracle/, bench.py takes them from the
library's own ddsp_plan_get_delays.  It serves both the oracle and the CUDA path, and
imports neither.

The noise generator is a counter-based integer hash (splitmix64 of (seed, channel, t))
evaluated with int64 torch ops, so the same bytes come out on CPU and on CUDA and no
chunking can change the stream.  Gaussian-like values come from the sum of the hash's 8
bytes (Irwin-Hall, mean 1020, std 209.02), scaled with integer arithmetic.

Stand-ins: the paper's 150 s / 2048-channel / 8-bit observation and its
synthetic 8-bit sets are not available; these inputs take only their
shapes (channels, band, tsamp, duration, bit width, DM range).  Recipe: DESIGN.md section 4.
"""
from dataclasses import dataclass, field, replace
from typing import Callable, Optional

import numpy as np
import torch

_GOLD = -7046029254386353131          # 0x9E3779B97F4A7C15 as int64
_M1 = -4658895280553007687            # 0xBF58476D1CE4E5B9
_M2 = -7723592293110705685            # 0x94D049BB133111EB
_SUM8_MEAN = 1020                     # 8 * 127.5
_SUM8_STD = 209.02392207591933        # sqrt(8 * (256**2 - 1) / 12)


def _lsr(z, k):
    """Logical shift right of an int64 tensor."""
    return (z >> k) & ((1 << (64 - k)) - 1)


def _splitmix64(z):
    z = z + _GOLD
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    return z ^ _lsr(z, 31)


def _hash_rows(seed, c0, c1, n, device, t0=0):
    """int64 hash of (seed, c, t) for c in [c0,c1), t in [t0, t0+n)."""
    c = torch.arange(c0, c1, dtype=torch.int64, device=device).unsqueeze(1)
    t = torch.arange(t0, t0 + n, dtype=torch.int64, device=device).unsqueeze(0)
    key = _splitmix64(c * 1000003 + int(seed) * 7919 + 12345)
    return _splitmix64(key ^ (t * 2 + 1))


def _sum8(h):
    s = h & 255
    for k in range(1, 8):
        s = s + (_lsr(h, 8 * k) & 255)
    return s


def noise_u8(seed, c0, c1, n, mean, std, device, t0=0):
    """uint8 rows: clamp(mean + round(std * z), 0, 255), z ~ Irwin-Hall(8) standardised."""
    s = _sum8(_hash_rows(seed, c0, c1, n, device, t0)) - _SUM8_MEAN
    m = int(round(std / _SUM8_STD * 65536.0))
    v = ((s * m + 32768) >> 16) + int(mean)
    return v.clamp_(0, 255).to(torch.uint8)


def noise_f32(seed, c0, c1, n, device, t0=0):
    """float32 rows ~ N(0,1): ((sum8-1020)*4096 + 12 extra hash bits - 2048) * const."""
    h = _hash_rows(seed, c0, c1, n, device, t0)
    fine = _splitmix64(h) & 4095
    v = (_sum8(h) - _SUM8_MEAN) * 4096 + fine - 2048        # |v| < 2**23: exact in fp32
    scale = np.float32(1.0 / (_SUM8_STD * 4096.0))
    return v.to(torch.float32) * float(scale)


@dataclass
class Workload:
    name: str
    seed: int
    nchan: int
    f_top: float            # MHz, centre of channel 0 (reference frequency)
    chan_bw: float          # MHz, negative
    tsamp: float            # s
    nsamp: int
    dm_list: np.ndarray     # float64
    downsample: int = 1
    dtype: str = "u8"       # "u8" -> uint32 out, "f32" -> float32 out
    mean: float = 128.0
    std: float = 20.0
    n_pulses: int = 0
    pulse_amp: float = 0.0
    pulse_dm_range: tuple = (0.0, 0.0)
    pulse_wexp_max: int = 0          # width = 2**U{0..wexp_max}
    fixed_pulses: tuple = ()         # ((dm, width, t_p), ...) overrides the draw
    n_rfi: int = 0                   # narrowband RFI channels (mean 250)
    n_zap: int = 0                   # total zapped channels (includes the RFI ones)
    n_spikes: int = 0                # broadband zero-DM spikes (+60, 2 samples)
    mask: Optional[np.ndarray] = field(default=None, repr=False)
    rfi_channels: Optional[np.ndarray] = field(default=None, repr=False)

    @property
    def ndm(self):
        return int(self.dm_list.size)

    @property
    def torch_dtype(self):
        return torch.uint8 if self.dtype == "u8" else torch.float32

    @property
    def elem_size(self):
        return 1 if self.dtype == "u8" else 4

    def cropped(self, nsamp):
        return replace(self, nsamp=int(nsamp), name=self.name + "-crop")


def _finish(wl):
    """Channel selections that depend only on the seed (not on the method)."""
    if wl.n_zap or wl.n_rfi:
        perm = np.random.default_rng(wl.seed).permutation(wl.nchan)
        wl.rfi_channels = np.sort(perm[: wl.n_rfi])
        mask = np.zeros(wl.nchan, dtype=np.uint8)
        mask[perm[: wl.n_zap]] = 1
        wl.mask = mask
    return wl


def config(name):
    """The five BASELINE.json configs (index or name)."""
    names = ["tiny", "fast", "wide", "lowfreq", "rfids"]
    if isinstance(name, int):
        name = names[name]
    if name == "tiny":
        return _finish(Workload("tiny", 0, 64, 1500.0, -2.0, 1e-3, 8192,
                                np.arange(0, 201, dtype=np.float64), std=16.0,
                                fixed_pulses=((100.0, 3, 4096),), pulse_amp=40.0))
    if name == "fast":
        return _finish(Workload("fast", 1, 2048, 1500.0, -0.244140625, 49.152e-6, 3051758,
                                np.arange(0, 1001, dtype=np.float64), n_pulses=10,
                                pulse_amp=12.0, pulse_dm_range=(50.0, 1000.0), pulse_wexp_max=6))
    if name == "wide":
        return _finish(Workload("wide", 2, 4096, 1500.0, -0.1220703125, 64e-6, 937500,
                                0.5 * np.arange(0, 6001, dtype=np.float64)))
    if name == "lowfreq":
        return _finish(Workload("lowfreq", 3, 1024, 800.0, -0.390625, 0.98304e-3, 305176,
                                np.arange(0, 3001, dtype=np.float64), dtype="f32", mean=0.0,
                                std=1.0, n_pulses=5, pulse_amp=1.0,
                                pulse_dm_range=(100.0, 3000.0), pulse_wexp_max=4))
    if name == "rfids":
        return _finish(Workload("rfids", 4, 2048, 1500.0, -0.244140625, 49.152e-6, 3051758,
                                np.arange(0, 2001, dtype=np.float64), downsample=4,
                                n_rfi=8, n_zap=205, n_spikes=3))
    # Context sweeps shaped like the paper's E1 / E2 timing experiments (synthetic 8-bit data,
    # 22 s at 40 us, 1000-1500 MHz, DM 0-1024; E1: 1500 trials, channels swept; E2: 2048 channels, trials swept).
    # Not BASELINE.json configs and not targets: `bench.py --config e1:4096` / `e2:8192` give numbers to set
    # beside the paper's RTX 4090 figures.
    if isinstance(name, str) and name[:3] in ("e1:", "e2:"):
        n = int(name[3:])
        nchan, ndm = (n, 1500) if name[:2] == "e1" else (2048, n)
        return _finish(Workload(name, 10 + n % 97, nchan, 1500.0, -500.0 / nchan, 40e-6, 550000,
                                np.linspace(0.0, 1024.0, ndm)))
    raise KeyError(name)


CONFIG_NAMES = ("tiny", "fast", "wide", "lowfreq", "rfids")


def pulses(wl, nsamp_out):
    """[(dm, width, t_p)] on the native grid; t_p is the arrival sample at f_top.
    nsamp_out (on the downsampled grid) is supplied by the caller."""
    if wl.fixed_pulses:
        return [tuple(p) for p in wl.fixed_pulses]
    rng = np.random.default_rng(wl.seed)
    out = []
    for p in range(wl.n_pulses):
        dm = float(rng.uniform(*wl.pulse_dm_range))
        width = int(2 ** int(rng.integers(0, wl.pulse_wexp_max + 1)))
        t_p = int((p + 0.5) * nsamp_out / wl.n_pulses) * wl.downsample
        out.append((dm, width, t_p))
    return out


def round_up(n, m):
    return (int(n) + m - 1) // m * m


def make_input(wl, device, pitch=None, native_delays: Optional[Callable] = None,
               nsamp_out: Optional[int] = None, row_chunk=None):
    """(nchan, pitch) tensor of wl.torch_dtype on `device`; columns >= nsamp are zero.

    native_delays(dm) -> int array [nchan] of sample delays on the NATIVE grid (ds = 1);
    required when the workload injects dispersed pulses.  nsamp_out likewise.
    """
    pitch = wl.nsamp if pitch is None else int(pitch)
    assert pitch >= wl.nsamp
    x = torch.zeros((wl.nchan, pitch), dtype=wl.torch_dtype, device=device)
    if row_chunk is None:
        row_chunk = max(1, min(wl.nchan, (1 << 25) // max(1, wl.nsamp)))
    for c0 in range(0, wl.nchan, row_chunk):
        c1 = min(wl.nchan, c0 + row_chunk)
        if wl.dtype == "u8":
            x[c0:c1, : wl.nsamp] = noise_u8(wl.seed, c0, c1, wl.nsamp, wl.mean, wl.std, device)
        else:
            x[c0:c1, : wl.nsamp] = noise_f32(wl.seed, c0, c1, wl.nsamp, device)
    if wl.rfi_channels is not None:
        for c in wl.rfi_channels.tolist():
            x[c, : wl.nsamp] = noise_u8(wl.seed + 101, c, c + 1, wl.nsamp, 250.0, wl.std, device)[0]
    for j in range(wl.n_spikes):
        t = (j + 1) * wl.nsamp // 4
        _add_sat(x, slice(None), t, min(t + 2, wl.nsamp), 60.0, wl.dtype)
    pl = pulses(wl, nsamp_out if nsamp_out is not None else wl.nsamp)
    if pl:
        if native_delays is None:
            raise ValueError("workload injects dispersed pulses: native_delays required")
        for dm, width, t_p in pl:
            d = np.asarray(native_delays(dm), dtype=np.int64)
            for c in range(wl.nchan):
                a = t_p + int(d[c])
                b = min(a + width, wl.nsamp)
                if a < wl.nsamp:
                    _add_sat(x, c, a, b, wl.pulse_amp, wl.dtype)
    return x


def _add_sat(x, rows, a, b, amp, dtype):
    if dtype == "u8":
        v = x[rows, a:b].to(torch.int32) + int(amp)
        x[rows, a:b] = v.clamp_(0, 255).to(torch.uint8)
    else:
        x[rows, a:b] += float(amp)
