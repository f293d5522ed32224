"""Thin ctypes binding of libddsp (include/ddsp.h): same names, argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels.  PyTorch appears only as the owner
of device memory and streams (`Plan.execute` takes torch CUDA tensors and passes their data pointers).
There is no CPU fallback: if libddsp.so is missing the import of the library raises, and executing a
plan without a CUDA device raises DdspError(DDSP_ERR_CUDA).
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libddsp.so")

DDSP_IN_U8, DDSP_IN_F32 = 0, 1
DDSP_OK, DDSP_ERR_INVALID_ARG, DDSP_ERR_NO_OUTPUT, DDSP_ERR_UNSUPPORTED, DDSP_ERR_ALLOC, DDSP_ERR_CUDA = range(6)
DDSP_KERNEL_AUTO, DDSP_KERNEL_DIRECT, DDSP_KERNEL_TILED, DDSP_KERNEL_LANES = 0, 1, 2, 3

# name -> (restype, argtypes); one entry per declaration in include/ddsp.h
_i, _i64, _f64, _vp, _cp = ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p, ctypes.c_char_p
SIGNATURES = {
    "ddsp_plan_create": (_i, [ctypes.POINTER(_vp), _i, _f64, _f64, _f64, _i64, _vp, _i, _i, _vp, _i]),
    "ddsp_plan_create_rows": (_i, [ctypes.POINTER(_vp), _i, _f64, _f64, _f64, _i64, _vp, _i, _i, _i, _i, _vp, _i]),
    "ddsp_plan_set_pitch": (_i, [_vp, _i64, _i64]),
    "ddsp_plan_set_kernel": (_i, [_vp, _i]),
    "ddsp_plan_nsamp_out": (_i64, [_vp]),
    "ddsp_plan_max_delay": (_i64, [_vp]),
    "ddsp_plan_nchan_unmasked": (_i, [_vp]),
    "ddsp_plan_kernel": (_i, [_vp]),
    "ddsp_plan_launches_per_execute": (_i, [_vp]),
    "ddsp_plan_workspace_bytes": (_i64, [_vp]),
    "ddsp_plan_device_status": (_i, [_vp, _vp]),
    "ddsp_plan_get_delays": (_i, [_vp, _vp]),
    "ddsp_execute": (_i, [_vp, _vp, _vp, _vp]),
    "ddsp_execute_ws": (_i, [_vp, _vp, _vp, _vp, _i64, _vp]),
    "ddsp_execute_host": (_i, [_vp, _vp, _vp, _vp]),
    "ddsp_execute_host_pipelined": (_i, [_vp, _vp, _vp, _vp, _i]),
    "ddsp_plan_destroy": (_i, [_vp]),
    "ddsp_strerror": (_cp, [_i]),
    "ddsp_last_cuda_error": (_i, [_vp]),
    "ddsp_version": (_cp, []),
}

_lib = None


class DdspError(RuntimeError):
    def __init__(self, code, where, cuda=0):
        self.code, self.cuda = code, cuda
        msg = lib().ddsp_strerror(code).decode()
        super().__init__("%s: %s (code %d%s)" % (where, msg, code, ", cudaError %d" % cuda if cuda else ""))


def lib():
    """Load libddsp.so (built by paper_2511_02328_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libddsp.so not built: run `python -m paper_2511_02328_b200.build` "
                              "(there is no CPU fallback)")
        l = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(l, name)
            fn.restype, fn.argtypes = res, args
        _lib = l
    return _lib


def _check(code, where, plan=None):
    if code != DDSP_OK:
        cuda = lib().ddsp_last_cuda_error(plan) if plan else 0
        raise DdspError(code, where, cuda)


class Plan:
    """ddsp_plan_create / ddsp_execute / ddsp_plan_destroy with the header's argument names."""

    def __init__(self, nchan, f_top_mhz, chan_bw_mhz, tsamp_s, nsamp, dm_list, downsample=1,
                 chan_mask=None, in_dtype=DDSP_IN_U8, rows=None):
        """rows = (row_begin, row_count): ddsp_plan_create_rows, a plan for that range of dm_list only."""
        self._h = None
        dm = np.ascontiguousarray(dm_list, dtype=np.float64)
        mask = None if chan_mask is None else np.ascontiguousarray(chan_mask, dtype=np.uint8)
        if mask is not None and mask.shape != (nchan,):
            raise ValueError("chan_mask must have nchan entries")
        h = _vp()
        begin, count = (0, int(dm.size)) if rows is None else (int(rows[0]), int(rows[1]))
        code = lib().ddsp_plan_create_rows(ctypes.byref(h), int(nchan), float(f_top_mhz), float(chan_bw_mhz),
                                           float(tsamp_s), int(nsamp), dm.ctypes.data, int(dm.size), begin, count,
                                           int(downsample), mask.ctypes.data if mask is not None else None,
                                           int(in_dtype))
        _check(code, "ddsp_plan_create_rows")
        self._h = h
        self.nchan, self.ndm, self.nsamp = int(nchan), count, int(nsamp)
        self.downsample, self.in_dtype = int(downsample), int(in_dtype)
        self.in_pitch, self.out_pitch = self.nsamp, self.nsamp_out

    # -- getters --------------------------------------------------------------------------------
    @property
    def nsamp_out(self):
        return int(lib().ddsp_plan_nsamp_out(self._h))

    @property
    def max_delay(self):
        return int(lib().ddsp_plan_max_delay(self._h))

    @property
    def nchan_unmasked(self):
        return int(lib().ddsp_plan_nchan_unmasked(self._h))

    @property
    def kernel(self):
        return int(lib().ddsp_plan_kernel(self._h))

    @property
    def launches_per_execute(self):
        return int(lib().ddsp_plan_launches_per_execute(self._h))

    @property
    def workspace_bytes(self):
        return int(lib().ddsp_plan_workspace_bytes(self._h))

    def device_status(self):
        """ddsp_plan_device_status: 0 ok, 1 bounded wait ran out, 2 table bounds check (synchronises)."""
        st = ctypes.c_int(0)
        _check(lib().ddsp_plan_device_status(self._h, ctypes.byref(st)), "ddsp_plan_device_status", self._h)
        return int(st.value)

    def get_delays(self):
        out = np.empty((self.ndm, self.nchan), dtype=np.int32)
        _check(lib().ddsp_plan_get_delays(self._h, out.ctypes.data), "ddsp_plan_get_delays", self._h)
        return out

    # -- setters --------------------------------------------------------------------------------
    def set_pitch(self, in_pitch_elems, out_pitch_elems):
        _check(lib().ddsp_plan_set_pitch(self._h, int(in_pitch_elems), int(out_pitch_elems)),
               "ddsp_plan_set_pitch", self._h)
        self.in_pitch, self.out_pitch = int(in_pitch_elems), int(out_pitch_elems)

    def set_kernel(self, kernel):
        _check(lib().ddsp_plan_set_kernel(self._h, int(kernel)), "ddsp_plan_set_kernel", self._h)

    # -- execute --------------------------------------------------------------------------------
    def execute_ptr(self, d_in, d_out, cuda_stream=0):
        """Raw form: device addresses as integers, cudaStream_t as integer."""
        _check(lib().ddsp_execute(self._h, _vp(d_in), _vp(d_out), _vp(cuda_stream)), "ddsp_execute", self._h)

    def execute(self, x, out, stream=None, workspace=None):
        """x, out: torch CUDA tensors shaped (nchan, in_pitch) and (ndm, out_pitch); workspace: optional torch
        CUDA uint8 tensor of at least workspace_bytes (ddsp_execute_ws), else the plan's own."""
        import torch
        self._check_buffers(x, out, cuda=True)
        s = torch.cuda.current_stream(x.device) if stream is None else stream
        if workspace is None:
            self.execute_ptr(x.data_ptr(), out.data_ptr(), s.cuda_stream)
        else:
            _check(lib().ddsp_execute_ws(self._h, _vp(x.data_ptr()), _vp(out.data_ptr()), _vp(workspace.data_ptr()),
                                         int(workspace.numel() * workspace.element_size()), _vp(s.cuda_stream)),
                   "ddsp_execute_ws", self._h)
        return out

    def execute_host(self, x, out, stream=None):
        """x, out: torch CPU tensors (pinned recommended) or numpy arrays; blocks until done."""
        import torch
        self._check_buffers(x, out, cuda=False)
        xp = x.data_ptr() if hasattr(x, "data_ptr") else x.ctypes.data
        op = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        s = torch.cuda.current_stream() if stream is None else stream
        _check(lib().ddsp_execute_host(self._h, _vp(xp), _vp(op), _vp(s.cuda_stream)),
               "ddsp_execute_host", self._h)
        return out

    def execute_host_pipelined(self, x, out, stream=None, npieces=8):
        """ddsp_execute_host_pipelined: copies and kernels overlapped over `npieces` runs of output columns."""
        import torch
        self._check_buffers(x, out, cuda=False)
        xp = x.data_ptr() if hasattr(x, "data_ptr") else x.ctypes.data
        op = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        s = torch.cuda.current_stream() if stream is None else stream
        _check(lib().ddsp_execute_host_pipelined(self._h, _vp(xp), _vp(op), _vp(s.cuda_stream), int(npieces)),
               "ddsp_execute_host_pipelined", self._h)
        return out

    def _check_buffers(self, x, out, cuda):
        in_size = 1 if self.in_dtype == DDSP_IN_U8 else 4
        def geom(a):
            if hasattr(a, "data_ptr"):
                return tuple(a.shape), a.element_size(), a.is_contiguous(), a.is_cuda
            return tuple(a.shape), a.itemsize, a.flags.c_contiguous, False
        (xs, xe, xc, xcu), (os_, oe, oc, ocu) = geom(x), geom(out)
        if xs != (self.nchan, self.in_pitch) or xe != in_size or not xc:
            raise ValueError("input must be a contiguous (nchan, in_pitch) = %s buffer of %d-byte elements, got %s"
                             % ((self.nchan, self.in_pitch), in_size, xs))
        if os_ != (self.ndm, self.out_pitch) or oe != 4 or not oc:
            raise ValueError("output must be a contiguous (ndm, out_pitch) = %s buffer of 4-byte elements, got %s"
                             % ((self.ndm, self.out_pitch), os_))
        if xcu != cuda or ocu != cuda:
            raise ValueError("buffers must be %s memory" % ("CUDA" if cuda else "host"))

    # -- lifetime -------------------------------------------------------------------------------
    def destroy(self):
        if self._h is not None:
            lib().ddsp_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()


def version():
    return lib().ddsp_version().decode()


def plan_for(wl, **kw):
    """Plan for a synth.Workload (argument marshalling only)."""
    return Plan(wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp, wl.dm_list, wl.downsample,
                wl.mask, DDSP_IN_U8 if wl.dtype == "u8" else DDSP_IN_F32, **kw)   # kw: rows=(begin, count)
