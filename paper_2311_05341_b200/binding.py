"""Thin ctypes face of libdd.so (include/dd.h).  Argument marshalling only: every step of
the transform runs in the library's CUDA kernels.  PyTorch appears only as the owner of
device memory and streams.  There is no CPU fallback -- a missing library or a missing
GPU raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdd.so")

DD_U8, DD_U16, DD_F32, DD_U4 = 0, 1, 2, 3
DD_OK = 0
DD_ERR_INVALID_ARG = -1
DD_ERR_SHIFT_TOO_LARGE = -2
DD_ERR_OVERFLOW = -3
DD_ERR_ALLOC = -4
DD_ERR_CUDA = -5
DD_ERR_UNSUPPORTED_DEVICE = -6
DD_ERR_UNSUPPORTED_PLAN = -7
DD_ERR_STATIC_LIMIT = -8
NOALLOC_MAX_TABLE = 1 << 20   # DD_NOALLOC_MAX_TABLE

INFO = {"D_DM": 0, "D_J": 1, "LANES": 2, "L": 3, "SMEM_BYTES": 4, "GRID": 5, "THREADS": 6,
        "WORKSPACE_BYTES": 7, "STAGE_BYTES": 8, "LAUNCHES": 9, "CH": 10, "NSTAGE": 11, "PANEL": 12,
        "HOST_CHUNKS": 13, "HOST_TAPER": 14}

# every symbol include/dd.h declares (tests check the .so exports all of them)
SYMBOLS = ("dd_shift_table_build", "dd_plan_create", "dd_plan_shift_table", "dd_execute",
           "dd_execute_noalloc",
           "dd_execute_host", "dd_execute_host_tm", "dd_execute_host_async", "dd_execute_tm", "dd_transpose", "dd_bin_time",
           "dd_plan_set_host_chunks", "dd_plan_host_timeline", "dd_plan_info", "dd_plan_set_timing", "dd_plan_kernel_times",
           "dd_probe", "dd_plan_destroy", "dd_strerror", "dd_version",
           "dd_survey_create", "dd_survey_num_ranges", "dd_survey_plan", "dd_survey_range_dtype",
           "dd_survey_execute", "dd_survey_execute_tm", "dd_survey_destroy")

# dd_probe keys (include/dd.h DD_PROBE_*)
PROBES = {"SM_COUNT": 0, "SM_CLOCK_MHZ": 1, "LDS32": 2, "LDS64": 3, "LDS128": 4, "IADD3": 5,
          "VIADD16X2": 6, "IMAD": 7, "FADD": 8, "LOP3": 9, "PRMT": 10, "SHIFT_ADD": 11, "IMAD_HI": 12,
          "IDP4A": 13, "SHF": 14}
# libdd_tuning.so only (use_tuning_library): the tensor-memory experiments of DESIGN.md section 10
TUNING_PROBES = {"TMEM_LD": 15, "TMEM_LD_WITH_LDS": 16, "F32_ADDS_SMEM_ONLY": 17,
                 "F32_ADDS_TMEM_4_OF_8": 18, "F32_ADDS_TMEM_4_OF_8_NO_FILL": 19}

_lib = None


def use_tuning_library() -> None:
    """Load libdd_tuning.so (build.py --tuning: extra A/B kernel shapes, DD_FORCE_VARIANT / DD_PANEL /
    DD_HOST_TAPER) instead of libdd.so in this process.  Call before anything else in this module."""
    global LIB_PATH
    if _lib is not None:
        raise RuntimeError("libdd.so is already loaded; call use_tuning_library() first")
    LIB_PATH = os.path.join(_HERE, "libdd_tuning.so")


class DDError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s: %s (dd_status %d)" % (where, strerror(status), status))


def lib() -> ctypes.CDLL:
    """Load libdd.so.  Raises if it has not been built (python -m paper_2311_05341_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s is not built: run `python -m paper_2311_05341_b200.build%s` "
                              "(there is no CPU fallback)"
                              % (os.path.basename(LIB_PATH), " --tuning" if "tuning" in LIB_PATH else ""))
        L = ctypes.CDLL(LIB_PATH)
        c = ctypes
        L.dd_shift_table_build.restype = c.c_int
        L.dd_shift_table_build.argtypes = [c.c_int, c.c_double, c.c_double, c.c_double,
                                           c.c_void_p, c.c_int, c.c_void_p, c.c_void_p]
        L.dd_plan_create.restype = c.c_int
        L.dd_plan_create.argtypes = [c.POINTER(c.c_void_p), c.c_int, c.c_int64, c.c_double,
                                     c.c_double, c.c_double, c.c_void_p, c.c_int, c.c_int]
        L.dd_plan_shift_table.restype = c.c_int
        L.dd_plan_shift_table.argtypes = [c.c_void_p, c.POINTER(c.c_void_p),
                                          c.POINTER(c.c_int64), c.POINTER(c.c_int32)]
        L.dd_execute.restype = c.c_int
        L.dd_execute.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p]
        L.dd_execute_noalloc.restype = c.c_int
        L.dd_execute_noalloc.argtypes = [c.c_void_p, c.c_int, c.c_int, c.c_int64, c.c_int, c.c_void_p, c.c_void_p,
                                         c.c_void_p]
        L.dd_execute_host.restype = c.c_int
        L.dd_execute_host.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p]
        L.dd_execute_host_tm.restype = c.c_int
        L.dd_execute_host_tm.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p]
        L.dd_execute_host_async.restype = c.c_int
        L.dd_execute_host_async.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.c_int]
        L.dd_execute_tm.restype = c.c_int
        L.dd_execute_tm.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p]
        L.dd_bin_time.restype = c.c_int
        L.dd_bin_time.argtypes = [c.c_void_p, c.c_void_p, c.c_int, c.c_int64, c.c_int, c.c_int, c.c_void_p]
        L.dd_transpose.restype = c.c_int
        L.dd_transpose.argtypes = [c.c_void_p, c.c_void_p, c.c_int, c.c_int64, c.c_int, c.c_void_p]
        L.dd_plan_set_host_chunks.restype = c.c_int
        L.dd_plan_set_host_chunks.argtypes = [c.c_void_p, c.c_int]
        L.dd_plan_host_timeline.restype = c.c_int
        L.dd_plan_host_timeline.argtypes = [c.c_void_p, c.c_int, c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p]
        L.dd_plan_info.restype = c.c_int64
        L.dd_plan_info.argtypes = [c.c_void_p, c.c_int]
        L.dd_plan_set_timing.restype = c.c_int
        L.dd_plan_set_timing.argtypes = [c.c_void_p, c.c_int]
        L.dd_plan_kernel_times.restype = c.c_int
        L.dd_plan_kernel_times.argtypes = [c.c_void_p, c.c_int, c.c_void_p, c.c_void_p]
        L.dd_probe.restype = c.c_int
        L.dd_probe.argtypes = [c.c_int, c.POINTER(c.c_double)]
        L.dd_plan_destroy.restype = None
        L.dd_plan_destroy.argtypes = [c.c_void_p]
        L.dd_strerror.restype = c.c_char_p
        L.dd_strerror.argtypes = [c.c_int]
        L.dd_version.restype = c.c_char_p
        L.dd_version.argtypes = []
        L.dd_survey_create.restype = c.c_int
        L.dd_survey_create.argtypes = [c.POINTER(c.c_void_p), c.c_int, c.c_int64, c.c_double, c.c_double,
                                       c.c_double, c.c_void_p, c.c_int, c.c_int]
        L.dd_survey_num_ranges.restype = c.c_int
        L.dd_survey_num_ranges.argtypes = [c.c_void_p]
        L.dd_survey_plan.restype = c.c_void_p
        L.dd_survey_plan.argtypes = [c.c_void_p, c.c_int]
        L.dd_survey_range_dtype.restype = c.c_int
        L.dd_survey_range_dtype.argtypes = [c.c_void_p, c.c_int]
        L.dd_survey_execute.restype = c.c_int
        L.dd_survey_execute.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p]
        L.dd_survey_execute_tm.restype = c.c_int
        L.dd_survey_execute_tm.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p]
        L.dd_survey_destroy.restype = None
        L.dd_survey_destroy.argtypes = [c.c_void_p]
        _lib = L
    return _lib


def strerror(status: int) -> str:
    return lib().dd_strerror(int(status)).decode()


def version() -> str:
    return lib().dd_version().decode()


def probe(what: str) -> float:
    """dd_probe: one measured on-chip peak of the current device (keys of PROBES)."""
    v = ctypes.c_double(0.0)
    rc = lib().dd_probe(PROBES[what] if what in PROBES else TUNING_PROBES[what], ctypes.byref(v))
    if rc != DD_OK:
        raise DDError(rc, "dd_probe(%s)" % what)
    return float(v.value)


def _dm_array(dm_list) -> np.ndarray:
    return np.ascontiguousarray(dm_list, dtype=np.float64)


def dd_shift_table_build(nchans, f_high_MHz, chan_bw_MHz, tsamp_s, dm_list):
    """Host delay table (no GPU needed).  Returns (int32 [ndm, nchans], max_shift)."""
    dm = _dm_array(dm_list)
    table = np.empty((dm.size, max(int(nchans), 0)), dtype=np.int32)
    mx = ctypes.c_int32(0)
    rc = lib().dd_shift_table_build(int(nchans), float(f_high_MHz), float(chan_bw_MHz),
                                    float(tsamp_s), dm.ctypes.data, int(dm.size),
                                    table.ctypes.data, ctypes.addressof(mx))
    if rc != DD_OK:
        raise DDError(rc, "dd_shift_table_build")
    return table, int(mx.value)


def transpose(d_in_tm, d_out, nchans: int, nsamps: int, dtype: int, stream=None) -> None:
    """dd_transpose: time-major [nsamps][nchans] -> channel-major [nchans][nsamps] (device tensors)."""
    rc = lib().dd_transpose(_dev_ptr(d_in_tm), _dev_ptr(d_out), int(nchans), int(nsamps), int(dtype),
                            _stream_ptr(stream))
    if rc != DD_OK:
        raise DDError(rc, "dd_transpose")


def bin_time(d_in, d_out, nchans: int, nsamps: int, factor: int, in_dtype: int, stream=None) -> None:
    """dd_bin_time: d_out[c][t] = sum of `factor` consecutive samples of d_in (device tensors)."""
    rc = lib().dd_bin_time(_dev_ptr(d_in), _dev_ptr(d_out), int(nchans), int(nsamps), int(factor),
                           int(in_dtype), _stream_ptr(stream))
    if rc != DD_OK:
        raise DDError(rc, "dd_bin_time")


def execute_noalloc(table, nsamps: int, in_dtype: int, d_in, d_out, stream=None) -> None:
    """dd_execute_noalloc: the transform for a caller that may not allocate device memory (its pool owns
    the card, or it cannot afford cudaMalloc's device-wide stall).  ``table``: host int32 [ndm, nchans]
    from dd_shift_table_build, at most NOALLOC_MAX_TABLE entries; d_in / d_out: device tensors the caller
    already owns.  Calls that can overlap on the GPU race on the library's built-in table array."""
    tab = np.ascontiguousarray(table, dtype=np.int32)
    if tab.ndim != 2:
        raise ValueError("table must be [ndm, nchans]")
    rc = lib().dd_execute_noalloc(tab.ctypes.data, int(tab.shape[0]), int(tab.shape[1]), int(nsamps),
                                  int(in_dtype), _dev_ptr(d_in), _dev_ptr(d_out), _stream_ptr(stream))
    if rc != DD_OK:
        raise DDError(rc, "dd_execute_noalloc")


class Plan:
    """dd_plan_create / dd_plan_shift_table / dd_execute / dd_plan_destroy with the same
    argument order as the C ABI."""

    def __init__(self, nchans, nsamps, f_high_MHz, chan_bw_MHz, tsamp_s, dm_list, in_dtype):
        dm = _dm_array(dm_list)
        h = ctypes.c_void_p()
        rc = lib().dd_plan_create(ctypes.byref(h), int(nchans), int(nsamps), float(f_high_MHz),
                                  float(chan_bw_MHz), float(tsamp_s), dm.ctypes.data,
                                  int(dm.size), int(in_dtype))
        if rc != DD_OK:
            raise DDError(rc, "dd_plan_create")
        self._h = h
        self.nchans, self.nsamps, self.ndm, self.in_dtype = int(nchans), int(nsamps), int(dm.size), int(in_dtype)
        tab = ctypes.c_void_p()
        out_len = ctypes.c_int64()
        mx = ctypes.c_int32()
        rc = lib().dd_plan_shift_table(self._h, ctypes.byref(tab), ctypes.byref(out_len),
                                       ctypes.byref(mx))
        if rc != DD_OK:
            raise DDError(rc, "dd_plan_shift_table")
        self.out_len, self.max_shift = int(out_len.value), int(mx.value)
        self._table_ptr = tab.value

    # -- dd_plan_shift_table
    def shift_table(self) -> np.ndarray:
        """A copy of the plan's host table, int32 [ndm, nchans]."""
        n = self.ndm * self.nchans
        buf = (ctypes.c_int32 * n).from_address(self._table_ptr)
        return np.frombuffer(buf, dtype=np.int32).reshape(self.ndm, self.nchans).copy()

    def info(self, key: str) -> int:
        return int(lib().dd_plan_info(self._h, INFO[key]))

    # -- dd_execute
    def execute(self, d_in, d_out, stream=None) -> None:
        """d_in / d_out: torch CUDA tensors (dense) or raw device addresses (int)."""
        rc = lib().dd_execute(self._h, _dev_ptr(d_in), _dev_ptr(d_out), _stream_ptr(stream))
        if rc != DD_OK:
            raise DDError(rc, "dd_execute")

    # -- dd_execute_tm
    def execute_tm(self, d_in_tm, d_out, stream=None) -> None:
        """d_in_tm: time-major [nsamps][nchans] torch CUDA tensor (dense) or raw device address."""
        rc = lib().dd_execute_tm(self._h, _dev_ptr(d_in_tm), _dev_ptr(d_out), _stream_ptr(stream))
        if rc != DD_OK:
            raise DDError(rc, "dd_execute_tm")

    # -- dd_execute_host
    def execute_host(self, h_in, h_out, stream=None) -> None:
        """h_in / h_out: host buffers (numpy arrays or CPU torch tensors, ideally pinned)."""
        rc = lib().dd_execute_host(self._h, _host_ptr(h_in), _host_ptr(h_out), _stream_ptr(stream))
        if rc != DD_OK:
            raise DDError(rc, "dd_execute_host")

    def execute_host_tm(self, h_in_tm, h_out, stream=None) -> None:
        """h_in_tm: time-major [nsamps][nchans] host buffer; h_out as execute_host."""
        rc = lib().dd_execute_host_tm(self._h, _host_ptr(h_in_tm), _host_ptr(h_out), _stream_ptr(stream))
        if rc != DD_OK:
            raise DDError(rc, "dd_execute_host_tm")

    # -- dd_execute_host_async
    def execute_host_async(self, h_in, h_out, stream=None, time_major: bool = False) -> None:
        """Queue the host-buffer pipeline and return; complete when `stream` reaches this point."""
        rc = lib().dd_execute_host_async(self._h, _host_ptr(h_in), _host_ptr(h_out), _stream_ptr(stream),
                                         1 if time_major else 0)
        if rc != DD_OK:
            raise DDError(rc, "dd_execute_host_async")

    # -- dd_plan_set_host_chunks
    def set_host_chunks(self, nchunks: int) -> None:
        """0 = the default schedule of dd_execute_host, 1..8 = that many equal chunks."""
        rc = lib().dd_plan_set_host_chunks(self._h, int(nchunks))
        if rc != DD_OK:
            raise DDError(rc, "dd_plan_set_host_chunks")

    # -- dd_plan_host_timeline
    def host_timeline(self, max_chunks: int = 16):
        """Per chunk of the latest execute_host[_tm]: (out_begin, h2d_ms, pre_ms, main_ms, d2h_ms) arrays."""
        ob = np.zeros(max_chunks, dtype=np.int64)
        t = [np.zeros(max_chunks, dtype=np.float32) for _ in range(4)]
        n = lib().dd_plan_host_timeline(self._h, int(max_chunks), ob.ctypes.data, *[a.ctypes.data for a in t])
        if n < 0:
            raise DDError(n, "dd_plan_host_timeline")
        return (ob[:n].copy(),) + tuple(a[:n].copy() for a in t)

    # -- dd_plan_set_timing / dd_plan_kernel_times
    def set_timing(self, on: bool) -> None:
        rc = lib().dd_plan_set_timing(self._h, 1 if on else 0)
        if rc != DD_OK:
            raise DDError(rc, "dd_plan_set_timing")

    def kernel_times(self, max_n: int = 64):
        """(interleave_ms[], main_ms[]) of the latest timed executions, oldest first."""
        a = np.zeros(max_n, dtype=np.float32)
        b = np.zeros(max_n, dtype=np.float32)
        n = lib().dd_plan_kernel_times(self._h, int(max_n), a.ctypes.data, b.ctypes.data)
        if n < 0:
            raise DDError(n, "dd_plan_kernel_times")
        return a[:n].copy(), b[:n].copy()

    def destroy(self) -> None:
        if getattr(self, "_h", None) is not None and self._h:
            lib().dd_plan_destroy(self._h)
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


def _dev_ptr(x) -> int:
    if isinstance(x, int):
        return x
    if not x.is_cuda or not x.is_contiguous():
        raise ValueError("dd_execute wants dense CUDA tensors")
    return x.data_ptr()


def _host_ptr(x) -> int:
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        if not x.flags.c_contiguous:
            raise ValueError("host buffer must be C-contiguous")
        return x.ctypes.data
    if x.is_cuda or not x.is_contiguous():
        raise ValueError("dd_execute_host wants dense host tensors")
    return x.data_ptr()


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


BIN_OUT_DTYPE = {DD_U8: DD_U16, DD_U4: DD_U8, DD_F32: DD_F32}   # dd_bin_time widens integer types


class _DmRange(ctypes.Structure):
    _fields_ = [("dm_start", ctypes.c_double), ("dm_step", ctypes.c_double),
                ("count", ctypes.c_int32), ("bin_factor", ctypes.c_int32)]


class Survey:
    """dd_survey_create / dd_survey_execute[_tm] / dd_survey_destroy: a multi-range DM survey plan in
    the style of the paper's Table 2.  ``ranges`` = (dm_start, dm_step, count,
    bin_factor) tuples.  Marshalling only: the plans, the binned blocks and the loop over ranges
    live in the library; this class allocates the output tensors (one per range) and hands their
    addresses over.  ``execute`` / ``execute_tm`` return those tensors."""

    def __init__(self, nchans, nsamps, f_high_MHz, chan_bw_MHz, tsamp_s, ranges, in_dtype):
        import torch
        arr = (_DmRange * len(ranges))(*[_DmRange(float(a), float(b), int(n), int(f)) for a, b, n, f in ranges])
        h = ctypes.c_void_p()
        rc = lib().dd_survey_create(ctypes.byref(h), int(nchans), int(nsamps), float(f_high_MHz),
                                    float(chan_bw_MHz), float(tsamp_s), ctypes.cast(arr, ctypes.c_void_p),
                                    len(ranges), int(in_dtype))
        if rc != DD_OK:
            raise DDError(rc, "dd_survey_create")
        self._h = h
        self.nranges = int(lib().dd_survey_num_ranges(self._h))
        self.ndm, self.out_len, self.max_shift, self.dtype, self.outs = [], [], [], [], []
        for r in range(self.nranges):
            plan = lib().dd_survey_plan(self._h, r)
            out_len, mx = ctypes.c_int64(), ctypes.c_int32()
            rc = lib().dd_plan_shift_table(plan, None, ctypes.byref(out_len), ctypes.byref(mx))
            if rc != DD_OK:
                raise DDError(rc, "dd_plan_shift_table")
            dt = int(lib().dd_survey_range_dtype(self._h, r))
            self.ndm.append(int(ranges[r][2]))
            self.out_len.append(int(out_len.value))
            self.max_shift.append(int(mx.value))
            self.dtype.append(dt)
            odt = torch.float32 if dt == DD_F32 else torch.int32
            self.outs.append(torch.empty((self.ndm[-1], self.out_len[-1]), dtype=odt, device="cuda"))
        self._ptrs = (ctypes.c_void_p * self.nranges)(*[o.data_ptr() for o in self.outs])

    def execute(self, d_in, stream=None):
        rc = lib().dd_survey_execute(self._h, _dev_ptr(d_in), ctypes.cast(self._ptrs, ctypes.c_void_p),
                                     _stream_ptr(stream))
        if rc != DD_OK:
            raise DDError(rc, "dd_survey_execute")
        return self.outs

    def execute_tm(self, d_in_tm, stream=None):
        rc = lib().dd_survey_execute_tm(self._h, _dev_ptr(d_in_tm), ctypes.cast(self._ptrs, ctypes.c_void_p),
                                        _stream_ptr(stream))
        if rc != DD_OK:
            raise DDError(rc, "dd_survey_execute_tm")
        return self.outs

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().dd_survey_destroy(self._h)
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
