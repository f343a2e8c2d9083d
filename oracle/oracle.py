"""Python face of the CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Thin ctypes marshalling around ``dedisp_oracle.c`` -- every number comes out of that C file,
which restates PAPER.md Eq. 1 / Eq. 7 (shift table) and Eq. 3 / Alg. 1 (the transform).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from
``paper_2311_05341_b200`` and the CUDA library imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dedisp_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

U8, U16, F32 = 0, 1, 2
_NP_DTYPE = {U8: np.uint8, U16: np.uint16, F32: np.float32}


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2, OpenMP, no FMA contraction).  Returns the .so path."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            c = ctypes
            lib.oracle_c_dm.restype = c.c_double
            lib.oracle_delay_seconds.restype = c.c_double
            lib.oracle_delay_seconds.argtypes = [c.c_double] * 3
            lib.oracle_shift_real.restype = c.c_double
            lib.oracle_shift_real.argtypes = [c.c_double] * 4
            lib.oracle_shift_table.restype = c.c_int
            lib.oracle_shift_table.argtypes = [c.c_int, c.c_double, c.c_double, c.c_double,
                                               c.c_void_p, c.c_int, c.c_void_p, c.c_void_p]
            for name in ("oracle_dedisperse_u8", "oracle_dedisperse_u16", "oracle_dedisperse_u4"):
                f = getattr(lib, name)
                f.restype = None
                f.argtypes = [c.c_void_p, c.c_int, c.c_int64, c.c_void_p, c.c_int, c.c_int64,
                              c.c_void_p]
            lib.oracle_dedisperse_f32.restype = None
            lib.oracle_dedisperse_f32.argtypes = [c.c_void_p, c.c_int, c.c_int64, c.c_void_p,
                                                  c.c_int, c.c_int64, c.c_void_p, c.c_void_p]
            lib.oracle_dedisperse_points.restype = None
            lib.oracle_dedisperse_points.argtypes = [c.c_void_p, c.c_int, c.c_int, c.c_int64,
                                                     c.c_void_p, c.c_void_p, c.c_void_p,
                                                     c.c_int64, c.c_void_p, c.c_void_p,
                                                     c.c_void_p]
            lib.oracle_bin_time.restype = None
            lib.oracle_bin_time.argtypes = [c.c_void_p, c.c_int, c.c_int, c.c_int64, c.c_int, c.c_void_p]
            lib.oracle_omp_threads.restype = c.c_int
            _lib = lib
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def c_dm() -> float:
    return _load().oracle_c_dm()


def delay_seconds(dm: float, f_low_MHz: float, f_high_MHz: float) -> float:
    """Eq. 1."""
    return _load().oracle_delay_seconds(float(dm), float(f_low_MHz), float(f_high_MHz))


def shift_real(dm: float, f_c_MHz: float, f_high_MHz: float, tsamp_s: float) -> float:
    return _load().oracle_shift_real(float(dm), float(f_c_MHz), float(f_high_MHz), float(tsamp_s))


def shift_table(nchans: int, f_high_MHz: float, chan_bw_MHz: float, tsamp_s: float, dm_list):
    """Eq. 7 x DM / tsamp, rint.  Returns (int32 [ndm, nchans], max_shift)."""
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    table = np.empty((dm.size, nchans), dtype=np.int32)
    mx = ctypes.c_int32(0)
    rc = _load().oracle_shift_table(int(nchans), float(f_high_MHz), float(chan_bw_MHz),
                                    float(tsamp_s), _ptr(dm), int(dm.size), _ptr(table),
                                    ctypes.byref(mx))
    if rc != 0:
        raise ValueError("oracle_shift_table: shift negative or beyond int32")
    return table, int(mx.value)


def _dtype_code(x: np.ndarray) -> int:
    for code, dt in _NP_DTYPE.items():
        if x.dtype == dt:
            return code
    raise TypeError("oracle: unsupported input dtype %s" % x.dtype)


def dedisperse(x: np.ndarray, table: np.ndarray, out_len: int):
    """Eq. 3 / Alg. 1 for the DM rows in ``table`` ([ndm, nchans] int32).

    ``out_len`` is nsamps - max shift of the FULL plan (reading R5); ``table`` may hold any
    subset of the plan's rows.  Returns uint32 [ndm, out_len] for integer input, or
    (float64 sums, float64 sums of |in|) for float32 input.
    """
    assert x.ndim == 2 and x.flags.c_contiguous
    table = np.ascontiguousarray(table, dtype=np.int32)
    nchans, nsamps = x.shape
    ndm = table.shape[0]
    assert table.shape == (ndm, nchans)
    assert out_len >= 0 and (table.size == 0 or int(table.max()) + out_len <= nsamps)
    code = _dtype_code(x)
    lib = _load()
    if code == F32:
        out = np.empty((ndm, out_len), dtype=np.float64)
        ab = np.empty((ndm, out_len), dtype=np.float64)
        lib.oracle_dedisperse_f32(_ptr(x), nchans, nsamps, _ptr(table), ndm, out_len,
                                  _ptr(out), _ptr(ab))
        return out, ab
    out = np.empty((ndm, out_len), dtype=np.uint32)
    fn = lib.oracle_dedisperse_u8 if code == U8 else lib.oracle_dedisperse_u16
    fn(_ptr(x), nchans, nsamps, _ptr(table), ndm, out_len, _ptr(out))
    return out


def dedisperse_u4(xp: np.ndarray, table: np.ndarray, out_len: int) -> np.ndarray:
    """Eq. 3 on packed 4-bit input: ``xp`` is uint8 [nchans, nsamps/2], sample t of a channel in
    nibble t & 1 (low first) of byte t >> 1 (reading R14).  Returns uint32 [ndm, out_len]."""
    assert xp.ndim == 2 and xp.flags.c_contiguous and xp.dtype == np.uint8
    table = np.ascontiguousarray(table, dtype=np.int32)
    nchans, nbytes = xp.shape
    nsamps = 2 * nbytes
    ndm = table.shape[0]
    assert table.shape == (ndm, nchans)
    assert out_len >= 0 and (table.size == 0 or int(table.max()) + out_len <= nsamps)
    out = np.empty((ndm, out_len), dtype=np.uint32)
    _load().oracle_dedisperse_u4(_ptr(xp), nchans, nsamps, _ptr(table), ndm, out_len, _ptr(out))
    return out


def bin_time(x: np.ndarray, factor: int, packed_u4: bool = False) -> np.ndarray:
    """Reading R15: out[c][t] = sum of `factor` consecutive samples (trailing partial bin dropped).
    uint8 -> uint16, float32 -> float64 (exact reference for the float32 kernel), packed 4-bit
    (``packed_u4``: x is uint8 [nchans, nsamps/2]) -> uint8."""
    assert x.ndim == 2 and x.flags.c_contiguous and factor >= 1
    lib = _load()
    if packed_u4:
        assert x.dtype == np.uint8
        nchans, nsamps, code, odt = x.shape[0], 2 * x.shape[1], 3, np.uint8
    else:
        code = _dtype_code(x)
        assert code in (U8, F32)
        nchans, nsamps = x.shape
        odt = np.uint16 if code == U8 else np.float64
    out = np.empty((nchans, nsamps // factor), dtype=odt)
    lib.oracle_bin_time(_ptr(x), code, nchans, nsamps, int(factor), _ptr(out))
    return out


def dedisperse_points(x: np.ndarray, table: np.ndarray, pd, pt):
    """The same definition for single outputs (d, t) = (pd[i], pt[i]), one by one."""
    assert x.ndim == 2 and x.flags.c_contiguous
    table = np.ascontiguousarray(table, dtype=np.int32)
    nchans, nsamps = x.shape
    pd = np.ascontiguousarray(pd, dtype=np.int32)
    pt = np.ascontiguousarray(pt, dtype=np.int64)
    assert pd.shape == pt.shape and pd.ndim == 1
    if pd.size:
        assert 0 <= pd.min() and pd.max() < table.shape[0] and pt.min() >= 0
        assert int((table[pd].max(axis=1) + pt).max()) < nsamps
    code = _dtype_code(x)
    lib = _load()
    if code == F32:
        out = np.empty(pd.size, dtype=np.float64)
        ab = np.empty(pd.size, dtype=np.float64)
        lib.oracle_dedisperse_points(_ptr(x), code, nchans, nsamps, _ptr(table), _ptr(pd),
                                     _ptr(pt), pd.size, None, _ptr(out), _ptr(ab))
        return out, ab
    out = np.empty(pd.size, dtype=np.uint32)
    lib.oracle_dedisperse_points(_ptr(x), code, nchans, nsamps, _ptr(table), _ptr(pd),
                                 _ptr(pt), pd.size, _ptr(out), None, None)
    return out


def omp_threads() -> int:
    """Threads the oracle's OpenMP loops actually use (reported as cpu_baseline.cores)."""
    return int(_load().oracle_omp_threads())
