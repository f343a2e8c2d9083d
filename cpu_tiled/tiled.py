"""ctypes face of cpu_tiled/dedisp_tiled.c: the paper's tiled OpenMP CPU kernel (Algorithm 2,
PAPER.md:91-141) as a STRONGER CPU BASELINE beside the plain oracle.  Not the product, not the
oracle: only tests/ and bench.py's ``cpu_baseline_tiled`` leg may import this module, and it
imports nothing from ``oracle`` or ``paper_2311_05341_b200``.

Built with ``gcc -O3 -march=native -mprefer-vector-width=512 -fopenmp`` on the machine that runs it (the .so name carries a
hash of the CPU's feature flags, so a library built elsewhere is never loaded).
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dedisp_tiled.c")
_lock = threading.Lock()
_lib = None

# (D_t, D_dm, D_f, acc16) candidates (the paper tunes the tile sizes per CPU and plan);
# acc16 = 0 is the printed `int S[D_t]`, acc16 = 1 keeps the channel tile's partial sum in uint16
CANDIDATES = ((4096, 8, 8, 0), (2048, 8, 64, 0), (4096, 4, 128, 0),
              (4096, 8, 64, 1), (4096, 8, 256, 1), (2048, 16, 128, 1), (4096, 4, 256, 1))
DEFAULT_TILE = (4096, 8, 8, 0)


def _cpu_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    return hashlib.sha1(flags.encode()).hexdigest()[:10]


def lib_path() -> str:
    return os.path.join(_HERE, "libtiled_%s.so" % _cpu_tag())


def build(force: bool = False) -> str:
    path = lib_path()
    if not force and os.path.exists(path) and os.path.getmtime(path) >= os.path.getmtime(_SRC):
        return path
    tmp = path + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-std=c99", "-O3", "-march=native", "-mprefer-vector-width=512", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", tmp, _SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, path)
    return path


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            c = ctypes
            lib.tiled_dedisperse_u8.restype = c.c_int
            lib.tiled_dedisperse_u8.argtypes = [c.c_void_p, c.c_int, c.c_int64, c.c_void_p, c.c_int,
                                                c.c_int64, c.c_void_p, c.c_int, c.c_int, c.c_int, c.c_int]
            lib.tiled_omp_threads.restype = c.c_int
            _lib = lib
    return _lib


def omp_threads() -> int:
    return int(_load().tiled_omp_threads())


def dedisperse_u8(x: np.ndarray, table: np.ndarray, out_len: int, tile=DEFAULT_TILE) -> np.ndarray:
    """Algorithm 2 on uint8 ``x`` [nchans, nsamps] for the DM rows of ``table`` ([ndm, nchans] int32
    shifts from the caller).  Returns uint32 [ndm, out_len] raw sums."""
    assert x.ndim == 2 and x.dtype == np.uint8 and x.flags.c_contiguous
    table = np.ascontiguousarray(table, dtype=np.int32)
    nchans, nsamps = x.shape
    ndm = table.shape[0]
    assert table.shape == (ndm, nchans)
    assert out_len >= 0 and (table.size == 0 or int(table.max()) + out_len <= nsamps)
    out = np.empty((ndm, out_len), dtype=np.uint32)
    rc = _load().tiled_dedisperse_u8(x.ctypes.data, nchans, nsamps, table.ctypes.data, ndm, out_len,
                                     out.ctypes.data, int(tile[0]), int(tile[1]), int(tile[2]),
                                     int(tile[3]) if len(tile) > 3 else 0)
    if rc != 0:
        raise ValueError("tiled_dedisperse_u8: bad tile %r" % (tile,))
    return out
