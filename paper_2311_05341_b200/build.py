"""Build libdd.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2311_05341_b200.build [--force] [--verbose] [--tuning]

--tuning adds -DDD_TUNING and writes a SEPARATE library, libdd_tuning.so: the A/B kernel shapes of
profiles/r02_tuning.md and the DD_FORCE_VARIANT / DD_PANEL / DD_HOST_TAPER environment variables exist
only there.  libdd.so is never a tuning build; binding.use_tuning_library() (before the first call into
the library) makes a process load the tuning one instead.

The .so is git-ignored and travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(_ROOT, "include")
LIB = os.path.join(_HERE, "libdd.so")
LIB_TUNING = os.path.join(_HERE, "libdd_tuning.so")
SOURCES = ["dd_host.cpp", "dd_kernels.cu", "dd_api.cu", "dd_survey.cu", "dd_probe.cu", "dd_noalloc.cu"]
HEADERS = [os.path.join(CSRC, "dd_internal.h"), os.path.join(INCLUDE, "dd.h")]

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "--cudart", "static",
    "-Xcompiler", "-fPIC,-O2,-ffp-contract=off,-Wall",
    "-shared",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, tuning: bool = False) -> str:
    lib = LIB_TUNING if tuning else LIB
    if not force and not needs_build(lib):
        return lib
    tmp = lib + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + ["-I", INCLUDE, "-I", CSRC]
    if tuning:
        cmd += ["-DDD_TUNING"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-o", tmp]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout)
    if res.returncode != 0:
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("nvcc failed (exit %d): %s" % (res.returncode, " ".join(cmd)))
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, tuning="--tuning" in sys.argv))
