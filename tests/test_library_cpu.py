"""-m "not gpu": the C-ABI library loads, exports every symbol include/dd.h declares, and its
HOST delay-table builder (no GPU involved) equals the oracle's table bit for bit.  No compute
entry point is called here."""
import ctypes
import os
import re
import zlib

import numpy as np
import pytest

from paper_2311_05341_b200 import binding as B
from paper_2311_05341_b200 import build as dd_build
from paper_2311_05341_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    dd_build.build()


def test_header_symbols_exported():
    with open(os.path.join(ROOT, "include", "dd.h")) as f:
        text = f.read()
    declared = set(re.findall(r"\b(dd_[a-z_]+)\s*\(", text))
    assert declared == set(B.SYMBOLS)
    raw = ctypes.CDLL(B.LIB_PATH)
    for name in declared:
        assert hasattr(raw, name), name


def test_version_and_strerror():
    assert "sm_100a" in B.version()
    assert B.strerror(0) == "ok"
    for code in range(-7, 0):
        assert B.strerror(code) not in ("ok", "unknown status")
    assert B.strerror(-99) == "unknown status"


@pytest.mark.parametrize("name", list(W.CONFIGS))
def test_host_table_equals_oracle_and_pins(oracle, golden, name):
    cfg = W.CONFIGS[name]
    g = golden("shift_pins.json")["configs"][name]
    tab, mx = B.dd_shift_table_build(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    otab, omx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    assert mx == omx == g["max_shift"]
    assert np.array_equal(tab, otab)
    assert zlib.crc32(tab.astype("<i4").tobytes()) == int(g["crc32"], 16)


def test_host_table_small_pins(golden):
    g = golden("shift_pins.json")
    fc = g["four_channel"]
    for dm, row in fc["rows"].items():
        tab, mx = B.dd_shift_table_build(fc["nchans"], fc["f_high"], fc["chan_bw"], fc["tsamp"], [float(dm)])
        assert tab[0].tolist() == row and mx == row[-1]
    for he in g["half_even"]:
        tab, _ = B.dd_shift_table_build(2, he["f_high"], he["chan_bw"], he["tsamp"], [he["dm"]])
        assert tab.tolist() == [[0, he["shift"]]]
    h = g["hand"]
    tab, _ = B.dd_shift_table_build(2, h["f_high"], h["f_low"] - h["f_high"], h["tsamp"], [h["dm"]])
    assert tab.tolist() == [[0, h["shift"]]]


def test_host_table_random_plans_equal_oracle(oracle):
    rng = np.random.default_rng(7)
    for _ in range(25):
        nchans = int(rng.integers(1, 300))
        f_high = float(rng.uniform(150, 2000))
        bw = -float(rng.uniform(0.001, 0.9)) * f_high / (nchans + 1)
        tsamp = float(10 ** rng.uniform(-5, -3))
        dms = np.sort(rng.uniform(0, 500, int(rng.integers(1, 40))))
        tab, mx = B.dd_shift_table_build(nchans, f_high, bw, tsamp, dms)
        otab, omx = oracle.shift_table(nchans, f_high, bw, tsamp, dms)
        assert mx == omx and np.array_equal(tab, otab)


@pytest.mark.parametrize("kwargs", [
    dict(nchans=0), dict(f_high=0.0), dict(f_high=-1.0), dict(chan_bw=0.0), dict(chan_bw=1.0),
    dict(tsamp=0.0), dict(tsamp=-1e-3), dict(dms=[-1.0]), dict(dms=[float("nan")]),
    dict(dms=[float("inf")]), dict(dms=[]), dict(nchans=100, chan_bw=-20.0),  # lowest channel <= 0 MHz
])
def test_host_table_rejects_bad_arguments(kwargs):
    a = dict(nchans=4, f_high=1500.0, chan_bw=-25.0, tsamp=1e-3, dms=[10.0])
    a.update(kwargs)
    with pytest.raises(B.DDError) as e:
        B.dd_shift_table_build(a["nchans"], a["f_high"], a["chan_bw"], a["tsamp"], a["dms"])
    assert e.value.status == B.DD_ERR_INVALID_ARG


def test_host_table_rejects_shift_beyond_int32():
    with pytest.raises(B.DDError) as e:
        B.dd_shift_table_build(2, 1500.0, -1400.0, 1e-9, [1e6])
    assert e.value.status == B.DD_ERR_SHIFT_TOO_LARGE


def test_plan_create_argument_errors_need_no_gpu():
    # These are rejected before any CUDA call, so they hold on a CPU-only box too.
    with pytest.raises(B.DDError) as e:
        B.Plan(4, 0, 1500.0, -25.0, 1e-3, [10.0], B.DD_U8)
    assert e.value.status == B.DD_ERR_INVALID_ARG
    with pytest.raises(B.DDError) as e:
        B.Plan(4, 32, 1500.0, -25.0, 1e-3, [10.0], 7)
    assert e.value.status == B.DD_ERR_INVALID_ARG
    with pytest.raises(B.DDError) as e:  # 60 >= 32 (SURVEY.md 8c closed-form pin)
        B.Plan(4, 32, 1500.0, -25.0, 1e-3, [0.0, 300.0], B.DD_U16)
    assert e.value.status == B.DD_ERR_SHIFT_TOO_LARGE
    with pytest.raises(B.DDError) as e:  # 65535 * 65538 >= 2^32
        B.Plan(65538, 64, 1500.0, -0.01, 1e-3, [0.0], B.DD_U16)
    assert e.value.status == B.DD_ERR_OVERFLOW
    with pytest.raises(B.DDError) as e:  # 255 * 16843010 >= 2^32
        B.Plan(16843010, 64, 1500.0, -1e-6, 1e-3, [0.0], B.DD_U8)
    assert e.value.status == B.DD_ERR_OVERFLOW


def test_product_path_does_not_import_oracle():
    # neither side imports the other; the product has no CPU fallback to route through
    pkg = os.path.join(ROOT, "paper_2311_05341_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cpp", ".h")):
                with open(os.path.join(dirpath, fn)) as f:
                    src = f.read()
                assert "import oracle" not in src and "from oracle" not in src, fn
                assert "dedisp_oracle" not in src and "liboracle" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            with open(os.path.join(ROOT, "oracle", fn)) as f:
                src = f.read()
            assert "import paper_2311_05341_b200" not in src and "from paper_2311_05341_b200" not in src
            assert "libdd" not in src and "dd.h" not in src


def test_header_is_plain_c(tmp_path):
    """include/dd.h is the C ABI: it must compile as C99 on its own (no C++ or CUDA types) and
    declare every symbol the binding loads."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    src = tmp_path / "use_dd.c"
    calls = "\n".join("    (void)&%s;" % name for name in B.SYMBOLS)
    src.write_text('#include "dd.h"\nint main(void) {\n%s\n    return DD_OK;\n}\n' % calls)
    inc = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include")
    res = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", inc, "-c",
                          str(src), "-o", str(tmp_path / "use_dd.o")], capture_output=True, text=True)
    assert res.returncode == 0, res.stderr


def test_survey_create_rejects_bad_ranges_without_a_gpu():
    """dd_survey_create validates its ranges before it touches the device."""
    import ctypes
    from paper_2311_05341_b200 import binding as B
    L = B.lib()
    h = ctypes.c_void_p(1)
    rng = (B._DmRange * 1)(B._DmRange(0.0, 1.0, 10, 3))          # 3 is not a binning factor
    assert L.dd_survey_create(ctypes.byref(h), 8, 1000, 1500.0, -1.0, 64e-6, ctypes.cast(rng, ctypes.c_void_p), 1, B.DD_U8) == B.DD_ERR_INVALID_ARG
    assert h.value is None
    rng = (B._DmRange * 1)(B._DmRange(0.0, 1.0, 0, 1))           # no trials
    assert L.dd_survey_create(ctypes.byref(h), 8, 1000, 1500.0, -1.0, 64e-6, ctypes.cast(rng, ctypes.c_void_p), 1, B.DD_U8) == B.DD_ERR_INVALID_ARG
    rng = (B._DmRange * 1)(B._DmRange(0.0, 1.0, 5, 2))           # 16-bit samples cannot be binned
    assert L.dd_survey_create(ctypes.byref(h), 8, 1000, 1500.0, -1.0, 64e-6, ctypes.cast(rng, ctypes.c_void_p), 1, B.DD_U16) == B.DD_ERR_UNSUPPORTED_PLAN
    assert L.dd_survey_create(ctypes.byref(h), 8, 1000, 1500.0, -1.0, 64e-6, None, 0, B.DD_U8) == B.DD_ERR_INVALID_ARG
    assert L.dd_survey_num_ranges(None) == B.DD_ERR_INVALID_ARG and L.dd_survey_plan(None, 0) is None
    L.dd_survey_destroy(None)
