"""-m "not gpu": the tiled OpenMP CPU kernel (cpu_tiled/, Algorithm 2, SURVEY.md 8(f)
rank 4) against the plain oracle, bit for bit on uint8 input.  It is a baseline, not the product
and not the oracle: nothing under paper_2311_05341_b200/ or oracle/ may import it."""
import os
import re

import numpy as np
import pytest

from cpu_tiled import tiled

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CASES = [
    # nchans, nsamps, ndm, dm_step, f_high, band, tsamp: ragged in time, DM and channel tiles
    (37, 5003, 19, 3.0, 1500.0, 300.0, 64e-6),
    (64, 9001, 33, 1.0, 1550.0, 400.0, 64e-6),
    (300, 3000, 17, 0.1, 190.0, 60.0, 655.36e-6),
    (1, 100, 1, 5.0, 1500.0, 1.0, 1e-3),
    (520, 4200, 9, 2.0, 1500.0, 300.0, 64e-6),
]


@pytest.mark.parametrize("case", CASES)
def test_tiled_kernel_equals_oracle_for_every_candidate_tile(oracle, case):
    nchans, nsamps, ndm, step, f_high, band, tsamp = case
    rng = np.random.default_rng([nchans, nsamps, ndm, 12])
    x = rng.integers(0, 256, (nchans, nsamps), dtype=np.uint8)
    dms = np.arange(ndm) * step
    tab, mx = oracle.shift_table(nchans, f_high, -band / nchans, tsamp, dms)
    out_len = nsamps - mx
    ref = oracle.dedisperse(x, tab, out_len)
    tiles = list(tiled.CANDIDATES) + [(7, 3, 5, 0), (33, 2, 256, 1), (4096, 64, 1, 0), (100, 1, 100, 1)]
    for tile in tiles:
        got = tiled.dedisperse_u8(x, tab, out_len, tile)
        assert np.array_equal(got, ref), tile


def test_tiled_kernel_all_255_many_channels(oracle):
    # more than 256 channels of 255 per 16-bit channel tile would overflow: D_f <= 256 is enforced
    nchans = 1031
    x = np.full((nchans, 900), 255, dtype=np.uint8)
    tab, mx = oracle.shift_table(nchans, 1500.0, -300.0 / nchans, 64e-6, [0.0, 3.0, 40.0])
    for tile in ((512, 2, 256, 1), (512, 2, 64, 0)):
        assert (tiled.dedisperse_u8(x, tab, 900 - mx, tile) == 255 * nchans).all()
    with pytest.raises(ValueError):
        tiled.dedisperse_u8(x, tab, 900 - mx, (512, 2, 257, 1))
    with pytest.raises(ValueError):
        tiled.dedisperse_u8(x, tab, 900 - mx, (8192, 2, 16, 0))


def test_tiled_baseline_is_not_on_any_product_or_oracle_path():
    pat = re.compile(r"cpu_tiled|dedisp_tiled|libtiled")
    for sub in ("paper_2311_05341_b200", "oracle", "include"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, sub)):
            for fn in files:
                if fn.endswith((".py", ".c", ".h", ".cu", ".cpp")):
                    with open(os.path.join(dirpath, fn)) as f:
                        assert not pat.search(f.read()), os.path.join(dirpath, fn)
    with open(os.path.join(ROOT, "cpu_tiled", "tiled.py")) as f:
        src = f.read()
    assert "import oracle" not in src and "from oracle" not in src and "paper_2311_05341_b200 import" not in src
