"""Pins for the CPU oracle (-m "not gpu").  Each test checks oracle/dedisp_oracle.c against
something OTHER than itself: values the specification prints (tests/golden/*.json, each with
its citation), closed forms, invariants, special cases that reduce to a numpy routine, and a
literal brute-force enumeration on tiny inputs.  A dropped term, wrong sign, wrong index or
transposed operand anywhere in the oracle fails at least one of these.
"""
import zlib

import numpy as np
import pytest

from paper_2311_05341_b200 import workloads as W


# --------------------------------------------------------------------------- delay law
def test_hand_value_delay(oracle, golden):
    # Eq. 1 with north_star's constant: DM=100, 1400 vs 1500 MHz -> 27.3 ms
    h = golden("shift_pins.json")["hand"]
    tau = oracle.delay_seconds(h["dm"], h["f_low"], h["f_high"])
    assert abs(tau - h["delay_s"]) < 5e-12
    assert abs(tau * 1e3 - 27.3) < 0.05
    assert oracle.c_dm() == 4148.808
    # arithmetic by hand, independent of the C code: 4148.808*100*(1/1.96e6 - 1/2.25e6)
    by_hand = 414880.8 * (2.25e6 - 1.96e6) / (1.96e6 * 2.25e6)
    assert abs(tau - by_hand) < 1e-15
    assert abs(oracle.shift_real(h["dm"], h["f_low"], h["f_high"], h["tsamp"]) - h["real_shift"]) < 1e-4
    tab, _ = oracle.shift_table(2, h["f_high"], h["f_low"] - h["f_high"], h["tsamp"], [h["dm"]])
    assert tab.tolist() == [[0, h["shift"]]]


def test_delay_sign_and_scaling(oracle):
    # lower frequency arrives later (positive delay); linear in DM; zero at equal frequency
    assert oracle.delay_seconds(50, 1200, 1500) > 0
    assert oracle.delay_seconds(50, 1500, 1500) == 0
    a, b = oracle.delay_seconds(10, 1000, 1400), oracle.delay_seconds(30, 1000, 1400)
    assert abs(b - 3 * a) < 1e-15
    # quadratic law: 1/f^2 dependence, (1/500^2 - 1/1000^2) = 3e-6
    assert abs(oracle.delay_seconds(1, 500, 1000) - 4148.808 * 3e-6) < 1e-15


def test_four_channel_rows(oracle, golden):
    g = golden("shift_pins.json")["four_channel"]
    for dm, row in g["rows"].items():
        tab, mx = oracle.shift_table(g["nchans"], g["f_high"], g["chan_bw"], g["tsamp"], [float(dm)])
        assert tab[0].tolist() == row
        assert mx == row[-1]
    for dm, raw in g["raw"].items():
        for c, r in enumerate(raw):
            x = oracle.shift_real(float(dm), g["f_high"] + c * g["chan_bw"], g["f_high"], g["tsamp"])
            assert abs(x - r) < 6e-5


def test_half_to_even_through_formula(oracle, golden):
    # the only pin that separates rint (ties-to-even) from floor(x+0.5)
    for g in golden("shift_pins.json")["half_even"]:
        x = oracle.shift_real(g["dm"], g["f_high"] + g["chan_bw"], g["f_high"], g["tsamp"])
        assert x == g["real"]
        tab, _ = oracle.shift_table(2, g["f_high"], g["chan_bw"], g["tsamp"], [g["dm"]])
        assert tab.tolist() == [[0, g["shift"]]]


@pytest.mark.parametrize("name", list(W.CONFIGS))
def test_config_tables_match_survey(oracle, golden, name):
    g = golden("shift_pins.json")["configs"][name]
    cfg = W.CONFIGS[name]
    tab, mx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    assert tab.shape == (cfg.ndm, cfg.nchans) and tab.dtype == np.int32
    assert mx == g["max_shift"] == int(tab.max())
    assert cfg.nsamps - mx == g["out_len"]
    assert int(tab.astype(np.int64).sum()) == g["sum"]
    assert zlib.crc32(tab.astype("<i4").tobytes()) == int(g["crc32"], 16)
    for d, c, s in g["spots"]:
        assert tab[d, c] == s
    if "row17_first8" in g:
        assert tab[17, :8].tolist() == g["row17_first8"]
        assert tab[17, -8:].tolist() == g["row17_last8"]
    # invariants (SURVEY.md 8c "Table invariants")
    assert not tab[:, 0].any() and not tab[0].any()
    assert (np.diff(tab, axis=1) >= 0).all() and (np.diff(tab, axis=0) >= 0).all()


@pytest.mark.parametrize("name", list(W.CONFIGS))
def test_table_independent_evaluation_order(oracle, name):
    # Independently written numpy evaluations in FOUR different double operation orders, and one in
    # extended precision (numpy longdouble, 64-bit mantissa on x86), give the oracle's integers for
    # every entry of every config table that does not sit within 1e-9 of a half-integer -- and no
    # entry of the five tables does: the rounding reading R3 is not fragile.
    cfg = W.CONFIGS[name]
    tab, _ = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    C = 4148.808
    fh, ts, dm = cfg.f_high, cfg.tsamp, cfg.dm_list
    f = fh + np.arange(cfg.nchans) * cfg.chan_bw
    orders = [
        np.outer(dm, C * (fh ** 2 - f ** 2) / (f ** 2 * fh ** 2) / ts),      # common denominator
        np.outer(dm / ts, C / f ** 2 - C / fh ** 2),                          # constant distributed
        np.outer(dm * C, (1.0 / f ** 2 - 1.0 / fh ** 2)) / ts,                # DM times constant first
        np.outer(dm, C * (1.0 / f - 1.0 / fh) * (1.0 / f + 1.0 / fh)) / ts,   # difference of squares
    ]
    fl = fh + np.arange(cfg.nchans, dtype=np.longdouble) * np.longdouble(cfg.chan_bw)
    ext = np.outer(dm.astype(np.longdouble),
                   np.longdouble(C) * (1 / fl ** 2 - 1 / np.longdouble(fh) ** 2)) / np.longdouble(ts)
    frac = np.abs(ext - np.floor(ext) - np.longdouble(0.5))
    assert frac.min() > 1e-9
    assert (np.rint(ext).astype(np.int64) == tab).all()
    for real in orders:
        assert (np.rint(real).astype(np.int32) == tab).all()


def test_shift_table_rejects_positive_bandwidth(oracle):
    with pytest.raises(ValueError):
        oracle.shift_table(4, 1500.0, +25.0, 1e-3, [100.0])


# --------------------------------------------------------------------------- transform
def _four_channel_plan(oracle, dms):
    return oracle.shift_table(4, 1500.0, -25.0, 1e-3, dms)


def test_closed_form_ramp(oracle):
    # in[c][t] = 100c + t  =>  out[d][t] = 600 + 4t + sum_c s(d,c)
    tab, mx = _four_channel_plan(oracle, [0.0, 50.0, 100.0])
    assert mx == 20
    nsamps, out_len = 32, 12
    x = (100 * np.arange(4)[:, None] + np.arange(nsamps)[None, :]).astype(np.uint16)
    out = oracle.dedisperse(x, tab, out_len)
    t = np.arange(out_len)
    for d, k in enumerate((600, 619, 639)):
        assert out[d].tolist() == (k + 4 * t).tolist()
    # same ramp as float32: exact in double
    o64, ab = oracle.dedisperse(x.astype(np.float32), tab, out_len)
    assert (o64 == out).all() and (ab == out).all()


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
def test_dm0_is_column_sum(oracle, dtype):
    rng = np.random.default_rng(5)
    x = rng.integers(0, 200, (37, 500)).astype(dtype)
    tab, mx = oracle.shift_table(37, 1400.0, -2.0, 256e-6, [0.0, 3.0, 11.0])
    out_len = 500 - mx
    out = oracle.dedisperse(x, tab, out_len)
    if dtype == np.float32:
        out = out[0]
    assert (out[0] == x.astype(np.int64).sum(axis=0)[:out_len]).all()


@pytest.mark.parametrize("dtype,val", [(np.uint8, 255), (np.uint16, 65535), (np.float32, 1.0)])
def test_constant_input(oracle, dtype, val):
    nchans = 300  # > 257: a 16-bit partial sum of 255s would overflow; uint32 must not
    x = np.full((nchans, 400), val, dtype=dtype)
    tab, mx = oracle.shift_table(nchans, 1500.0, -0.5, 64e-6, [0.0, 7.0, 20.0])
    out = oracle.dedisperse(x, tab, 400 - mx)
    if dtype == np.float32:
        out, ab = out
        assert (ab == nchans * val).all()
    assert (out == nchans * val).all()


def test_single_impulse_response(oracle):
    # one 1 at (c*, tau) in zeros -> out[d][tau - s(d,c*)] = 1, else 0
    nchans = 16
    tab, mx = oracle.shift_table(nchans, 1500.0, -12.5, 128e-6, np.arange(6) * 9.0)
    nsamps = 3 * mx + 20
    out_len = nsamps - mx
    cstar, tau = 11, mx + 5
    assert len(set(tab[:, cstar].tolist())) == 6  # six different landing times
    x = np.zeros((nchans, nsamps), dtype=np.uint8)
    x[cstar, tau] = 1
    out = oracle.dedisperse(x, tab, out_len)
    expect = np.zeros_like(out)
    for d in range(6):
        t = tau - tab[d, cstar]
        if 0 <= t < out_len:
            expect[d, t] = 1
    assert expect.sum() == 6 and (out == expect).all()


def test_shift_direction_lower_channels_read_later(oracle):
    # a transposed/negated shift would put the impulse at tau + s instead of tau - s
    tab, mx = _four_channel_plan(oracle, [100.0])
    x = np.zeros((4, 64), dtype=np.uint8)
    x[3, 40] = 9
    out = oracle.dedisperse(x, tab, 64 - mx)
    assert out[0, 40 - 20] == 9 and out[0].sum() == 9


def test_tiny_pulse_noise_free(oracle, golden):
    g = golden("tiny_pulse_pins.json")["noise_free"]
    cfg = W.CONFIGS["tiny"]
    tab, mx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    out_len = cfg.nsamps - mx
    x = W.make_input_numpy(cfg, tab, out_len, noise=False)
    out = oracle.dedisperse(x, tab, out_len).astype(np.int64)
    row = out[17]
    peak_t = np.nonzero(row == g["row17_peak_value"])[0].tolist()
    assert peak_t == g["row17_peak_t"]
    assert (np.delete(row, peak_t) == g["baseline"]).all()
    got = [int(out[d].max()) - g["baseline"] for d in range(g["dm_lo"], g["dm_lo"] + 15)]
    assert got == g["max_minus_baseline"]
    assert int(np.argmax(out.max(axis=1))) == 17


def test_tiny_pulse_noisy(oracle, golden):
    g = golden("tiny_pulse_pins.json")["noisy"]
    cfg = W.CONFIGS["tiny"]
    tab, mx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    out_len = cfg.nsamps - mx
    x = W.make_input_numpy(cfg, tab, out_len)
    out = oracle.dedisperse(x, tab, out_len).astype(np.int64)
    assert list(np.unravel_index(out.argmax(), out.shape)) == g["argmax"]
    assert out[17, 1000] == g["value_dm17_t1000"] and out[18].max() == g["max_dm18"]
    box = out[:, :-3] + out[:, 1:-2] + out[:, 2:-1] + out[:, 3:]
    assert box[17].max() == g["boxcar4_dm17"] and box[17].argmax() == g["boxcar4_dm17_t"]
    assert np.delete(box, 17, axis=0).max() == g["boxcar4_elsewhere_max"]


def _literal(x, tab, out_len):
    """Alg. 1 exactly as printed: t outer, dm, f inner; python ints/floats."""
    ndm, nchans = tab.shape
    out = [[0] * out_len for _ in range(ndm)]
    for t in range(out_len):
        for dm in range(ndm):
            s = 0
            for f in range(nchans):
                h = int(tab[dm][f])
                s = s + x[f][t + h].item()
            out[dm][t] = s
    return np.array(out)


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
@pytest.mark.parametrize("shape", [(8, 64, 5), (1, 40, 3), (5, 33, 1), (3, 50, 4)])
def test_brute_force_tiny(oracle, dtype, shape):
    nchans, nsamps, ndm = shape
    rng = np.random.default_rng(nchans * 1000 + nsamps)
    hi = {np.uint8: 256, np.uint16: 65536, np.float32: 1000}[dtype]
    x = rng.integers(0, hi, (nchans, nsamps)).astype(dtype)
    if dtype == np.float32:
        x = (x - 500).astype(np.float32) / 8  # exactly representable, sums exact in double
    tab, mx = oracle.shift_table(nchans, 1400.0, -30.0 if nchans > 1 else -1.0, 1e-3,
                                 np.arange(ndm) * 13.0)
    out_len = nsamps - mx
    assert out_len >= 1
    out = oracle.dedisperse(x, tab, out_len)
    ref = _literal(x, tab, out_len)
    if dtype == np.float32:
        assert (out[0] == ref).all()
        assert (out[1] == _literal(np.abs(x), tab, out_len)).all()
    else:
        assert (out == ref).all()


def test_out_len_one(oracle):
    # max_shift = nsamps - 1 -> exactly one output sample per DM
    tab, mx = _four_channel_plan(oracle, [0.0, 100.0])
    nsamps = mx + 1
    x = np.arange(4 * nsamps, dtype=np.uint16).reshape(4, nsamps)
    out = oracle.dedisperse(x, tab, 1)
    assert out[:, 0].tolist() == [int(x[:, 0].sum()), int(sum(x[c, tab[1, c]] for c in range(4)))]


def test_points_agree_with_definition(oracle):
    # dedisperse_points is the same definition per element; pin it against the plane,
    # which the tests above pin against the mathematics
    rng = np.random.default_rng(9)
    for dtype in (np.uint8, np.uint16, np.float32):
        x = rng.integers(0, 250, (24, 700)).astype(dtype)
        tab, mx = oracle.shift_table(24, 1300.0, -4.0, 128e-6, np.arange(9) * 2.5)
        out_len = 700 - mx
        pd = rng.integers(0, 9, 200)
        pt = rng.integers(0, out_len, 200)
        plane = oracle.dedisperse(x, tab, out_len)
        pts = oracle.dedisperse_points(x, tab, pd, pt)
        if dtype == np.float32:
            assert (pts[0] == plane[0][pd, pt]).all() and (pts[1] == plane[1][pd, pt]).all()
        else:
            assert (pts == plane[pd, pt]).all()


def test_row_subset_matches_full(oracle):
    cfg = W.CONFIGS["tiny"]
    tab, mx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    out_len = cfg.nsamps - mx
    x = W.noise_numpy(cfg)
    full = oracle.dedisperse(x, tab, out_len)
    rows = [0, 5, 31]
    assert (oracle.dedisperse(x, tab[rows], out_len) == full[rows]).all()


def test_f32_double_accumulation(oracle):
    # 1e8 + many small values: a float32 accumulator would lose them, double does not
    nchans = 64
    x = np.full((nchans, 8), 0.25, dtype=np.float32)
    x[0, :] = 1e8
    tab = np.zeros((1, nchans), dtype=np.int32)
    out, ab = oracle.dedisperse(x, tab, 8)
    assert (out == 1e8 + 63 * 0.25).all() and (ab == out).all()
    x[1, :] = -1e8
    out, ab = oracle.dedisperse(x, tab, 8)
    assert (out == 62 * 0.25).all() and (ab == 2e8 + 62 * 0.25).all()


# ------------------------------------------------------------------ packed 4-bit input (R14)
def _unpack_u4(xp):
    """numpy statement of reading R14: low nibble first."""
    out = np.empty((xp.shape[0], xp.shape[1] * 2), dtype=np.uint8)
    out[:, 0::2] = xp & 15
    out[:, 1::2] = xp >> 4
    return out


def test_u4_nibble_order_hand_row(oracle):
    # one channel, bytes 0x21 0x43 0x65 0x87 -> samples 1,2,3,4,5,6,7,8 (low nibble first)
    xp = np.array([[0x21, 0x43, 0x65, 0x87]], dtype=np.uint8)
    tab = np.zeros((1, 1), dtype=np.int32)
    assert oracle.dedisperse_u4(xp, tab, 8).tolist() == [[1, 2, 3, 4, 5, 6, 7, 8]]
    # a shift of 3 reads samples 4.. ; two channels with shifts (0, 3): 1+4, 2+5, ...
    xp2 = np.vstack([xp, xp])
    tab2 = np.array([[0, 3]], dtype=np.int32)
    assert oracle.dedisperse_u4(xp2, tab2, 5).tolist() == [[5, 7, 9, 11, 13]]


@pytest.mark.parametrize("shape", [(8, 64, 5), (1, 40, 3), (5, 34, 1), (3, 50, 4)])
def test_u4_equals_u8_transform_of_unpacked_block_and_brute_force(oracle, shape):
    nchans, nsamps, ndm = shape
    rng = np.random.default_rng([nchans, nsamps, ndm, 4])
    xp = rng.integers(0, 256, (nchans, nsamps // 2), dtype=np.uint8)
    x8 = _unpack_u4(xp)
    tab = np.sort(rng.integers(0, nsamps // 3, (ndm, nchans)), axis=1).astype(np.int32)
    out_len = nsamps - int(tab.max())
    got = oracle.dedisperse_u4(xp, tab, out_len)
    assert np.array_equal(got, oracle.dedisperse(x8, tab, out_len))
    assert np.array_equal(got, _literal(x8, tab, out_len))


def test_u4_constant_fifteen(oracle):
    xp = np.full((300, 50), 0xFF, dtype=np.uint8)
    tab = np.tile(np.arange(300, dtype=np.int32) % 7, (2, 1))
    assert (oracle.dedisperse_u4(xp, tab, 90) == 15 * 300).all()


# ------------------------------------------------------------------ time binning (R15)
def test_bin_time_hand_row_and_dropped_tail(oracle):
    x = np.array([[1, 2, 3, 4, 5, 6, 7], [250, 255, 255, 255, 0, 1, 9]], dtype=np.uint8)
    assert oracle.bin_time(x, 2).tolist() == [[3, 7, 11], [505, 510, 1]]      # 7th sample dropped
    assert oracle.bin_time(x, 4).tolist() == [[10], [1015]]
    xp = np.array([[0x21, 0x43, 0xFF, 0xFF]], dtype=np.uint8)                   # samples 1,2,3,4,15,15,15,15
    assert oracle.bin_time(xp, 4, packed_u4=True).tolist() == [[10, 60]]


@pytest.mark.parametrize("factor", [2, 4, 8, 16])
def test_bin_time_equals_numpy_reshape_sum(oracle, factor):
    rng = np.random.default_rng(factor)
    x8 = rng.integers(0, 256, (5, 1003), dtype=np.uint8)
    n = 1003 // factor
    assert np.array_equal(oracle.bin_time(x8, factor),
                          x8[:, :n * factor].reshape(5, n, factor).astype(np.uint32).sum(axis=2))
    xf = rng.standard_normal((3, 517)).astype(np.float32)
    n = 517 // factor
    assert np.allclose(oracle.bin_time(xf, factor),
                       xf[:, :n * factor].astype(np.float64).reshape(3, n, factor).sum(axis=2), rtol=0, atol=1e-12)
    xp = rng.integers(0, 256, (4, 400), dtype=np.uint8)
    n = 800 // factor
    assert np.array_equal(oracle.bin_time(xp, factor, packed_u4=True),
                          _unpack_u4(xp)[:, :n * factor].reshape(4, n, factor).astype(np.uint32).sum(axis=2))
