"""-m gpu: the CUDA path (through the C ABI of libdd.so) against the CPU oracle, element by
element on the same seeded inputs.  Integer inputs: bit-exact.  float32: |gpu - oracle| <=
1e-4 * sum_c |in| per output (BASELINE.json north_star), and bit-exact on integer-valued
floats (every partial sum < 2^24, so any summation order gives the same float)."""

import numpy as np
import pytest

from paper_2311_05341_b200 import workloads as W

pytestmark = pytest.mark.gpu

F32_RTOL_OF_ABS_SUM = 1e-4


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device; the product has no CPU fallback")
    from paper_2311_05341_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def _torch_in(x):
    import torch
    if x.dtype == np.uint16:
        return torch.from_numpy(x.view(np.int16)).cuda().view(torch.uint16)
    return torch.from_numpy(x).cuda()


def gpu_dedisperse(B, x, f_high, chan_bw, tsamp, dms, stream=None):
    """Run the library on numpy input x [nchans, nsamps]; returns (out numpy, plan facts)."""
    import torch
    code = {np.dtype(np.uint8): B.DD_U8, np.dtype(np.uint16): B.DD_U16, np.dtype(np.float32): B.DD_F32}[x.dtype]
    plan = B.Plan(x.shape[0], x.shape[1], f_high, chan_bw, tsamp, dms, code)
    try:
        d_in = _torch_in(np.ascontiguousarray(x))
        odt = torch.float32 if code == B.DD_F32 else torch.int32
        d_out = torch.full((plan.ndm, plan.out_len), -7, dtype=odt, device="cuda")
        plan.execute(d_in, d_out, stream)
        torch.cuda.synchronize()
        out = d_out.cpu().numpy()
        if code != B.DD_F32:
            out = out.view(np.uint32)
        return out, plan.shift_table(), plan.out_len, plan.max_shift
    finally:
        plan.destroy()


def check_against_oracle(oracle, x, gpu_out, table, out_len):
    if x.dtype == np.float32:
        ref, ab = oracle.dedisperse(x, table, out_len)
        err = np.abs(gpu_out.astype(np.float64) - ref)
        tol = F32_RTOL_OF_ABS_SUM * ab
        assert (err <= tol).all(), "max err %g, worst err/tol %g" % (err.max(), (err / np.maximum(tol, 1e-300)).max())
        return float(err.max())
    ref = oracle.dedisperse(x, table, out_len)
    bad = np.argwhere(ref != gpu_out)
    assert bad.size == 0, "first mismatches (d,t): %s of %d" % (bad[:5].tolist(), len(bad))
    return 0.0


def _rand_input(rng, dtype, nchans, nsamps):
    if dtype == np.float32:
        return rng.standard_normal((nchans, nsamps)).astype(np.float32)
    hi = 256 if dtype == np.uint8 else 65536
    return rng.integers(0, hi, (nchans, nsamps)).astype(dtype)


# ------------------------------------------------------------------ configs[0]: tiny, full
def test_tiny_config_bit_exact_and_pulse(B, oracle, golden):
    cfg = W.CONFIGS["tiny"]
    otab, omx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    x = W.make_input_numpy(cfg, otab, cfg.nsamps - omx)
    out, tab, out_len, mx = gpu_dedisperse(B, x, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    assert np.array_equal(tab, otab) and mx == omx and out_len == 3966
    check_against_oracle(oracle, x, out, otab, out_len)
    # the paper's own check: the injected pulse is recovered at its DM
    g = golden("tiny_pulse_pins.json")["noisy"]
    box = out[:, :-3].astype(np.int64) + out[:, 1:-2] + out[:, 2:-1] + out[:, 3:]
    d, t = np.unravel_index(np.argmax(box), box.shape)
    assert (d, t) == (17, g["boxcar4_dm17_t"]) and box[d, t] == g["boxcar4_dm17"]
    assert out[17, 1000] == g["value_dm17_t1000"]


def test_tiny_noise_free_pulse_profile(B, oracle, golden):
    cfg = W.CONFIGS["tiny"]
    otab, omx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    x = W.make_input_numpy(cfg, otab, cfg.nsamps - omx, noise=False)
    out, _, _, _ = gpu_dedisperse(B, x, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    g = golden("tiny_pulse_pins.json")["noise_free"]
    peaks = (out.max(axis=1).astype(np.int64) - g["baseline"])[g["dm_lo"]:g["dm_lo"] + 15]
    assert peaks.tolist() == g["max_minus_baseline"]
    assert np.flatnonzero(out[17] == g["row17_peak_value"]).tolist() == g["row17_peak_t"]


# ------------------------------------------------------------------ closed forms on the GPU
def test_closed_form_ramp_all_dtypes(B):
    # in[c][t] = 100c + t => out[d][t] = 600 + 4t + sum_c s(d,c); table rows (0,3,6,10),(0,6,13,20)
    nsamps = 32
    ramp = 100 * np.arange(4)[:, None] + np.arange(nsamps)[None, :]
    for dt in (np.uint16, np.float32):
        out, tab, out_len, mx = gpu_dedisperse(B, ramp.astype(dt), 1500.0, -25.0, 1e-3, [0.0, 50.0, 100.0])
        assert mx == 20 and out_len == 12
        t = np.arange(12)
        for d, k in enumerate((600, 619, 639)):
            assert out[d].tolist() == (k + 4 * t).tolist()
    small = (10 * np.arange(4)[:, None] + np.arange(nsamps)[None, :]).astype(np.uint8)
    out, _, _, _ = gpu_dedisperse(B, small, 1500.0, -25.0, 1e-3, [0.0, 50.0, 100.0])
    for d, k in enumerate((60, 79, 99)):
        assert out[d].tolist() == (k + 4 * np.arange(12)).tolist()


@pytest.mark.parametrize("nchans", [256, 257, 258, 520, 1031])
def test_u8_packed_lane_flush_all_255(B, nchans):
    # a 16-bit lane holds at most 257 samples of 255: the flush must come in time
    x = np.full((nchans, 700), 255, dtype=np.uint8)
    out, _, _, _ = gpu_dedisperse(B, x, 1500.0, -300.0 / nchans, 64e-6, [0.0, 3.0, 40.0])
    assert (out == 255 * nchans).all()


def test_u16_all_max(B):
    nchans = 600
    x = np.full((nchans, 900), 65535, dtype=np.uint16)
    out, _, _, _ = gpu_dedisperse(B, x, 400.0, -0.05, 1e-4, [0.0, 1.0, 2.5])
    assert (out == 65535 * nchans).all()


def test_f32_all_ones(B):
    x = np.ones((300, 1500), dtype=np.float32)
    out, _, _, _ = gpu_dedisperse(B, x, 1500.0, -1.0, 64e-6, [0.0, 10.0, 20.0])
    assert (out == 300.0).all()


# ------------------------------------------------------------------ random plans, ragged everything
CASES = [
    # nchans, nsamps, ndm, dm_step, f_high, band, tsamp   (several tiles + ragged tails)
    (37, 5003, 19, 3.0, 1500.0, 300.0, 64e-6),
    (64, 9001, 33, 1.0, 1550.0, 400.0, 64e-6),
    (130, 4100, 70, 0.5, 400.0, 100.0, 256e-6),
    (16, 70001, 5, 11.0, 1400.0, 200.0, 32e-6),
    (300, 3000, 17, 0.1, 190.0, 60.0, 655.36e-6),
]


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
@pytest.mark.parametrize("case", CASES)
def test_random_plans_match_oracle(B, oracle, dtype, case):
    nchans, nsamps, ndm, step, f_high, band, tsamp = case
    rng = np.random.default_rng([nchans, nsamps, ndm])
    x = _rand_input(rng, dtype, nchans, nsamps)
    dms = np.arange(ndm) * step
    out, tab, out_len, mx = gpu_dedisperse(B, x, f_high, -band / nchans, tsamp, dms)
    otab, omx = oracle.shift_table(nchans, f_high, -band / nchans, tsamp, dms)
    assert np.array_equal(tab, otab) and mx == omx and out_len == nsamps - omx
    check_against_oracle(oracle, x, out, otab, out_len)


def test_f32_integer_valued_is_bit_exact(B, oracle):
    # pins the f32 kernel's indexing as tightly as the integer paths
    rng = np.random.default_rng(11)
    x = rng.integers(0, 256, (200, 6000)).astype(np.float32)
    dms = np.arange(40) * 2.0
    out, tab, out_len, _ = gpu_dedisperse(B, x, 1500.0, -1.5, 64e-6, dms)
    ref, _ = oracle.dedisperse(x, tab, out_len)
    assert np.array_equal(out.astype(np.float64), ref)


# ------------------------------------------------------------------ degenerate cases
@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
def test_single_dm_single_channel(B, oracle, dtype):
    rng = np.random.default_rng(3)
    x = _rand_input(rng, dtype, 1, 100)
    out, tab, out_len, mx = gpu_dedisperse(B, x, 1500.0, -1.0, 1e-3, [5.0])
    assert mx == 0 and out_len == 100 and tab.tolist() == [[0]]
    assert np.array_equal(out[0], x[0].astype(out.dtype))


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
def test_out_len_one(B, oracle, dtype):
    # max_shift = nsamps - 1: one output sample per DM
    rng = np.random.default_rng(4)
    tab, mx = B.dd_shift_table_build(4, 1500.0, -25.0, 1e-3, [0.0, 50.0, 100.0])
    x = _rand_input(rng, dtype, 4, mx + 1)
    if dtype == np.float32:
        x = np.rint(x * 8).astype(np.float32)
    out, tab2, out_len, _ = gpu_dedisperse(B, x, 1500.0, -25.0, 1e-3, [0.0, 50.0, 100.0])
    assert out_len == 1 and np.array_equal(tab, tab2)
    for d in range(3):
        assert float(out[d, 0]) == float(sum(float(x[c, tab[d, c]]) for c in range(4)))


def test_unsorted_and_repeated_dm_list(B, oracle):
    rng = np.random.default_rng(5)
    x = _rand_input(rng, np.uint8, 48, 4000)
    dms = np.array([30.0, 0.0, 12.5, 30.0, 7.0, 99.0, 1.0, 55.5, 0.0, 80.0] * 4)
    out, tab, out_len, _ = gpu_dedisperse(B, x, 1400.0, -2.0, 64e-6, dms)
    otab, _ = oracle.shift_table(48, 1400.0, -2.0, 64e-6, dms)
    assert np.array_equal(tab, otab)
    check_against_oracle(oracle, x, out, otab, out_len)


def test_rasterisation_panel_does_not_depend_on_dm_order(B):
    """The panel size (a DRAM-traffic heuristic, never a correctness matter) is taken from the shift span
    between the smallest and the largest DM, wherever they sit in dm_list: a descending list plans the
    same panel as the ascending one (round-2 advice: it used rows 0 and ndm-1 and fell back to one panel)."""
    dms = np.arange(480) * 0.5
    panels = []
    for order in (dms, dms[::-1].copy()):
        with B.Plan(2048, 60000, 1500.0, -300.0 / 2048, 64e-6, order, B.DD_U8) as plan:
            panels.append(plan.info("PANEL"))
            ndb = -(-plan.ndm // plan.info("D_DM"))
    assert panels[0] == panels[1] and 1 <= panels[0] < ndb   # more than one panel, so the order could matter


def test_single_impulse_response(B):
    # a single 1 at (c*, tau) in zeros -> out[d][tau - s(d,c*)] = 1 and 0 elsewhere
    nchans, nsamps, cstar, tau = 40, 3000, 29, 1777
    x = np.zeros((nchans, nsamps), dtype=np.uint16)
    x[cstar, tau] = 1
    dms = np.arange(24) * 4.0
    out, tab, out_len, _ = gpu_dedisperse(B, x, 1500.0, -5.0, 64e-6, dms)
    expect = np.zeros_like(out)
    for d in range(len(dms)):
        t = tau - tab[d, cstar]
        if 0 <= t < out_len:
            expect[d, t] = 1
    assert np.array_equal(out, expect)


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
def test_misaligned_input_pointer_and_odd_row_length(B, oracle, dtype):
    # rows that are not 4/8/16-byte aligned take the scalar path of the pre-pass
    import torch
    rng = np.random.default_rng(6)
    nchans, nsamps = 21, 2999
    x = _rand_input(rng, dtype, nchans, nsamps)
    if dtype == np.float32:
        x = np.rint(x * 16).astype(np.float32)
    dms = np.arange(9) * 7.0
    code = {np.uint8: B.DD_U8, np.uint16: B.DD_U16, np.float32: B.DD_F32}[dtype]
    plan = B.Plan(nchans, nsamps, 1500.0, -10.0, 64e-6, dms, code)
    flat = _torch_in(np.concatenate([np.zeros(1, dtype=dtype), x.ravel()]))
    d_in = flat[1:]  # element-misaligned view
    assert d_in.data_ptr() % 16 != 0
    odt = torch.float32 if code == B.DD_F32 else torch.int32
    d_out = torch.empty((plan.ndm, plan.out_len), dtype=odt, device="cuda")
    plan.execute(d_in.data_ptr(), d_out)
    torch.cuda.synchronize()
    out = d_out.cpu().numpy()
    out = out if code == B.DD_F32 else out.view(np.uint32)
    check_against_oracle(oracle, x, out, plan.shift_table(), plan.out_len)
    plan.destroy()


def test_repeat_execute_streams_and_host_path(B, oracle):
    import torch
    rng = np.random.default_rng(8)
    nchans, nsamps = 96, 20000
    dms = np.arange(50) * 3.0
    plan = B.Plan(nchans, nsamps, 1500.0, -3.0, 64e-6, dms, B.DD_U8)
    ref = None
    st = torch.cuda.Stream()
    for it in range(3):
        x = _rand_input(rng, np.uint8, nchans, nsamps)
        d_in = _torch_in(x)
        d_out = torch.empty((plan.ndm, plan.out_len), dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            plan.execute(d_in, d_out)  # picks up the current (side) stream
        st.synchronize()
        out = d_out.cpu().numpy().view(np.uint32)
        ref = oracle.dedisperse(x, plan.shift_table(), plan.out_len)
        assert np.array_equal(out, ref)
    # dd_execute_host on the last input
    h_in = torch.from_numpy(x).pin_memory()
    h_out = torch.empty((plan.ndm, plan.out_len), dtype=torch.int32).pin_memory()
    plan.execute_host(h_in, h_out)
    assert np.array_equal(h_out.numpy().view(np.uint32), ref)
    plan.destroy()


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
@pytest.mark.parametrize("case", CASES)
def test_host_path_pipelined_chunks_match_oracle(B, oracle, dtype, case):
    """dd_execute_host cuts the output into time chunks (input range = chunk + max_shift halo,
    strided 2-D copies on copy streams); 3 chunks forced here, pinned and pageable buffers,
    sentinel-filled output, ragged sizes, every dtype."""
    import torch
    nchans, nsamps, ndm, step, f_high, band, tsamp = case
    rng = np.random.default_rng([nchans, nsamps, ndm, 5])
    x = _rand_input(rng, dtype, nchans, nsamps)
    dms = np.arange(ndm) * step
    plan = B.Plan(nchans, nsamps, f_high, -band / nchans, tsamp, dms,
                  {np.uint8: B.DD_U8, np.uint16: B.DD_U16, np.float32: B.DD_F32}[dtype])
    plan.set_host_chunks(3)
    try:
        xt = torch.from_numpy(x.view(np.int16) if dtype == np.uint16 else x)
        odt = torch.float32 if dtype == np.float32 else torch.int32
        for pinned in (True, False):
            h_in = xt.pin_memory() if pinned else xt
            h_out = torch.full((plan.ndm, plan.out_len), -7, dtype=odt)
            if pinned:
                h_out = h_out.pin_memory()
            plan.execute_host(h_in, h_out)
            got = h_out.numpy()
            check_against_oracle(oracle, x, got if dtype == np.float32 else got.view(np.uint32),
                                 plan.shift_table(), plan.out_len)
            # the same block delivered time-major
            h_tm = xt.t().contiguous()
            h_tm = h_tm.pin_memory() if pinned else h_tm
            h_out.fill_(-7)
            plan.execute_host_tm(h_tm, h_out)
            got = h_out.numpy()
            check_against_oracle(oracle, x, got if dtype == np.float32 else got.view(np.uint32),
                                 plan.shift_table(), plan.out_len)
    finally:
        plan.destroy()


TM_CASES = [
    # nchans, nsamps: whole tiles, ragged both ways, rows not 4-byte aligned, tiny
    (256, 4096), (130, 5003), (37, 999), (1, 300), (129, 1000), (64, 70001),
    (128, 30002), (256, 10001),   # full tiles whose output rows start 1, 2 or 3 bytes off a word
]


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
@pytest.mark.parametrize("shape", TM_CASES)
def test_standalone_transpose_equals_numpy(B, dtype, shape):
    import torch
    nchans, nsamps = shape
    rng = np.random.default_rng([nchans, nsamps, 3])
    x_tm = np.ascontiguousarray(_rand_input(rng, dtype, nchans, nsamps).T)
    d_out = torch.empty((nchans, nsamps), dtype=_torch_in(x_tm[:1]).dtype, device="cuda")
    B.transpose(_torch_in(x_tm), d_out, nchans, nsamps,
                {np.uint8: B.DD_U8, np.uint16: B.DD_U16, np.float32: B.DD_F32}[dtype])
    torch.cuda.synchronize()
    got = d_out.view(torch.int16).cpu().numpy().view(np.uint16) if dtype == np.uint16 else d_out.cpu().numpy()
    assert np.array_equal(got, x_tm.T)


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
@pytest.mark.parametrize("shape", TM_CASES)
def test_time_major_input_matches_oracle_on_transposed_block(B, oracle, dtype, shape):
    """dd_execute_tm: the transpose pre-step.  The expected result is the
    oracle run on numpy's transpose of the same time-major block."""
    import torch
    nchans, nsamps = shape
    rng = np.random.default_rng([nchans, nsamps, 11])
    x_tm = np.ascontiguousarray(_rand_input(rng, dtype, nchans, nsamps).T)  # [nsamps][nchans]
    dms = np.arange(9) * 7.0
    f_high, chan_bw, tsamp = 1500.0, -200.0 / nchans, 64e-6
    code = {np.uint8: B.DD_U8, np.uint16: B.DD_U16, np.float32: B.DD_F32}[dtype]
    plan = B.Plan(nchans, nsamps, f_high, chan_bw, tsamp, dms, code)
    try:
        odt = torch.float32 if dtype == np.float32 else torch.int32
        d_out = torch.full((plan.ndm, plan.out_len), -7, dtype=odt, device="cuda")
        # second run from a device pointer that is only 1-element aligned
        for shift in (0, 1):
            flat = torch.empty(x_tm.size + shift, dtype=_torch_in(x_tm[:1]).dtype, device="cuda")
            view = flat[shift:].view(nsamps, nchans)
            view.copy_(_torch_in(x_tm))
            d_out.fill_(-7)
            plan.execute_tm(view, d_out)
            torch.cuda.synchronize()
            got = d_out.cpu().numpy()
            x_cm = np.ascontiguousarray(x_tm.T)
            check_against_oracle(oracle, x_cm, got if dtype == np.float32 else got.view(np.uint32),
                                 plan.shift_table(), plan.out_len)
    finally:
        plan.destroy()


# ------------------------------------------------------------------ packed 4-bit input (DD_U4)
U4_CASES = CASES + [(520, 3000, 9, 2.0, 1500.0, 300.0, 64e-6)]  # > 256 channels: flush path


@pytest.mark.parametrize("case", U4_CASES)
def test_u4_packed_input_matches_oracle(B, oracle, case):
    """Two samples per byte, low nibble first (reading R14): device path, host path (3 chunks,
    odd chunk lengths) and a byte-misaligned device pointer, bit-exact against oracle.dedisperse_u4."""
    import torch
    nchans, nsamps, ndm, step, f_high, band, tsamp = case
    nsamps -= nsamps & 1
    rng = np.random.default_rng([nchans, nsamps, ndm, 4])
    xp = rng.integers(0, 256, (nchans, nsamps // 2), dtype=np.uint8)
    dms = np.arange(ndm) * step
    plan = B.Plan(nchans, nsamps, f_high, -band / nchans, tsamp, dms, B.DD_U4)
    try:
        ref = oracle.dedisperse_u4(xp, plan.shift_table(), plan.out_len)
        d_out = torch.full((plan.ndm, plan.out_len), -7, dtype=torch.int32, device="cuda")
        for shift in (0, 1):
            flat = torch.empty(xp.size + shift, dtype=torch.uint8, device="cuda")
            view = flat[shift:].view(nchans, nsamps // 2)
            view.copy_(torch.from_numpy(xp))
            d_out.fill_(-7)
            plan.execute(view, d_out)
            torch.cuda.synchronize()
            assert np.array_equal(d_out.cpu().numpy().view(np.uint32), ref)
        plan.set_host_chunks(3)
        h_out = torch.full((plan.ndm, plan.out_len), -7, dtype=torch.int32).pin_memory()
        plan.execute_host(torch.from_numpy(xp).pin_memory(), h_out)
        assert np.array_equal(h_out.numpy().view(np.uint32), ref)
    finally:
        plan.destroy()


@pytest.mark.parametrize("shape", [(256, 4096), (130, 5002), (38, 1000), (2, 300), (600, 3000)])
def test_u4_time_major_matches_oracle(B, oracle, shape):
    """Packed 4-bit delivered time-major ([nsamps][nchans/2], even channel in the low nibble,
    reading R16) through dd_execute_tm and the chunked dd_execute_host_tm."""
    import torch
    nchans, nsamps = shape
    rng = np.random.default_rng([nchans, nsamps, 44])
    x8 = rng.integers(0, 16, (nchans, nsamps), dtype=np.uint8)
    xp_cm = W.pack_u4(x8)                                             # oracle input: packed along time
    x_tm = np.ascontiguousarray(x8.T)                                 # [nsamps][nchans]
    xp_tm = (x_tm[:, 0::2] | (x_tm[:, 1::2] << 4)).astype(np.uint8)   # packed along channels
    dms = np.arange(7) * 9.0
    with B.Plan(nchans, nsamps, 1500.0, -200.0 / nchans, 64e-6, dms, B.DD_U4) as plan:
        ref = oracle.dedisperse_u4(xp_cm, plan.shift_table(), plan.out_len)
        d_out = torch.full((plan.ndm, plan.out_len), -7, dtype=torch.int32, device="cuda")
        plan.execute_tm(torch.from_numpy(xp_tm).cuda(), d_out)
        torch.cuda.synchronize()
        assert np.array_equal(d_out.cpu().numpy().view(np.uint32), ref)
        plan.set_host_chunks(3)
        h_out = torch.full((plan.ndm, plan.out_len), -7, dtype=torch.int32).pin_memory()
        plan.execute_host_tm(torch.from_numpy(xp_tm).pin_memory(), h_out)
        assert np.array_equal(h_out.numpy().view(np.uint32), ref)


def test_u4_all_fifteen_and_errors(B):
    import torch
    nchans, nsamps = 1031, 2000
    dms = np.arange(5) * 1.0
    with B.Plan(nchans, nsamps, 1500.0, -0.1, 64e-6, dms, B.DD_U4) as plan:
        d_in = torch.full((nchans, nsamps // 2), 0xFF, dtype=torch.uint8, device="cuda")
        d_out = torch.empty((plan.ndm, plan.out_len), dtype=torch.int32, device="cuda")
        plan.execute(d_in, d_out)
        torch.cuda.synchronize()
        assert (d_out == 15 * nchans).all().item()
        with pytest.raises(B.DDError) as e:
            plan.execute_tm(d_in, d_out)
        assert e.value.status == B.DD_ERR_UNSUPPORTED_PLAN
    with pytest.raises(B.DDError) as e:
        B.Plan(8, 1001, 1500.0, -1.0, 64e-6, dms, B.DD_U4)  # odd nsamps: rows are not whole bytes
    assert e.value.status == B.DD_ERR_INVALID_ARG


# ------------------------------------------------------------------ large shifts: the DM-block ladder
LARGE_SHIFT_CASES = [
    # nchans, nsamps, ndm, dm_step, f_high, band, tsamp, expected: 0 = any rung (smaller stages may
    # do), 1 = a smaller DM block than the first choice, 2 = one DM per block
    (64, 12000, 40, 0.5, 400.0, 100.0, 64e-6, 0),   # ~150 samples per DM step at the bottom channel
    (64, 20000, 24, 2.0, 400.0, 100.0, 64e-6, 1),   # ~600
    (32, 90000, 13, 20.0, 400.0, 100.0, 64e-6, 2),  # ~6000: one DM per block
]


@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.float32])
@pytest.mark.parametrize("case", LARGE_SHIFT_CASES)
def test_large_shift_plans_fall_back_to_smaller_dm_blocks(B, oracle, dtype, case):
    """Large DM step x small sampling time (the regime of the paper's 'cache kernel',
    PAPER.md:153, 380): when the windows of a 12/16/32-DM block no longer fit shared memory the
    plan goes down its ladder (smaller stages first: 8 instead of 16 channels; then smaller DM
    blocks) and must still match the oracle.  `expect` (last field of a case): 0 = any rung (for
    8-bit input case 0 still fits the first DM block with 8-channel stages since the flush
    accumulators moved to tensor memory), 1 = a smaller DM block than the
    first choice, 2 = the last rung (one DM trial per block)."""
    nchans, nsamps, ndm, step, f_high, band, tsamp, expect = case
    rng = np.random.default_rng([nchans, nsamps, ndm, 77])
    x = _rand_input(rng, dtype, nchans, nsamps)
    dms = np.arange(ndm) * step
    code = {np.uint8: B.DD_U8, np.uint16: B.DD_U16, np.float32: B.DD_F32}[dtype]
    with B.Plan(nchans, nsamps, f_high, -band / nchans, tsamp, dms, code) as plan:
        first_choice = {np.uint8: 12, np.uint16: 16, np.float32: 32}[dtype]
        assert plan.info("D_DM") <= first_choice
        if expect >= 1:
            assert plan.info("D_DM") < first_choice, plan.info("D_DM")
        if expect == 2:
            assert plan.info("D_DM") == 1
    out, tab, out_len, mx = gpu_dedisperse(B, x, f_high, -band / nchans, tsamp, dms)
    check_against_oracle(oracle, x, out, tab, out_len)


# ------------------------------------------------------------------ time binning (dd_bin_time, R15)
BIN_SHAPES = [(64, 4096), (37, 5003), (5, 1001), (1, 70), (130, 20000),
              (12, 156250), (7, 30002)]   # rows that are not 16-byte aligned: the funnel-shift kernel


@pytest.mark.parametrize("factor", [2, 4, 8, 16])
@pytest.mark.parametrize("shape", BIN_SHAPES)
def test_bin_time_matches_oracle(B, oracle, shape, factor):
    import torch
    nchans, nsamps = shape
    rng = np.random.default_rng([nchans, nsamps, factor])
    nout = nsamps // factor
    # u8 -> u16, bit-exact (also from a 1-byte-misaligned device pointer)
    x8 = rng.integers(0, 256, (nchans, nsamps), dtype=np.uint8)
    ref8 = oracle.bin_time(x8, factor)
    for shift in (0, 1):
        flat = torch.empty(x8.size + shift, dtype=torch.uint8, device="cuda")
        view = flat[shift:].view(nchans, nsamps)
        view.copy_(torch.from_numpy(x8))
        d_out = torch.full((nchans, nout), -1, dtype=torch.int16, device="cuda")
        B.bin_time(view, d_out, nchans, nsamps, factor, B.DD_U8)
        torch.cuda.synchronize()
        assert np.array_equal(d_out.cpu().numpy().view(np.uint16), ref8)
    # packed u4 -> u8, bit-exact
    ns4 = nsamps - (nsamps & 1)
    xp = rng.integers(0, 256, (nchans, ns4 // 2), dtype=np.uint8)
    if ns4 // factor:
        d_out = torch.full((nchans, ns4 // factor), 7, dtype=torch.uint8, device="cuda")
        B.bin_time(torch.from_numpy(xp).cuda(), d_out, nchans, ns4, factor, B.DD_U4)
        torch.cuda.synchronize()
        assert np.array_equal(d_out.cpu().numpy(), oracle.bin_time(xp, factor, packed_u4=True))
    # f32: float accumulation of <= 16 terms against the double oracle, and bit-exact on integers
    xf = rng.standard_normal((nchans, nsamps)).astype(np.float32)
    d_out = torch.empty((nchans, nout), dtype=torch.float32, device="cuda")
    B.bin_time(torch.from_numpy(xf).cuda(), d_out, nchans, nsamps, factor, B.DD_F32)
    torch.cuda.synchronize()
    ab = oracle.bin_time(np.abs(xf), factor)
    assert (np.abs(d_out.cpu().numpy().astype(np.float64) - oracle.bin_time(xf, factor)) <= 1e-6 * ab + 1e-30).all()
    xi = rng.integers(0, 1000, (nchans, nsamps)).astype(np.float32)
    B.bin_time(torch.from_numpy(xi).cuda(), d_out, nchans, nsamps, factor, B.DD_F32)
    torch.cuda.synchronize()
    assert np.array_equal(d_out.cpu().numpy().astype(np.float64), oracle.bin_time(xi, factor))


def test_binned_range_pipeline_matches_oracle_chain(B, oracle):
    """One DM range of a Table-2 style plan: bin by 4, then dedisperse the
    binned block with tsamp*4 -- GPU chain against the oracle chain, bit-exact."""
    import torch
    nchans, nsamps, factor = 96, 40000, 4
    f_high, chan_bw, tsamp = 1500.0, -2.0, 64e-6
    dms = 100.0 + np.arange(40) * 2.0
    rng = np.random.default_rng(31)
    x8 = rng.integers(0, 256, (nchans, nsamps), dtype=np.uint8)
    nb = nsamps // factor
    d_bin = torch.empty((nchans, nb), dtype=torch.int16, device="cuda")
    B.bin_time(torch.from_numpy(x8).cuda(), d_bin, nchans, nsamps, factor, B.DD_U8)
    with B.Plan(nchans, nb, f_high, chan_bw, tsamp * factor, dms, B.DD_U16) as plan:
        d_out = torch.empty((plan.ndm, plan.out_len), dtype=torch.int32, device="cuda")
        plan.execute(d_bin.view(torch.uint16), d_out)
        torch.cuda.synchronize()
        otab, omx = oracle.shift_table(nchans, f_high, chan_bw, tsamp * factor, dms)
        ref = oracle.dedisperse(oracle.bin_time(x8, factor), otab, nb - omx)
        assert plan.out_len == nb - omx
        assert np.array_equal(d_out.cpu().numpy().view(np.uint32), ref)


@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
def test_multi_range_survey_matches_oracle_chain(B, oracle, dtype):
    """Three DM ranges with binning 1, 2, 4 (Table-2 style) through
    binding.Survey against the oracle chain (oracle.bin_time -> oracle.dedisperse) per range."""
    import torch
    nchans, nsamps = 80, 30000
    f_high, chan_bw, tsamp = 1500.0, -2.5, 64e-6
    ranges = [(0.0, 1.0, 20, 1), (20.0, 2.0, 15, 2), (50.0, 4.0, 10, 4)]
    rng = np.random.default_rng(17)
    x = _rand_input(rng, dtype, nchans, nsamps)
    code = B.DD_U8 if dtype == np.uint8 else B.DD_F32
    with B.Survey(nchans, nsamps, f_high, chan_bw, tsamp, ranges, code) as sv:
        outs = sv.execute(_torch_in(x))
        torch.cuda.synchronize()
        for (start, step, count, factor), got_t in zip(ranges, outs):
            dms = start + np.arange(count) * step
            if factor == 1:
                xb = x
            elif dtype == np.uint8:
                xb = oracle.bin_time(x, factor)                       # uint16
            else:
                xb = oracle.bin_time(x, factor).astype(np.float32)    # what the f32 kernel hands on
            otab, omx = oracle.shift_table(nchans, f_high, chan_bw, tsamp * factor, dms)
            out_len = xb.shape[1] - omx
            got = got_t.cpu().numpy()
            assert got.shape == (count, out_len)
            if dtype == np.uint8:
                assert np.array_equal(got.view(np.uint32), oracle.dedisperse(xb, otab, out_len))
            else:
                # binned values may differ from the double oracle's rounding by 1 ulp each: compare
                # against the transform of the GPU's own binned block too (bit-level chain) --
                # here the tolerance form: 1e-4 * sum |in| as for every f32 plan
                ref, ab = oracle.dedisperse(xb, otab, out_len)
                assert (np.abs(got.astype(np.float64) - ref) <= 1e-4 * ab).all()
        # the same survey from the time-major block (dd_survey_execute_tm: one transpose, then the
        # same binning and plans): identical bits
        first = [o.clone() for o in outs]
        for o in outs:
            o.fill_(0)
        outs_tm = sv.execute_tm(_torch_in(np.ascontiguousarray(x.T)))
        torch.cuda.synchronize()
        for a, b in zip(first, outs_tm):
            assert torch.equal(a, b)


def test_survey_without_binning_time_major_and_errors(B, oracle):
    """dd_survey_* with no binned range reads the time-major block through the fused pre-pass
    (Table 2 itself has no binning); argument errors of dd_survey_create."""
    import torch
    nchans, nsamps = 72, 20000
    ranges = [(0.0, 0.5, 30, 1), (15.0, 1.0, 12, 1)]
    rng = np.random.default_rng(5)
    x = _rand_input(rng, np.uint8, nchans, nsamps)
    with B.Survey(nchans, nsamps, 1500.0, -2.0, 64e-6, ranges, B.DD_U8) as sv:
        assert sv.nranges == 2
        outs = sv.execute_tm(_torch_in(np.ascontiguousarray(x.T)))
        torch.cuda.synchronize()
        for (start, step, count, _), got in zip(ranges, outs):
            dms = start + np.arange(count) * step
            otab, omx = oracle.shift_table(nchans, 1500.0, -2.0, 64e-6, dms)
            assert np.array_equal(got.cpu().numpy().view(np.uint32), oracle.dedisperse(x, otab, nsamps - omx))
    for bad, status in (([(0.0, 1.0, 10, 3)], B.DD_ERR_INVALID_ARG), ([(0.0, 1.0, 0, 1)], B.DD_ERR_INVALID_ARG),
                        ([], B.DD_ERR_INVALID_ARG)):
        with pytest.raises(B.DDError) as e:
            B.Survey(nchans, nsamps, 1500.0, -2.0, 64e-6, bad, B.DD_U8)
        assert e.value.status == status
    with pytest.raises(B.DDError) as e:   # no wider integer type to bin 16-bit samples into
        B.Survey(nchans, nsamps, 1500.0, -2.0, 64e-6, [(0.0, 1.0, 10, 2)], B.DD_U16)
    assert e.value.status == B.DD_ERR_UNSUPPORTED_PLAN


def test_plans_of_one_shape_with_different_ring_sizes_coexist(B, oracle):
    """The opt-in shared-memory attribute is per kernel function: creating a second plan with a
    smaller ring must not break launches of an earlier plan with a larger one."""
    rng = np.random.default_rng(23)
    big = (96, 30000, np.arange(24) * 6.0)     # long windows -> large stages
    small = (96, 30000, np.arange(24) * 0.1)   # short windows -> small stages
    xs, plans = [], []
    try:
        for nchans, nsamps, dms in (big, small):
            xs.append(_rand_input(rng, np.uint8, nchans, nsamps))
            plans.append(B.Plan(nchans, nsamps, 1500.0, -3.0, 64e-6, dms, B.DD_U8))
        import torch
        for x, plan in zip(xs, plans):          # the big plan runs after the small one was created
            d_out = torch.empty((plan.ndm, plan.out_len), dtype=torch.int32, device="cuda")
            plan.execute(_torch_in(x), d_out)
            torch.cuda.synchronize()
            assert np.array_equal(d_out.cpu().numpy().view(np.uint32),
                                  oracle.dedisperse(x, plan.shift_table(), plan.out_len))
    finally:
        for p in plans:
            p.destroy()


def test_bin_time_errors(B):
    import torch
    x = torch.zeros((4, 64), dtype=torch.uint8, device="cuda")
    o = torch.zeros((4, 64), dtype=torch.int16, device="cuda")
    for factor in (0, 1, 3, 32):
        with pytest.raises(B.DDError) as e:
            B.bin_time(x, o, 4, 64, factor, B.DD_U8)
        assert e.value.status == B.DD_ERR_INVALID_ARG
    with pytest.raises(B.DDError) as e:
        B.bin_time(x, o, 4, 32, 2, B.DD_U16)
    assert e.value.status == B.DD_ERR_UNSUPPORTED_PLAN
    with pytest.raises(B.DDError) as e:
        B.bin_time(x, o, 4, 63, 2, B.DD_U4)
    assert e.value.status == B.DD_ERR_INVALID_ARG


def test_many_channels_up_to_the_uint32_edge(B):
    """Maximum sizes of the exact integer paths: u16 with the largest accepted channel count
    (65537 * 65535 = 2^32 - 65536 - 1 fits uint32 by 65536) on all-max input, and u8 with
    70000 channels of 255 (274 flushes of the packed lanes)."""
    import torch
    dms = np.arange(3) * 0.5
    nchans, nsamps = 65537, 1024
    with B.Plan(nchans, nsamps, 1500.0, -300.0 / nchans, 64e-6, dms, B.DD_U16) as plan:
        d_in = torch.full((nchans, nsamps), -1, dtype=torch.int16, device="cuda")  # 0xFFFF
        d_out = torch.zeros((plan.ndm, plan.out_len), dtype=torch.int32, device="cuda")
        plan.execute(d_in.view(torch.uint16), d_out)
        torch.cuda.synchronize()
        got = d_out.cpu().numpy().view(np.uint32)
        assert (got == np.uint32(65537 * 65535)).all()
    with pytest.raises(B.DDError) as e:
        B.Plan(65538, nsamps, 1500.0, -300.0 / 65538, 64e-6, dms, B.DD_U16)
    assert e.value.status == B.DD_ERR_OVERFLOW
    nchans = 70000
    with B.Plan(nchans, nsamps, 1500.0, -300.0 / nchans, 64e-6, dms, B.DD_U8) as plan:
        d_in = torch.full((nchans, nsamps), 255, dtype=torch.uint8, device="cuda")
        d_out = torch.zeros((plan.ndm, plan.out_len), dtype=torch.int32, device="cuda")
        plan.execute(d_in, d_out)
        torch.cuda.synchronize()
        assert (d_out == 255 * nchans).all().item()


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_fuzz_random_plans_all_rungs_bit_exact(B, oracle, seed):
    """80 random plans per seed over channel counts 1..1500, bands at 150-3000 MHz, sampling
    times 16 us..1 ms, DM steps 0.01..50 (so every rung of the DM-block ladder is exercised),
    all four input types, unsorted DM lists, device path and chunked host path.  float32 inputs
    are integer-valued, so every comparison is bit-exact.  (The same generator ran 2400 plans
    without a mismatch during development.)"""
    import torch
    rng = np.random.default_rng(seed)
    seen_rungs = set()
    for it in range(80):
        dt = [np.uint8, np.uint16, np.float32, "u4"][rng.integers(0, 4)]
        nchans = int(rng.choice([1, 2, 3, 7, 16, 33, 64, 100, 255, 256, 257, 300, 513, 1024, 1500]))
        f_high = float(rng.choice([150.0, 400.0, 800.0, 1500.0, 3000.0]))
        band = f_high * float(rng.uniform(0.05, 0.4))
        tsamp = float(rng.choice([16e-6, 64e-6, 256e-6, 1e-3]))
        ndm = int(rng.choice([1, 2, 5, 12, 13, 24, 31, 32, 33, 50, 100]))
        step = float(rng.choice([0.01, 0.1, 0.5, 1.0, 3.0, 10.0, 50.0]))
        dms = float(rng.choice([0.0, 0.0, 10.0, 100.0])) + np.arange(ndm) * step
        if rng.random() < 0.2:
            dms = rng.permutation(dms)
        tab, mx = oracle.shift_table(nchans, f_high, -band / nchans, tsamp, dms)
        nsamps = mx + int(rng.choice([1, 2, 17, 100, 1000, 5000, 20000]))
        if dt == "u4":
            nsamps += nsamps & 1
        if nchans * nsamps > 1e8 or nsamps > 1e6:
            continue
        code = {np.uint8: B.DD_U8, np.uint16: B.DD_U16, np.float32: B.DD_F32, "u4": B.DD_U4}[dt]
        with B.Plan(nchans, nsamps, f_high, -band / nchans, tsamp, dms, code) as plan:
            seen_rungs.add((code, plan.info("D_DM")))
            out_len = plan.out_len
            assert np.array_equal(plan.shift_table(), tab) and out_len == nsamps - mx
            if dt == "u4":
                x = rng.integers(0, 256, (nchans, nsamps // 2), dtype=np.uint8)
                ref = oracle.dedisperse_u4(x, tab, out_len)
            elif dt == np.float32:
                x = rng.integers(-1000, 1000, (nchans, nsamps)).astype(np.float32)
                ref = oracle.dedisperse(x, tab, out_len)[0]
            else:
                x = _rand_input(rng, dt, nchans, nsamps)
                ref = oracle.dedisperse(x, tab, out_len)
            d_in = _torch_in(x)
            odt = torch.float32 if dt == np.float32 else torch.int32
            d_out = torch.full((ndm, out_len), -7, dtype=odt, device="cuda")
            plan.execute(d_in, d_out)
            torch.cuda.synchronize()
            h_out = torch.full((ndm, out_len), -7, dtype=odt)
            plan.set_host_chunks(int(rng.integers(0, 6)))
            plan.execute_host(d_in.cpu(), h_out)
            for got in (d_out.cpu().numpy(), h_out.numpy()):
                same = (np.array_equal(got.astype(np.float64), ref) if dt == np.float32
                        else np.array_equal(got.view(np.uint32), ref))
                assert same, (str(dt), nchans, nsamps, ndm, step, f_high, band, tsamp, plan.info("D_DM"))
    assert len({d for _, d in seen_rungs}) >= 3   # several rungs of the ladder were hit


def test_plan_errors_on_gpu(B):
    with pytest.raises(B.DDError) as e:
        B.Plan(4, 32, 1500.0, -25.0, 1e-3, [0.0, 300.0], B.DD_U8)
    assert e.value.status == B.DD_ERR_SHIFT_TOO_LARGE
    plan = B.Plan(4, 32, 1500.0, -25.0, 1e-3, [0.0], B.DD_U8)
    with pytest.raises(B.DDError) as e:
        plan.execute(0, 0)
    assert e.value.status == B.DD_ERR_INVALID_ARG
    plan.destroy()
    plan.destroy()  # idempotent


def test_runs_beside_a_tensor_core_gemm(B, oracle):
    """The u8 and u4 kernels park accumulators in tensor memory (tcgen05.alloc sized per shape).  A
    bf16 GEMM (a tcgen05 / TMEM user) running on another stream at the same time must neither
    block nor disturb them: results stay bit-exact against the oracle."""
    import torch
    rng = np.random.default_rng(77)
    nchans, nsamps = 600, 60000
    dms = np.arange(48) * 1.0
    x8 = rng.integers(0, 256, (nchans, nsamps), dtype=np.uint8)
    xp = W.pack_u4(rng.integers(0, 16, (nchans, nsamps)).astype(np.uint8))
    a = torch.randn((4096, 4096), dtype=torch.bfloat16, device="cuda")
    b = torch.randn((4096, 4096), dtype=torch.bfloat16, device="cuda")
    side = torch.cuda.Stream()
    for code, x in ((B.DD_U8, x8), (B.DD_U4, xp)):
        with B.Plan(nchans, nsamps, 1500.0, -300.0 / nchans, 64e-6, dms, code) as plan:
            d_in = torch.from_numpy(x).cuda()
            d_out = torch.full((plan.ndm, plan.out_len), -1, dtype=torch.int32, device="cuda")
            torch.cuda.synchronize()
            with torch.cuda.stream(side):
                for _ in range(40):
                    c = a @ b
            for _ in range(6):
                plan.execute(d_in, d_out)
            torch.cuda.synchronize()
            run = oracle.dedisperse_u4 if code == B.DD_U4 else oracle.dedisperse
            assert np.array_equal(d_out.cpu().numpy().view(np.uint32), run(x, plan.shift_table(), plan.out_len))
            assert torch.isfinite(c.float()).all()


def _pack_channels(x8_tm):
    """[nsamps][nchans] values 0..15 -> time-major packed rows of nchans/2 bytes, the even channel of a
    byte in the low nibble (reading R16); layout only."""
    return np.ascontiguousarray((x8_tm[:, 0::2] | (x8_tm[:, 1::2] << 4)).astype(np.uint8))


@pytest.mark.parametrize("shape", [(256, 4096), (512, 1000), (130, 5002), (38, 998), (2, 2), (300, 70002)])
def test_standalone_transpose_packed_u4(B, shape):
    """dd_transpose for DD_U4: time-major packed along channels -> channel-major packed along time,
    against numpy's transpose of the unpacked values (whole tiles, ragged tiles, output rows that do
    not start on a word)."""
    import torch
    nchans, nsamps = shape
    rng = np.random.default_rng([nchans, nsamps, 4])
    x8 = rng.integers(0, 16, (nchans, nsamps)).astype(np.uint8)          # [c][t]
    x_tm = _pack_channels(np.ascontiguousarray(x8.T))                    # [t][c/2]
    d_out = torch.full((nchans, nsamps // 2), 0xAB, dtype=torch.uint8, device="cuda")
    B.transpose(torch.from_numpy(x_tm).cuda(), d_out, nchans, nsamps, B.DD_U4)
    torch.cuda.synchronize()
    assert np.array_equal(d_out.cpu().numpy(), W.pack_u4(x8))
    for bad in ((nchans + 1, nsamps), (nchans, nsamps + 1)):
        with pytest.raises(B.DDError) as e:
            B.transpose(torch.from_numpy(x_tm).cuda(), d_out, bad[0], bad[1], B.DD_U4)
        assert e.value.status == B.DD_ERR_INVALID_ARG


def test_survey_packed_u4_time_major_with_binning(B, oracle):
    """A 4-bit survey from a time-major block with binned ranges: packed transpose, dd_bin_time (4-bit
    -> 8-bit sums), 4-bit and 8-bit plans; against the oracle chain."""
    import torch
    nchans, nsamps = 96, 24000
    ranges = [(0.0, 1.0, 24, 1), (24.0, 2.0, 12, 2), (48.0, 4.0, 8, 4)]
    rng = np.random.default_rng(9)
    x8 = rng.integers(0, 16, (nchans, nsamps)).astype(np.uint8)
    xp = W.pack_u4(x8)
    x_tm = _pack_channels(np.ascontiguousarray(x8.T))
    with B.Survey(nchans, nsamps, 1500.0, -2.0, 64e-6, ranges, B.DD_U4) as sv:
        outs = sv.execute_tm(torch.from_numpy(x_tm).cuda())
        torch.cuda.synchronize()
        for (start, step, count, factor), got in zip(ranges, outs):
            dms = start + np.arange(count) * step
            otab, omx = oracle.shift_table(nchans, 1500.0, -2.0, 64e-6 * factor, dms)
            if factor == 1:
                ref = oracle.dedisperse_u4(xp, otab, nsamps - omx)
            else:
                xb = oracle.bin_time(xp, factor, packed_u4=True)          # uint8 sums
                ref = oracle.dedisperse(xb, otab, xb.shape[1] - omx)
            assert np.array_equal(got.cpu().numpy().view(np.uint32), ref)


def test_host_timeline_reports_every_chunk(B, oracle):
    """dd_plan_host_timeline: one entry per chunk of the latest dd_execute_host call, times in order."""
    rng = np.random.default_rng(3)
    nchans, nsamps = 64, 40000
    x = _rand_input(rng, np.uint8, nchans, nsamps)
    with B.Plan(nchans, nsamps, 1500.0, -2.0, 64e-6, np.arange(16) * 2.0, B.DD_U8) as plan:
        assert len(plan.host_timeline()[0]) == 0          # no host call yet
        plan.set_host_chunks(4)
        h_out = np.zeros((plan.ndm, plan.out_len), dtype=np.uint32)
        plan.execute_host(x, h_out)
        assert np.array_equal(h_out, oracle.dedisperse(x, plan.shift_table(), plan.out_len))
        ob, h2d, pre, main, d2h = plan.host_timeline()
        assert len(ob) == 4 and ob[0] == 0 and (np.diff(ob) > 0).all()
        assert (h2d <= pre).all() and (pre <= main).all() and (main <= d2h).all()
        assert (np.diff(main) >= 0).all() and d2h[-1] > 0


@pytest.mark.parametrize("time_major", [False, True])
def test_execute_host_async_two_blocks_in_flight(B, oracle, time_major):
    """dd_execute_host_async: two plans on two streams with different blocks in flight at once, and
    the same plan called twice in a row (serialised by its stream dependency); results are complete
    when the streams have been synchronised and equal the oracle's."""
    import torch
    rng = np.random.default_rng(12)
    nchans, nsamps = 96, 50000
    dms = np.arange(30) * 1.5
    xs = [_rand_input(rng, np.uint8, nchans, nsamps) for _ in range(3)]
    hin = [torch.from_numpy(np.ascontiguousarray(x.T if time_major else x)).pin_memory() for x in xs]
    plans = [B.Plan(nchans, nsamps, 1500.0, -2.0, 64e-6, dms, B.DD_U8) for _ in range(2)]
    try:
        for p in plans:
            p.set_host_chunks(3)
        houts = [torch.zeros((plans[0].ndm, plans[0].out_len), dtype=torch.int32).pin_memory() for _ in range(3)]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        plans[0].execute_host_async(hin[0], houts[0], streams[0], time_major)
        plans[1].execute_host_async(hin[1], houts[1], streams[1], time_major)
        plans[0].execute_host_async(hin[2], houts[2], streams[0], time_major)   # same plan again: after block 0
        for s in streams:
            s.synchronize()
        assert [p.info("HOST_CHUNKS") for p in plans] == [3, 3] and plans[0].info("HOST_TAPER") == 0
        tab = plans[0].shift_table()
        for x, h in zip(xs, houts):
            assert np.array_equal(h.numpy().view(np.uint32), oracle.dedisperse(x, tab, plans[0].out_len))
    finally:
        for p in plans:
            p.destroy()


def test_one_plan_host_calls_from_different_streams_are_serialised(B, oracle):
    """One plan, host calls queued from DIFFERENT streams with nothing ordering them, then a dd_execute
    on a third: the plan owns one set of device buffers, so each call must wait for the previous host
    call's last copy back (round-2 advice: before, the second call's copies in could overwrite the
    first call's input while its kernels were still reading it).  A long first block makes the overlap
    window wide; every plane must equal the oracle's."""
    import torch
    rng = np.random.default_rng(77)
    nchans, nsamps = 256, 400000
    dms = np.arange(96) * 1.0
    xs = [_rand_input(rng, np.uint8, nchans, nsamps) for _ in range(3)]
    hin = [torch.from_numpy(x).pin_memory() for x in xs]
    with B.Plan(nchans, nsamps, 1500.0, -1.0, 64e-6, dms, B.DD_U8) as plan:
        houts = [torch.zeros((plan.ndm, plan.out_len), dtype=torch.int32).pin_memory() for _ in range(2)]
        d_in = torch.from_numpy(xs[2]).cuda()
        d_out = torch.zeros((plan.ndm, plan.out_len), dtype=torch.int32, device="cuda")
        s = [torch.cuda.Stream() for _ in range(3)]
        torch.cuda.synchronize()
        for rep in range(2):
            plan.execute_host_async(hin[0], houts[0], s[0])
            plan.execute_host_async(hin[1], houts[1], s[1])   # another stream, nothing orders it after s[0]
            plan.execute(d_in, d_out, s[2])                   # device path while both are pending
            torch.cuda.synchronize()
            tab = plan.shift_table()
            for x, got in ((xs[0], houts[0].numpy()), (xs[1], houts[1].numpy()), (xs[2], d_out.cpu().numpy())):
                assert np.array_equal(got.view(np.uint32), oracle.dedisperse(x, tab, plan.out_len)), rep
            for h in houts:
                h.zero_()
            d_out.zero_()


def test_plan_refuses_a_call_from_another_current_device(B, oracle):
    """An in-process multi-GPU caller (the 'replicas driven by the caller' of SURVEY.md 8(e)): a plan runs
    on the device it was made on and refuses, with DD_ERR_INVALID_ARG and no launch, a call made while
    another device is current; two plans on two devices from one process both equal the oracle."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs in one process")
    rng = np.random.default_rng(3)
    x = _rand_input(rng, np.uint8, 64, 6000)
    dms = np.arange(16) * 2.0
    outs, plans = [], []
    try:
        for dev in (0, 1):
            torch.cuda.set_device(dev)
            plan = B.Plan(64, 6000, 1500.0, -2.0, 64e-6, dms, B.DD_U8)
            plans.append(plan)
            d_in = torch.from_numpy(x).to("cuda:%d" % dev)
            out = torch.zeros((plan.ndm, plan.out_len), dtype=torch.int32, device="cuda:%d" % dev)
            plan.execute(d_in, out)
            torch.cuda.synchronize(dev)
            outs.append(out.cpu().numpy().view(np.uint32))
        ref = oracle.dedisperse(x, plans[0].shift_table(), plans[0].out_len)
        assert np.array_equal(outs[0], ref) and np.array_equal(outs[1], ref)
        with pytest.raises(B.DDError) as e:      # device 1 is current, plan 0 lives on device 0
            plans[0].execute(d_in, out)
        assert e.value.status == B.DD_ERR_INVALID_ARG
    finally:
        torch.cuda.set_device(0)
        for p in plans:
            p.destroy()
