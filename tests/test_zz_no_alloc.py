"""dd_execute_noalloc: the entry point for callers that cannot allocate device memory -- a process whose
own pool already owns the whole card (cudaMalloc would fail), or a real-time stage that cannot take the
device-wide stall of cudaMalloc / cudaFree.  Its scratch (the device copy of the shift table) is a 4 MiB
array built into libdd.so, shared by every call and never cleared.

The GPU tests compare it with the existing plan path (dd_plan_create + dd_execute) on the same input:
bit-exact for integer input, |a - b| <= 1e-4 * sum_c |in| for float32 (the tolerance of the parity
tests), on two calls in a row -- the second with a different, smaller table, so that a call relying on
what the previous one left in the shared array would be caught.

This file is named to be collected last: pytest -x stops at the first failure, and a failure here must
not hide the parity tests.  It passes on its own in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

F32_RTOL_OF_ABS_SUM = 1e-4


@pytest.fixture(scope="module")
def B():
    from paper_2311_05341_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def _torch_in(x):
    import torch
    if x.dtype == np.uint16:
        return torch.from_numpy(x.view(np.int16)).cuda().view(torch.uint16)
    return torch.from_numpy(x).cuda()


def _plan_path(B, d_in, nchans, nsamps, f_high, chan_bw, tsamp, dms, code):
    """The existing path: a plan (which allocates) and dd_execute."""
    import torch
    with B.Plan(nchans, nsamps, f_high, chan_bw, tsamp, dms, code) as plan:
        odt = torch.float32 if code == B.DD_F32 else torch.int32
        out = torch.full((plan.ndm, plan.out_len), -7, dtype=odt, device="cuda")
        plan.execute(d_in, out)
        torch.cuda.synchronize()
        return out, plan.shift_table(), plan.out_len


def _noalloc_path(B, d_in, table, nsamps, out_len, code):
    import torch
    odt = torch.float32 if code == B.DD_F32 else torch.int32
    out = torch.full((table.shape[0], out_len), -9, dtype=odt, device="cuda")   # allocated by the caller
    B.execute_noalloc(table, nsamps, code, d_in, out)
    torch.cuda.synchronize()
    return out


def _compare(B, rng, code, nchans, nsamps, chan_bw, dms):
    import torch
    f_high, tsamp = 1500.0, 64e-6
    if code == B.DD_F32:
        x = rng.standard_normal((nchans, nsamps)).astype(np.float32)
    elif code == B.DD_U16:
        x = rng.integers(0, 65536, (nchans, nsamps)).astype(np.uint16)
    elif code == B.DD_U8:
        x = rng.integers(0, 256, (nchans, nsamps)).astype(np.uint8)
    else:   # packed 4-bit: random bytes are random nibble pairs
        x = rng.integers(0, 256, (nchans, nsamps // 2)).astype(np.uint8)
    d_in = _torch_in(x)
    want, table, out_len = _plan_path(B, d_in, nchans, nsamps, f_high, chan_bw, tsamp, dms, code)
    # the caller's own host table, from the pure-host builder (no plan involved)
    tab2, mx = B.dd_shift_table_build(nchans, f_high, chan_bw, tsamp, dms)
    assert np.array_equal(tab2, table) and nsamps - mx == out_len
    got = _noalloc_path(B, d_in, tab2, nsamps, out_len, code)
    if code == B.DD_F32:
        ab, _, _ = _plan_path(B, d_in.abs(), nchans, nsamps, f_high, chan_bw, tsamp, dms, code)
        err = (got.double() - want.double()).abs()
        assert bool((err <= F32_RTOL_OF_ABS_SUM * ab.double()).all()), "max err %g" % float(err.max())
    else:
        assert torch.equal(got, want), "%d elements differ" % int((got != want).sum())


@pytest.mark.gpu
@pytest.mark.parametrize("code_name", ["DD_U8", "DD_U16", "DD_F32", "DD_U4"])
def test_noalloc_equals_plan_path_two_calls_in_a_row(B, code_name):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device; the product has no CPU fallback")
    code = getattr(B, code_name)
    rng = np.random.default_rng(2311 + code)
    # first call: 300 channels x 40 trials, several time tiles and a ragged tail
    _compare(B, rng, code, 300, 9000, -0.9, np.arange(40) * 3.0)
    # second call straight after: fewer entries, other shifts -- stale rows of the first table sit behind them
    _compare(B, rng, code, 130, 4096 + 2 * 77, -1.7, np.arange(17) * 5.5)


@pytest.mark.gpu
def test_noalloc_tiny_config_and_size_limit_on_device(B):
    """configs[0] through the no-allocation call equals the plan path; one entry beyond the built-in array
    is refused with DD_ERR_STATIC_LIMIT and the output stays untouched."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device; the product has no CPU fallback")
    from paper_2311_05341_b200 import workloads as W
    cfg = W.CONFIGS["tiny"]
    table, mx = B.dd_shift_table_build(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    x = W.make_input_numpy(cfg, table, cfg.nsamps - mx)
    d_in = torch.from_numpy(x).cuda()
    want, _, out_len = _plan_path(B, d_in, cfg.nchans, cfg.nsamps, cfg.f_high, cfg.chan_bw, cfg.tsamp,
                                  cfg.dm_list, cfg.in_dtype)
    got = _noalloc_path(B, d_in, table, cfg.nsamps, out_len, cfg.in_dtype)
    assert torch.equal(got, want)
    big = np.zeros((B.NOALLOC_MAX_TABLE // 64 + 1, 64), dtype=np.int32)
    out = torch.full((4,), -9, dtype=torch.int32, device="cuda")
    with pytest.raises(B.DDError) as e:
        B.execute_noalloc(big, 4096, B.DD_U8, d_in, out)
    assert e.value.status == B.DD_ERR_STATIC_LIMIT and "DD_NOALLOC_MAX_TABLE" in str(e.value)
    torch.cuda.synchronize()
    assert out.tolist() == [-9] * 4


def test_noalloc_argument_checks_need_no_gpu(B):
    """Every argument check comes before the first CUDA call, so a bad call fails the same way anywhere."""
    ok = np.zeros((2, 3), dtype=np.int32)
    fake_in, fake_out = 4096, 8192   # never dereferenced: the checks below all fail first

    def status(table, nsamps, code, d_in=fake_in, d_out=fake_out):
        with pytest.raises(B.DDError) as e:
            B.execute_noalloc(table, nsamps, code, d_in, d_out, stream=0)
        return e.value.status

    assert status(ok, 0, B.DD_U8) == B.DD_ERR_INVALID_ARG
    assert status(ok, 100, 9) == B.DD_ERR_INVALID_ARG
    assert status(ok, 100, B.DD_U8, d_in=0) == B.DD_ERR_INVALID_ARG
    assert status(ok, 100, B.DD_U8, d_out=0) == B.DD_ERR_INVALID_ARG
    assert status(ok, 101, B.DD_U4) == B.DD_ERR_INVALID_ARG                      # packed pairs need even nsamps
    neg = ok.copy(); neg[1, 2] = -1
    assert status(neg, 100, B.DD_U8) == B.DD_ERR_INVALID_ARG
    far = ok.copy(); far[0, 1] = 100
    assert status(far, 100, B.DD_U8) == B.DD_ERR_SHIFT_TOO_LARGE
    assert status(np.zeros((1, B.NOALLOC_MAX_TABLE + 1), dtype=np.int32), 100, B.DD_U8) == B.DD_ERR_STATIC_LIMIT
    assert status(np.zeros((1, 65538), dtype=np.int32), 100, B.DD_U16) == B.DD_ERR_OVERFLOW
    assert "DD_NOALLOC_MAX_TABLE" in B.strerror(B.DD_ERR_STATIC_LIMIT)
