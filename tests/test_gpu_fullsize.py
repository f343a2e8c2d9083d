"""-m gpu: the large configs at FULL size, in the launch configuration bench.py times.

Three layers (sampling is allowed only if the full-output comparison has been
run per config and kernel variant):
  * test_full_size_sampled_parity   -- the oracle computes ~3600 sampled outputs one by one
    (oracle_dedisperse_points) plus three complete DM rows; sample points include every kind of
    tile edge the kernel has (lane boundaries k*L, word-tile boundaries, DM-block boundaries,
    first/last sample and DM).  Seconds per config.
  * test_full_output_parity (also marked slow) -- EVERY output element of dd_execute against the
    oracle's whole plane, default kernel variant, for c2, headline, lowfreq, c3, headline_u4,
    paper52 (rows that are not 16-byte aligned) and largeshift (a lower rung of the DM-block ladder).  About a minute of oracle time per config.
  * test_other_entry_points_equal_device_output_full_size -- dd_execute_host and
    dd_execute_host_tm on their DEFAULT chunk schedule (the one bench.py's e2e leg times) and
    dd_execute_tm must reproduce dd_execute's plane bit for bit (same kernels, same per-output
    summation order, so float32 too); dd_execute's plane is tied to the oracle by sampled points
    in the same test.
  * test_binned_range_full_size -- dd_bin_time + dd_execute of a binned DM range at headline size.
Integer configs: bit-exact.  c3 (f32): |gpu - oracle| <= 1e-4 * sum_c|in|."""
import dataclasses

import numpy as np
import pytest

from paper_2311_05341_b200 import workloads as W

pytestmark = pytest.mark.gpu

NPOINTS = 3000
FULL_ROWS = 3


def _to_numpy(x):
    import torch
    if x.dtype == torch.uint16:
        return x.view(torch.int16).cpu().numpy().view(np.uint16)
    return x.cpu().numpy()


def _sample_points(rng, ndm, out_len, L, D_J, D_DM, lanes, npoints=NPOINTS):
    pd = list(rng.integers(0, ndm, npoints))
    pt = list(rng.integers(0, out_len, npoints))
    d_edges = {0, ndm - 1}
    for b in range(D_DM, ndm, max(D_DM, (ndm // 8) // D_DM * D_DM or D_DM)):
        d_edges.update((b - 1, b))
    t_edges = {0, out_len - 1}
    for k in range(1, lanes):
        t_edges.update((k * L - 1, k * L, k * L + 1))
    for j in (D_J, 2 * D_J, (L // D_J) * D_J):
        for k in range(lanes):
            t_edges.update((k * L + j - 1, k * L + j))
    t_edges = sorted(t for t in t_edges if 0 <= t < out_len)
    for d in sorted(d for d in d_edges if 0 <= d < ndm):
        for t in t_edges:
            pd.append(d)
            pt.append(t)
    return np.array(pd, dtype=np.int32), np.array(pt, dtype=np.int64)


def _gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device; the product has no CPU fallback")
    from paper_2311_05341_b200 import binding as B, build
    build.build()
    return B


def _plan_and_input(B, oracle, cfg):
    plan = B.Plan(cfg.nchans, cfg.nsamps, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list, cfg.in_dtype)
    otab, omx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    assert np.array_equal(plan.shift_table(), otab) and omx == plan.max_shift
    x = W.make_input_torch(cfg, "cuda", otab, plan.out_len)
    return plan, otab, x


def _points_check(oracle, cfg, xh, otab, out, pd, pt):
    """`out` (device tensor) at the sampled (d, t) against the oracle's one-by-one evaluation."""
    import torch
    got = out[torch.from_numpy(pd.astype(np.int64)).cuda(), torch.from_numpy(pt).cuda()].cpu().numpy()
    if cfg.in_dtype == W.F32:
        ref, ab = oracle.dedisperse_points(xh, otab, pd, pt)
        err = np.abs(got.astype(np.float64) - ref)
        assert (err <= 1e-4 * ab).all(), "points: max err %g" % err.max()
    elif cfg.in_dtype == W.U4:
        # the oracle's 4-bit transform on the packed rows, evaluated for the sampled DM rows only
        rows = np.unique(pd)
        ref_rows = oracle.dedisperse_u4(xh, otab[rows], out.shape[1])
        ref = ref_rows[np.searchsorted(rows, pd), pt]
        assert np.array_equal(got.view(np.uint32), ref)
    else:
        ref = oracle.dedisperse_points(xh, otab, pd, pt)
        bad = np.flatnonzero(got.view(np.uint32) != ref)
        assert bad.size == 0, "points differ at (d,t)=%s" % [(int(pd[i]), int(pt[i])) for i in bad[:5]]


@pytest.mark.parametrize("name", ["c2", "headline", "lowfreq", "c3"])
def test_full_size_sampled_parity(oracle, golden, name):
    import torch
    B = _gpu()
    cfg = W.CONFIGS[name]
    g = golden("shift_pins.json")["configs"][name]
    plan, otab, x = _plan_and_input(B, oracle, cfg)
    try:
        assert plan.max_shift == g["max_shift"] and plan.out_len == g["out_len"]
        odt = torch.float32 if cfg.in_dtype == W.F32 else torch.int32
        out = torch.full((plan.ndm, plan.out_len), -3, dtype=odt, device="cuda")
        plan.execute(x, out)
        torch.cuda.synchronize()
        xh = _to_numpy(x)
        del x
        rng = np.random.default_rng([cfg.seed, 99])
        pd, pt = _sample_points(rng, plan.ndm, plan.out_len, plan.info("L"), plan.info("D_J"),
                                plan.info("D_DM"), plan.info("LANES"))
        _points_check(oracle, cfg, xh, otab, out, pd, pt)
        rows = sorted({0, plan.ndm - 1, int(rng.integers(1, plan.ndm - 1))})[:FULL_ROWS]
        got_rows = out[torch.tensor(rows, device="cuda")].cpu().numpy()
        if cfg.in_dtype == W.F32:
            rref, rab = oracle.dedisperse(xh, otab[rows], plan.out_len)
            rerr = np.abs(got_rows.astype(np.float64) - rref)
            assert (rerr <= 1e-4 * rab).all(), "rows: max err %g" % rerr.max()
            # the injected pulses are recovered at their DM
            for d, t0 in W.pulse_plan(cfg, plan.out_len):
                row = out[d].cpu().numpy()
                box = np.convolve(row, np.ones(cfg.pulse_width), mode="valid")
                assert abs(int(np.argmax(box)) - t0) <= 1
        else:
            rref = oracle.dedisperse(xh, otab[rows], plan.out_len)
            assert np.array_equal(got_rows.view(np.uint32), rref)
        # no element left unwritten (the buffer was pre-filled with a sentinel; sums are >> 0)
        if cfg.in_dtype != W.F32:
            assert int((out[:: max(1, plan.ndm // 16)] == -3).sum().item()) == 0
    finally:
        plan.destroy()


FULL_OUTPUT_CONFIGS = ["c2", "headline", "lowfreq", "c3", "headline_u4", "paper52", "largeshift"]


@pytest.mark.slow
@pytest.mark.parametrize("name", FULL_OUTPUT_CONFIGS)
def test_full_output_parity(oracle, name):
    """the whole output plane of dd_execute, every DM row and every sample, against
    the oracle's plane, with the kernel variant dd_plan_create picks by default."""
    import torch
    B = _gpu()
    cfg = W.ALL_CONFIGS[name]
    plan, otab, x = _plan_and_input(B, oracle, cfg)
    try:
        odt = torch.float32 if cfg.in_dtype == W.F32 else torch.int32
        out = torch.full((plan.ndm, plan.out_len), -3, dtype=odt, device="cuda")
        plan.execute(x, out)
        torch.cuda.synchronize()
        xh = _to_numpy(x)
        del x
        got = out.cpu().numpy()
        del out
        if cfg.in_dtype == W.F32:
            # row blocks keep the oracle's two float64 planes small
            worst = 0.0
            for d0 in range(0, plan.ndm, 256):
                ref, ab = oracle.dedisperse(xh, otab[d0:d0 + 256], plan.out_len)
                err = np.abs(got[d0:d0 + 256].astype(np.float64) - ref)
                assert (err <= 1e-4 * ab).all(), "rows %d..: max err %g" % (d0, err.max())
                worst = max(worst, float((err / np.maximum(ab, 1e-300)).max()))
            print("%s: full plane within tolerance, worst err / sum|in| = %.3g" % (name, worst))
        else:
            run = oracle.dedisperse_u4 if cfg.in_dtype == W.U4 else oracle.dedisperse
            ref = run(xh, otab, plan.out_len)
            same = np.array_equal(got.view(np.uint32), ref)
            if not same:
                bad = np.argwhere(got.view(np.uint32) != ref)
                pytest.fail("%s: %d of %d outputs differ, first (d,t) = %s"
                            % (name, len(bad), ref.size, bad[:5].tolist()))
    finally:
        plan.destroy()


@pytest.mark.parametrize("name", ["headline", "lowfreq", "c3", "headline_u4"])
def test_other_entry_points_equal_device_output_full_size(oracle, name):
    """dd_execute_host / dd_execute_host_tm with NO chunk override (the tapered 8-chunk pipeline with its
    two workspaces and two main streams), dd_execute_host_async on its own default schedule, channel- and
    time-major (what bench.py's e2e leg times; the schedule taken is asserted through dd_plan_info) and
    dd_execute_tm reproduce dd_execute's plane bit for bit; that plane is tied to
    the oracle by sampled points here and as a whole in test_full_output_parity."""
    import torch
    B = _gpu()
    cfg = W.ALL_CONFIGS[name]
    plan, otab, x = _plan_and_input(B, oracle, cfg)
    try:
        odt = torch.float32 if cfg.in_dtype == W.F32 else torch.int32
        out = torch.full((plan.ndm, plan.out_len), -3, dtype=odt, device="cuda")
        plan.execute(x, out)
        torch.cuda.synchronize()
        xh = _to_numpy(x)
        rng = np.random.default_rng([cfg.seed, 7])
        pd, pt = _sample_points(rng, plan.ndm, plan.out_len, plan.info("L"), plan.info("D_J"),
                                plan.info("D_DM"), plan.info("LANES"), npoints=400)
        if cfg.in_dtype == W.U4:  # the 4-bit oracle evaluates whole rows: keep the sampled rows few
            sel = np.unique(np.concatenate([[0, plan.ndm - 1], rng.integers(0, plan.ndm, 10)])).astype(np.int32)
            pd = sel[np.arange(pd.size) % sel.size]
        _points_check(oracle, cfg, xh, otab, out, pd, pt)
        del xh
        # ---- host path, channel-major, default schedule
        h_in = torch.empty(x.shape, dtype=x.dtype).pin_memory()
        h_in.copy_(x)
        h_out = torch.full((plan.ndm, plan.out_len), -5, dtype=odt).pin_memory()
        plan.execute_host(h_in, h_out)
        assert torch.equal(h_out, out.cpu()), "dd_execute_host differs from dd_execute"
        assert plan.info("HOST_TAPER") == 1 and plan.info("HOST_CHUNKS") == 8
        # ---- the asynchronous form on ITS default schedule (what bench.py's e2e times): 4 equal chunks,
        # the taper only for a block whose copies outlast its kernels (lowfreq)
        side = torch.cuda.Stream()
        h_out.fill_(-5)
        plan.execute_host_async(h_in, h_out, side)
        side.synchronize()
        assert torch.equal(h_out, out.cpu()), "dd_execute_host_async differs from dd_execute"
        assert plan.info("HOST_TAPER") == (1 if name == "lowfreq" else 0)
        assert plan.info("HOST_CHUNKS") == (8 if name == "lowfreq" else 4)
        del h_in
        # ---- time-major: device path (fused transpose pre-pass) and host path
        if cfg.in_dtype == W.U4:
            # packed along channels instead of along time (reading R16): repack on the device
            lo, hi = x & 15, x >> 4
            x8 = torch.stack((lo, hi), dim=2).reshape(cfg.nchans, cfg.nsamps)   # [c][t] values 0..15
            del lo, hi
            x8t = x8.t().contiguous()                                         # [t][c]
            del x8
            x_tm = (x8t[:, 0::2] | (x8t[:, 1::2] << 4)).contiguous()
            del x8t
        else:
            x_tm = x.t().contiguous()
        del x
        out_tm = torch.full((plan.ndm, plan.out_len), -9, dtype=odt, device="cuda")
        plan.execute_tm(x_tm, out_tm)
        torch.cuda.synchronize()
        assert torch.equal(out_tm, out), "dd_execute_tm differs from dd_execute"
        del out_tm
        h_tm = torch.empty(x_tm.shape, dtype=x_tm.dtype).pin_memory()
        h_tm.copy_(x_tm)
        del x_tm
        h_out.fill_(-5)
        plan.execute_host_tm(h_tm, h_out)
        assert torch.equal(h_out, out.cpu()), "dd_execute_host_tm differs from dd_execute"
        h_out.fill_(-5)
        plan.execute_host_async(h_tm, h_out, side, time_major=True)
        side.synchronize()
        assert torch.equal(h_out, out.cpu()), "dd_execute_host_async (time-major) differs from dd_execute"
        assert plan.info("HOST_TAPER") == (1 if name == "lowfreq" else 0)
    finally:
        plan.destroy()


def test_binned_range_full_size(oracle):
    """One binned DM range at headline size (a Table 2 style range run on time-binned data,
    PAPER.md:295, 303-309, 370): dd_bin_time by 4 of the 8192 x 2^18 uint8 block, then dd_execute of
    DM 500..755 with tsamp*4 on the uint16 result.  The binned block is compared with the oracle's
    as a whole; the dedispersed plane at sampled points plus two complete rows."""
    import torch
    B = _gpu()
    base = W.CONFIGS["headline"]
    factor = 4
    x = W.make_input_torch(base, "cuda", None, None)
    nb = base.nsamps // factor
    d_bin = torch.empty((base.nchans, nb), dtype=torch.int16, device="cuda")
    B.bin_time(x, d_bin, base.nchans, base.nsamps, factor, B.DD_U8)
    torch.cuda.synchronize()
    xh = x.cpu().numpy()
    del x
    xb = oracle.bin_time(xh, factor)
    del xh
    assert np.array_equal(d_bin.cpu().numpy().view(np.uint16), xb), "dd_bin_time differs from the oracle"
    dms = 500.0 + np.arange(512) * 0.5
    cfg = dataclasses.replace(base, in_dtype=W.U16, nsamps=nb, tsamp=base.tsamp * factor)
    with B.Plan(base.nchans, nb, base.f_high, base.chan_bw, cfg.tsamp, dms, B.DD_U16) as plan:
        otab, omx = oracle.shift_table(base.nchans, base.f_high, base.chan_bw, cfg.tsamp, dms)
        assert np.array_equal(plan.shift_table(), otab) and plan.out_len == nb - omx
        out = torch.full((plan.ndm, plan.out_len), -3, dtype=torch.int32, device="cuda")
        plan.execute(d_bin.view(torch.uint16), out)
        torch.cuda.synchronize()
        rng = np.random.default_rng(41)
        pd, pt = _sample_points(rng, plan.ndm, plan.out_len, plan.info("L"), plan.info("D_J"),
                                plan.info("D_DM"), plan.info("LANES"), npoints=1500)
        _points_check(oracle, cfg, xb, otab, out, pd, pt)
        rows = [0, plan.ndm - 1]
        got_rows = out[torch.tensor(rows, device="cuda")].cpu().numpy().view(np.uint32)
        assert np.array_equal(got_rows, oracle.dedisperse(xb, otab[rows], plan.out_len))


def test_survey_full_size(oracle):
    """dd_survey_execute_tm on the survey52 workload (time-major 8192 x 156250 uint8 block, four DM
    ranges binned by 1, 2, 2, 4; bench.py --config survey52): the whole planes of the two ranges binned
    by 2 and two complete DM rows of the other two against the oracle chain (numpy transpose -> oracle_bin_time -> oracle transform)."""
    import torch
    B = _gpu()
    sc = W.SURVEYS["survey52"]
    gen = W.Config(sc.name, sc.nchans, sc.nsamps, sc.in_dtype, sc.f_high, sc.chan_bw, sc.tsamp, 1, 0.0,
                   seed=sc.seed, mean=sc.mean, sd=sc.sd)
    x = W.noise_torch(gen, "cuda")
    xh = x.cpu().numpy()
    x_tm = x.t().contiguous()
    del x
    with B.Survey(sc.nchans, sc.nsamps, sc.f_high, sc.chan_bw, sc.tsamp, sc.ranges, sc.in_dtype) as sv:
        outs = sv.execute_tm(x_tm)
        torch.cuda.synchronize()
        binned = {1: xh}
        for (start, step, count, factor), got, out_len in zip(sc.ranges, outs, sv.out_len):
            if factor not in binned:
                binned[factor] = oracle.bin_time(xh, factor)
            xb = binned[factor]
            dms = start + np.arange(count, dtype=np.float64) * step
            otab, omx = oracle.shift_table(sc.nchans, sc.f_high, sc.chan_bw, sc.tsamp * factor, dms)
            assert out_len == xb.shape[1] - omx
            if factor == 2:
                # the two ranges binned by 2 (750 and 800 trials on the uint16 block): EVERY row and sample,
                # about 20 s of oracle on the box's 16 cores -- the binned u16 chain as a whole plane
                ref = oracle.dedisperse(xb, otab, out_len)
                same = np.array_equal(got.cpu().numpy().view(np.uint32), ref)
                del ref
                assert same, "range (%g, %g, %d, %d): plane differs from the oracle chain" % (start, step, count, factor)
                continue
            rows = [0, count - 1]
            ref = oracle.dedisperse(xb, otab[rows], out_len)
            assert np.array_equal(got[torch.tensor(rows, device="cuda")].cpu().numpy().view(np.uint32), ref)
