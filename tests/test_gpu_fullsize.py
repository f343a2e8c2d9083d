"""-m gpu: the four large BASELINE.json configs at FULL size, in the launch configuration
bench.py times.  The oracle computes sampled outputs one by one (oracle_dedisperse_points)
plus a few complete DM rows; sample points include every kind of tile edge the kernel has
(lane boundaries k*L, word-tile boundaries, DM-block boundaries, first/last sample and DM).
Integer configs: bit-exact.  c3 (f32): |gpu - oracle| <= 1e-4 * sum_c|in|."""
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


def _sample_points(rng, ndm, out_len, L, D_J, D_DM, lanes):
    pd = list(rng.integers(0, ndm, NPOINTS))
    pt = list(rng.integers(0, out_len, NPOINTS))
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


@pytest.mark.parametrize("name", ["c2", "headline", "lowfreq", "c3"])
def test_full_size_sampled_parity(oracle, golden, name):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device; the product has no CPU fallback")
    from paper_2311_05341_b200 import binding as B, build
    build.build()
    cfg = W.CONFIGS[name]
    g = golden("shift_pins.json")["configs"][name]
    plan = B.Plan(cfg.nchans, cfg.nsamps, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list, cfg.in_dtype)
    try:
        table = plan.shift_table()
        assert plan.max_shift == g["max_shift"] and plan.out_len == g["out_len"]
        otab, omx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
        assert np.array_equal(table, otab) and omx == plan.max_shift
        x = W.make_input_torch(cfg, "cuda", otab, plan.out_len)
        odt = torch.float32 if cfg.in_dtype == W.F32 else torch.int32
        out = torch.full((plan.ndm, plan.out_len), -3, dtype=odt, device="cuda")
        plan.execute(x, out)
        torch.cuda.synchronize()
        xh = _to_numpy(x)
        del x
        rng = np.random.default_rng([cfg.seed, 99])
        pd, pt = _sample_points(rng, plan.ndm, plan.out_len, plan.info("L"), plan.info("D_J"),
                                plan.info("D_DM"), plan.info("LANES"))
        got_pts = out[torch.from_numpy(pd.astype(np.int64)).cuda(), torch.from_numpy(pt).cuda()].cpu().numpy()
        rows = sorted({0, plan.ndm - 1, int(rng.integers(1, plan.ndm - 1))})[:FULL_ROWS]
        got_rows = out[torch.tensor(rows, device="cuda")].cpu().numpy()
        if cfg.in_dtype == W.F32:
            ref, ab = oracle.dedisperse_points(xh, otab, pd, pt)
            err = np.abs(got_pts.astype(np.float64) - ref)
            assert (err <= 1e-4 * ab).all(), "points: max err %g" % err.max()
            rref, rab = oracle.dedisperse(xh, otab[rows], plan.out_len)
            rerr = np.abs(got_rows.astype(np.float64) - rref)
            assert (rerr <= 1e-4 * rab).all(), "rows: max err %g" % rerr.max()
            # the injected pulses are recovered at their DM
            for d, t0 in W.pulse_plan(cfg, plan.out_len):
                row = out[d].cpu().numpy()
                box = np.convolve(row, np.ones(cfg.pulse_width), mode="valid")
                assert abs(int(np.argmax(box)) - t0) <= 1
        else:
            ref = oracle.dedisperse_points(xh, otab, pd, pt)
            bad = np.flatnonzero(got_pts.view(np.uint32) != ref)
            assert bad.size == 0, "points differ at (d,t)=%s" % [(int(pd[i]), int(pt[i])) for i in bad[:5]]
            rref = oracle.dedisperse(xh, otab[rows], plan.out_len)
            assert np.array_equal(got_rows.view(np.uint32), rref)
        # no element left unwritten (the buffer was pre-filled with a sentinel; sums are >> 0)
        if cfg.in_dtype != W.F32:
            assert int((out[:: max(1, plan.ndm // 16)] == -3).sum().item()) == 0
    finally:
        plan.destroy()
