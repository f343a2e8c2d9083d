#!/usr/bin/env python
"""bench.py -- dedispersion adds/s on synthetic filterbank data (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config NAME] [--impl reference]

One "step" = one pass of the whole hot path (dd_execute: lane-interleave pre-pass + the
dedispersion kernel) over one block of synthetic input of the named config.  Default
workload: `headline` (BASELINE.json configs[3], 8192 channels x 2^18 samples uint8, 1024 DM
trials -- the config north_star's target is quoted on; it fits one GPU).  Prints ONE JSON line.

N > 1 (launched by torch.distributed.run): every rank processes its own block of the same
shape (independent time shards of a longer observation); no data-path
collective; value = units of all ranks / max-over-ranks time ("scaling": "weak").

--impl reference: the CPU oracle (oracle/dedisp_oracle.c), as it stands, timed on the host
cores on a bounded sample of the same workload (a subset of DM rows per step).

Besides the contract's keys the line carries: `e2e` (dd_execute_host_async, pinned host buffers, copies
inside the timed region), `roofline` (shared-memory pipe, for every input type; peak at the SM clock
sampled during the timed region, `frac_at_probe_clock` beside it) with `roofline_alu`, `roofline_hbm`
and, for 4-bit input, `roofline_alu_pipe`; `configs` (default headline run at N = 1 only: c2, c3,
lowfreq, headline_u4, paper52, largeshift and survey52, device-resident, each with its own clocks and
roofline; --no-configs leaves it out); `cpu_baseline` (the oracle on the host cores, about 10 s), `kernels_ms`,
`realtime_factor` (Eq. 10), `time_major` (dd_execute_tm / dd_execute_host_tm / dd_transpose) and
`time_binning` (dd_bin_time).  Extra workloads: headline_u4 (packed 4-bit), paper52 (the paper's
section 5.2 plan), survey52 (a multi-range binned plan over a time-major block through
dd_survey_execute_tm: the paper's pipeline real-time factor); --nsamps overrides the block length.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2311_05341_b200 import workloads as W  # noqa: E402

METRIC = "dedispersion adds/s (DM*sample*channel per s)"
UNIT = "adds/s"
N_SM = 148
# Plain integer ALU peak: 64 INT32 add lanes per SM per clock (alu
# pipe: 4 sub-partitions x 16 lanes, B300_MICROARCH.md "Pipe rates") x 148 SMs x max SM clock.
INT_LANES_PER_SM_CLK = 64
# Shared-memory bandwidth (paper's Eq. 8): 32 banks x 4 B per SM per clock.
SMEM_BYTES_PER_SM_CLK = 128


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), float(p.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float):
        res = self.window(t0, t1)
        self.close()
        return res

    def close(self):
        if self.proc is not None:
            self.proc.terminate()

    def window(self, t0: float, t1: float):
        """Clocks and throttle reasons of the samples taken in [t0, t1] (the sampler keeps running)."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in list(self.rows):
            if not (t0 <= ts <= t1 + 0.12):
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
                "samples": len(sm), "reasons": sorted(reasons)}


def _dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


# ------------------------------------------------------------------------- reference arm
def _oracle_sample(cfg, oracle, rows_per_step: int):
    """A bounded sample of the workload for the CPU oracle: the full-shape input, a subset of
    DM rows spread over the plan (adds/s of the triple loop does not depend on which rows)."""
    table, mx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    out_len = cfg.nsamps - mx
    rows = np.unique(np.linspace(0, cfg.ndm - 1, rows_per_step).astype(np.int64))
    return table[rows], out_len, len(rows)


def _host_input(cfg):
    # same distribution as the device generator; values do not matter for CPU timing
    rng = np.random.default_rng(cfg.seed)
    if cfg.in_dtype == W.F32:
        return rng.standard_normal((cfg.nchans, cfg.nsamps), dtype=np.float32)
    hi = {W.U8: 255, W.U16: 65535, W.U4: 15}[cfg.in_dtype]
    if cfg.in_dtype == W.U4:
        return rng.integers(0, 256, (cfg.nchans, cfg.nsamps // 2), dtype=np.uint8)
    x = np.empty((cfg.nchans, cfg.nsamps), dtype=cfg.np_dtype)
    step = max(1, (1 << 24) // cfg.nsamps)
    for c0 in range(0, cfg.nchans, step):
        blk = rng.standard_normal((min(step, cfg.nchans - c0), cfg.nsamps), dtype=np.float32)
        x[c0:c0 + step] = np.clip(np.rint(blk * cfg.sd + cfg.mean), 0, hi).astype(cfg.np_dtype)
    return x


def time_oracle(cfg, steps: int, warmup: int, rows_per_step: int | None = None, x=None):
    from oracle import oracle
    oracle.build()
    threads = oracle.omp_threads()
    if rows_per_step is None:
        # bounded sample: about 10-20 s of host work for the cpu_baseline leg (one step), about
        # 5-10 s per step for the reference arm (K steps), at the oracle's ~3 G adds/s per core
        target_adds = (6e11 if steps == 1 else 3e11) * (0.12 if cfg.in_dtype == W.F32 else 1.0)
        mx_rows = int(np.ceil(target_adds / (float(cfg.nsamps) * cfg.nchans)))
        rows_per_step = int(min(cfg.ndm, max(threads, 4, mx_rows)))
    sub, out_len, nrows = _oracle_sample(cfg, oracle, rows_per_step)
    if x is None:
        x = _host_input(cfg)
    run = oracle.dedisperse_u4 if cfg.in_dtype == W.U4 else oracle.dedisperse
    for _ in range(warmup):
        run(x, sub[:max(1, min(nrows, threads))], out_len)
    t0 = time.perf_counter()
    for _ in range(steps):
        run(x, sub, out_len)
    dt = time.perf_counter() - t0
    adds = float(nrows) * out_len * cfg.nchans * steps
    return {"value": adds / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": "%d of %d DM rows x full out_len x all %d channels per step, %d step(s), %.1f s"
                      % (nrows, cfg.ndm, cfg.nchans, steps, dt)}, dt / steps


def time_tiled(cfg, x, budget_s: float = 10.0):
    """cpu_baseline_tiled: the paper's tiled OpenMP CPU kernel (Algorithm 2, PAPER.md:91-141;
    cpu_tiled/) on a bounded sample of the workload -- a contiguous block of DM rows (its DM tiles
    share cache lines only between neighbouring trials), full out_len, all channels.  Tile sizes:
    the fastest of cpu_tiled.tiled.CANDIDATES on a short sub-sample (the paper autotunes them per
    CPU and plan).  8-bit input only, as in the paper."""
    if cfg.in_dtype != W.U8:
        return None
    from cpu_tiled import tiled
    from oracle import oracle   # only its shift table: the tiled kernel takes shifts as an input
    tiled.build()
    threads = tiled.omp_threads()
    table, mx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
    out_len = cfg.nsamps - mx
    d0 = (cfg.ndm // 2) // 64 * 64
    per_row = float(out_len) * cfg.nchans
    probe_rows = int(min(cfg.ndm - d0, max(64, 2 * threads)))
    best, best_rate = None, 0.0
    for tile in tiled.CANDIDATES:
        t0 = time.perf_counter()
        tiled.dedisperse_u8(x, table[d0:d0 + probe_rows], out_len, tile)
        rate = probe_rows * per_row / (time.perf_counter() - t0)
        if rate > best_rate:
            best, best_rate = tile, rate
    rows = int(min(cfg.ndm - d0, max(probe_rows, budget_s * best_rate / per_row)))
    t0 = time.perf_counter()
    tiled.dedisperse_u8(x, table[d0:d0 + rows], out_len, best)
    dt = time.perf_counter() - t0
    return {"value": rows * per_row / dt, "unit": UNIT, "cores": threads,
            "kind": "paper Algorithm 2 (tiled OpenMP + SIMD CPU kernel, cpu_tiled/)",
            "tile": {"D_t": best[0], "D_dm": best[1], "D_f": best[2], "acc16": best[3]},
            "sample": "DM rows %d..%d of %d x full out_len x all %d channels, %.1f s"
                      % (d0, d0 + rows, cfg.ndm, cfg.nchans, dt)}


def run_reference(args):
    rank, _, world = _dist_env()
    if rank != 0:
        return 0
    cfg = W.ALL_CONFIGS[args.config]
    base, ms = time_oracle(cfg, args.steps, args.warmup)
    from oracle import oracle
    line = {"impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT,
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": _dtype_name(cfg), "data": "synthetic",
            "config": _config_dict(cfg, _OracleFacts(cfg, oracle)), "cpu_baseline": base,
            "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def _dtype_name(cfg):
    return {W.U8: "u8 in, packed u16/u32 integer accumulate, u32 out",
            W.U16: "u16 in, u32 integer accumulate, u32 out",
            W.F32: "f32",
            W.U4: "u4 in (eight 4-bit lanes per word on chip), packed u8/u16/u32 integer accumulate, u32 out"}[cfg.in_dtype]


class _OracleFacts:
    """out_len / max_shift / ndm of a config from the ORACLE's shift table, for the reference
    arm's `config` (same keys and values as our arm's, which takes them from the plan)."""

    def __init__(self, cfg, oracle):
        _, mx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
        self.max_shift, self.out_len, self.ndm = mx, cfg.nsamps - mx, cfg.ndm


def _config_dict(cfg, plan):
    d = {"workload": cfg.name + ("" if (cfg.nsamps, cfg.ndm, cfg.dm_step) == W.ALL_CONFIGS_SHAPE.get(cfg.name)
                                 else " (nsamps / ndm / dm_step overridden)"), "nchans": cfg.nchans, "nsamps": cfg.nsamps, "ndm": cfg.ndm,
         "dm_step": cfg.dm_step, "f_high_MHz": cfg.f_high, "chan_bw_MHz": cfg.chan_bw,
         "tsamp_s": cfg.tsamp, "in_dtype": W.DTYPE_NAME[cfg.in_dtype],
         "l2": "input (%.2f GiB) and output are each larger than the 126 MB L2; no flush needed"
               % (cfg.nchans * cfg.nsamps * W.ELEM_BYTES[cfg.in_dtype] / 2 ** 30)}
    d.update({"out_len": plan.out_len, "max_shift": plan.max_shift,
              "adds_per_step": plan.ndm * plan.out_len * cfg.nchans,
              "adds_nominal": cfg.ndm * cfg.nsamps * cfg.nchans})
    return d


def _tile_string(plan):
    return ("D_DM=%d x D_J=%d superwords x %d lanes, CH=%d, %d stages, %d B smem, grid %d x %d threads"
            % (plan.info("D_DM"), plan.info("D_J"), plan.info("LANES"), plan.info("CH"),
               plan.info("NSTAGE"), plan.info("SMEM_BYTES"), plan.info("GRID"), plan.info("THREADS")))


# ------------------------------------------------------------------------- measured on-chip peaks
PROBE_UNITS = {"SM_COUNT": "SMs", "SM_CLOCK_MHZ": "MHz", "LDS32": "B/clk/SM", "LDS64": "B/clk/SM",
               "LDS128": "B/clk/SM", "TMEM_LD": "B/clk/SM", "TMEM_LD_WITH_LDS": "B/clk/SM (each of TMEM and LDS.64)",
               "F32_ADDS_SMEM_ONLY": "f32 adds/clk/SM", "F32_ADDS_TMEM_4_OF_8": "f32 adds/clk/SM",
               "F32_ADDS_TMEM_4_OF_8_NO_FILL": "f32 adds/clk/SM"}


ROOFLINE_PROBES = ("SM_COUNT", "SM_CLOCK_MHZ", "LDS32", "LDS64", "LDS128", "IADD3", "FADD")


def measure_peaks(B, keys=None):
    """dd_probe key -> value (lane-instructions or bytes per clock per SM, SM clock, SM count); every key
    for --probe-peaks, only the roofline denominators (ROOFLINE_PROBES) inside a benchmark run."""
    return {k: B.probe(k) for k in (keys or B.PROBES)}


def run_probe_peaks(args):
    """--probe-peaks: run the library's on-chip probes (include/dd.h dd_probe) and print them as one
    JSON line: the measured denominators of `roofline` / `roofline_alu`."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    from paper_2311_05341_b200 import binding as B, build
    build.build()
    p = measure_peaks(B)
    nsm, mhz = p["SM_COUNT"], p["SM_CLOCK_MHZ"]
    line = {"probe": "dd_probe", "device": torch.cuda.get_device_name(0),
            "per_clk_per_sm": {k: v for k, v in p.items() if k not in ("SM_COUNT", "SM_CLOCK_MHZ")},
            "units": {k: PROBE_UNITS.get(k, "lane-instructions/clk/SM") for k in p},
            "sm_count": nsm, "sm_clock_mhz": mhz,
            "smem_read_peak_gbs": max(p["LDS32"], p["LDS64"], p["LDS128"]) * nsm * mhz * 1e6 / 1e9,
            "int_add_peak_tlane_s": p["IADD3"] * nsm * mhz * 1e6 / 1e12,
            "fp32_add_peak_tlane_s": p["FADD"] * nsm * mhz * 1e6 / 1e12}
    print(json.dumps(line))
    return 0


def _sources_sha16():
    """First 16 hex digits of the sha256 of the sources that decide the main kernel's DRAM traffic (the
    kernels and the plan-time tiling / rasterisation): a traffic capture is quoted only for the tree it
    was taken on (the GPU box has no .git to ask)."""
    import hashlib
    h = hashlib.sha256()
    for f in ("dd_kernels.cu", "dd_host.cpp"):
        with open(os.path.join(ROOT, "paper_2311_05341_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


TRAFFIC_CSV = os.path.join("profiles", "r03_traffic.csv")


def _traffic_for(name: str):
    """(DRAM bytes per dedisperse_kernel launch, note) from the committed ncu capture of this workload,
    or (None, why) when there is none for the current sources."""
    path = os.path.join(ROOT, TRAFFIC_CSV)
    if not os.path.exists(path):
        return None, "no " + TRAFFIC_CSV
    sha = _sources_sha16()
    with open(path) as f:
        rows = [ln.split(",") for ln in f.read().splitlines()[1:] if ln and not ln.startswith("#")]
    for fld in rows:
        if fld[0] == name:
            if fld[-1].strip() != sha:
                return None, ("%s holds a capture of other kernel sources (%s, now %s): not quoted"
                              % (TRAFFIC_CSV, fld[-1].strip(), sha))
            return int(fld[1]), ("ncu dram__bytes_read.sum + dram__bytes_write.sum of one launch, %s, "
                                 "sources sha16 %s" % (TRAFFIC_CSV, sha))
    return None, "no row for %s in %s" % (name, TRAFFIC_CSV)


def _smem_roofline(name, adds, in_b, hbm_alg_bytes, main_s, share, probed, run_mhz, overridden=False):
    """The main kernel against the shared-memory pipe (one sample read from shared memory per add,
    DESIGN.md section 7).  The peak is dd_probe's measured bytes per clock per SM times the SM clock
    SAMPLED DURING THE TIMED REGION (the probes themselves run cooler and clock a little lower); the
    fraction at the probe's own clock is printed beside it."""
    n_sm = int(probed["SM_COUNT"])
    b_clk = max(probed["LDS32"], probed["LDS64"], probed["LDS128"])
    probe_mhz = probed["SM_CLOCK_MHZ"]
    mhz = run_mhz if run_mhz else probe_mhz
    peak = n_sm * b_clk * mhz * 1e6 / 1e9
    ach = adds * in_b / main_s / 1e9
    traffic, tnote = (None, "shape overridden on the command line") if overridden else _traffic_for(name)
    return {"bound": "smem", "kernel": "dedisperse_kernel", "achieved": ach, "peak": peak, "unit": "GB/s",
            "frac": ach / peak, "peak_clock_mhz": mhz,
            "peak_clock": "clocks.sm_mhz of this timed region" if run_mhz else "dd_probe clock (no nvidia-smi sample)",
            "frac_at_probe_clock": ach / (n_sm * b_clk * probe_mhz * 1e6 / 1e9),
            "peak_kind": "measured (dd_probe) %.1f B/clk/SM x %d SMs x %.0f MHz; paper Eq. 8 form: 128 B/clk/SM"
                         % (b_clk, n_sm, mhz),
            "traffic": traffic, "traffic_note": tnote, "algorithmic_hbm_bytes": hbm_alg_bytes,
            "hbm_waste": (traffic / hbm_alg_bytes) if traffic else None,
            "algorithmic_bytes_per_add": in_b, "adds_per_launch": adds,
            "kernel_ms": main_s * 1e3, "share_of_step": share}


def _time_config(B, name, sampler, probed, min_region_s=0.6):
    """One extra workload for the default line's `configs` block: device-resident step time (CUDA
    events, >= 5 timed steps after 2 warm-ups, at least `min_region_s` of timed work so that nvidia-smi
    sees it), adds/s, the main kernel's shared-memory roofline and the real-time factor."""
    import torch
    cfg = W.ALL_CONFIGS[name]
    plan = B.Plan(cfg.nchans, cfg.nsamps, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list, cfg.in_dtype)
    try:
        table = plan.shift_table() if cfg.npulses else None
        x = W.make_input_torch(cfg, "cuda", table, plan.out_len)
        del table
        odt = torch.float32 if cfg.in_dtype == W.F32 else torch.int32
        out = torch.empty((plan.ndm, plan.out_len), dtype=odt, device="cuda")
        adds = plan.ndm * plan.out_len * cfg.nchans
        stream = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        plan.execute(x, out)
        e0.record(stream)
        plan.execute(x, out)
        e1.record(stream)
        torch.cuda.synchronize()
        steps = int(min(64, max(5, np.ceil(min_region_s * 1e3 / max(e0.elapsed_time(e1), 1e-3)))))
        plan.set_timing(True)
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(steps):
            plan.execute(x, out)
        e1.record(stream)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        ms_step = e0.elapsed_time(e1) / steps
        plan.set_timing(False)
        il_ms, main_ms = plan.kernel_times(steps)
        clocks = sampler.window(t0, t1)
        main_s, il_s = float(np.mean(main_ms)) * 1e-3, float(np.mean(il_ms)) * 1e-3
        in_b = W.ELEM_BYTES[cfg.in_dtype]
        hbm_alg = int(cfg.nchans * cfg.nsamps * in_b) + plan.ndm * plan.out_len * 4
        return {"value": adds / (ms_step * 1e-3), "unit": UNIT, "ms_per_step": ms_step, "steps": steps, "warmup": 2,
                "in_dtype": W.DTYPE_NAME[cfg.in_dtype], "nchans": cfg.nchans, "nsamps": cfg.nsamps, "ndm": cfg.ndm,
                "dm_step": cfg.dm_step, "out_len": plan.out_len, "adds_per_step": adds, "tile": _tile_string(plan),
                "kernels_ms": {"interleave_kernel": il_s * 1e3, "dedisperse_kernel": main_s * 1e3},
                "roofline": _smem_roofline(name, adds, in_b, hbm_alg, main_s, main_s / (main_s + il_s), probed,
                                           clocks.get("sm_mhz")),
                "realtime_factor": cfg.nsamps * cfg.tsamp / (ms_step * 1e-3), "clocks": clocks,
                "gpu_launches": steps * plan.info("LAUNCHES")}
    finally:
        plan.destroy()


def _time_survey(B, name, sampler, min_region_s=0.6):
    """A survey workload for the `configs` block: dd_survey_execute_tm over a resident time-major block
    (transpose + time binning + every range), the paper's pipeline real-time factor (Eq. 10)."""
    import torch
    sc = W.SURVEYS[name]
    gen = W.Config(sc.name, sc.nchans, sc.nsamps, sc.in_dtype, sc.f_high, sc.chan_bw, sc.tsamp, 1, 0.0,
                   seed=sc.seed, mean=sc.mean, sd=sc.sd)
    x_tm = W.noise_torch(gen, "cuda").t().contiguous()
    sv = B.Survey(sc.nchans, sc.nsamps, sc.f_high, sc.chan_bw, sc.tsamp, sc.ranges, sc.in_dtype)
    try:
        adds = sum(n * ol * sc.nchans for n, ol in zip(sv.ndm, sv.out_len))
        stream = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sv.execute_tm(x_tm)
        e0.record(stream)
        sv.execute_tm(x_tm)
        e1.record(stream)
        torch.cuda.synchronize()
        steps = int(min(32, max(5, np.ceil(min_region_s * 1e3 / max(e0.elapsed_time(e1), 1e-3)))))
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(steps):
            sv.execute_tm(x_tm)
        e1.record(stream)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        ms_step = e0.elapsed_time(e1) / steps
        nbin = len({r[3] for r in sc.ranges if r[3] > 1})
        return {"value": adds / (ms_step * 1e-3), "unit": UNIT, "ms_per_step": ms_step, "steps": steps, "warmup": 2,
                "api": "dd_survey_execute_tm (transpose + time binning + dedispersion of every range)",
                "layout": "time-major", "nchans": sc.nchans, "nsamps": sc.nsamps,
                "ranges": [list(r) for r in sc.ranges], "adds_per_step": adds,
                "realtime_factor": {"R_eq10": sc.t_obs / (ms_step * 1e-3), "t_obs_s": sc.t_obs, "t_c_ms": ms_step},
                "clocks": sampler.window(t0, t1),
                "gpu_launches": steps * ((1 if nbin else 0) + nbin + 2 * len(sc.ranges))}
    finally:
        sv.destroy()


EXTRA_LINE_CONFIGS = ("c2", "c3", "lowfreq", "headline_u4", "paper52", "largeshift")
EXTRA_LINE_SURVEYS = ("survey52",)


# ------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    rank, local_rank, world = _dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    # stdout carries exactly ONE JSON line: anything libraries print (NCCL's version banner) goes
    # to stderr until the line is written
    sys.stdout.flush()
    saved_stdout = os.dup(1)
    os.dup2(2, 1)
    dist = None
    if world > 1 or "TORCHELASTIC_RUN_ID" in os.environ:  # under torch.distributed.run, also at N = 1
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2311_05341_b200 import binding as B, build, shard
    if rank == 0:
        build.build()
    if dist is not None:
        dist.barrier()
    B.lib()

    cfg = W.ALL_CONFIGS[args.config]
    hbm_gbs, sm_max_mhz, peak_kind = _peaks()
    probed = measure_peaks(B, ROOFLINE_PROBES) if rank == 0 else None   # before the timed region
    plan = B.Plan(cfg.nchans, cfg.nsamps, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list, cfg.in_dtype)
    table = plan.shift_table() if cfg.npulses else None
    # every rank: its own block (seed offset by rank), resident in HBM before timing starts
    import dataclasses
    x = W.make_input_torch(dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank), "cuda", table, plan.out_len)
    odt = torch.float32 if cfg.in_dtype == W.F32 else torch.int32
    out = torch.empty((plan.ndm, plan.out_len), dtype=odt, device="cuda")
    adds = plan.ndm * plan.out_len * cfg.nchans
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing
    for _ in range(args.warmup):
        plan.execute(x, out)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    plan.set_timing(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_host0 = time.perf_counter()
    e0.record(stream)
    for _ in range(args.steps):
        plan.execute(x, out)
    e1.record(stream)
    barrier()
    t_host1 = time.perf_counter()
    ms_total = e0.elapsed_time(e1)
    plan.set_timing(False)
    il_ms, main_ms = plan.kernel_times(min(64, args.steps))
    clocks = sampler.stop(t_host0, t_host1) if rank == 0 else None
    # whole job = sum of units over ranks / max of time over ranks (no data-path collective)
    value, ms_total = shard.job_throughput(float(adds) * args.steps, ms_total, dist, "cuda")
    ms_step = ms_total / args.steps

    if args.quick:
        # profiler captures (ncu -k regex:dedisperse ...): the device-resident region only, said in the line
        if rank == 0:
            line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                    "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                    "vs_baseline": None, "dtype": _dtype_name(cfg), "data": "synthetic",
                    "config": _config_dict(cfg, plan), "tile": _tile_string(plan),
                    "kernels_ms": {"interleave_kernel": float(np.mean(il_ms)), "dedisperse_kernel": float(np.mean(main_ms))},
                    "quick": "device-resident region only: no e2e, roofline, cpu_baseline or configs (--quick)",
                    "gpu_launches": args.steps * plan.info("LAUNCHES"), "clocks": clocks}
            sys.stdout.flush()
            os.dup2(saved_stdout, 1)
            print(json.dumps(line), flush=True)
        plan.destroy()
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    # ---- end to end through the C ABI with HOST buffers (H2D + kernels + D2H in the timed region)
    # A streaming caller keeps two blocks in flight: dd_execute_host_async on two plans and two streams,
    # so that the copies of block n+1 overlap the kernels of block n.  Every step copies its whole input
    # from pinned host memory and its whole output plane back.  The latency of one synchronous call
    # (dd_execute_host, nothing else in flight) is reported beside it.
    h_in = torch.empty(x.shape, dtype=x.dtype).pin_memory()
    h_in.copy_(x)
    plan_b = B.Plan(cfg.nchans, cfg.nsamps, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list, cfg.in_dtype)
    pipe_plans = [plan, plan_b]
    h_outs = [torch.empty(out.shape, dtype=out.dtype).pin_memory() for _ in pipe_plans]
    h_out = h_outs[0]
    side = [torch.cuda.Stream() for _ in pipe_plans]
    for p_, h_, s_ in zip(pipe_plans, h_outs, side):   # warm-up (allocates the plans' device buffers)
        p_.execute_host_async(h_in, h_, s_)
    barrier()
    single_steps = max(1, min(args.steps, 3))
    e0.record(stream)
    for _ in range(single_steps):
        plan.execute_host(h_in, h_out)
    e1.record(stream)
    barrier()
    ms_single = e0.elapsed_time(e1) / single_steps
    tl = plan.host_timeline()   # of that synchronous call: where its time goes
    e2e_steps = max(6, min(args.steps, 12))
    for h_ in h_outs:
        h_.zero_()
    barrier()
    e0.record(stream)
    for s_ in side:
        s_.wait_event(e0)
    for i in range(e2e_steps):
        pipe_plans[i % 2].execute_host_async(h_in, h_outs[i % 2], side[i % 2])
    for s_ in side:
        stream.wait_stream(s_)
    e1.record(stream)
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    e2e_value, ms_e2e = shard.job_throughput(float(adds) * e2e_steps, ms_e2e, dist, "cuda")
    ms_e2e /= e2e_steps
    h2d = h_in.numel() * h_in.element_size()
    d2h = h_out.numel() * h_out.element_size()
    e2e_timeline = [{"out_begin": int(o), "h2d_done_ms": round(float(a_), 2), "prepass_done_ms": round(float(b_), 2),
                     "main_done_ms": round(float(c_), 2), "d2h_done_ms": round(float(d_), 2)}
                    for o, a_, b_, c_, d_ in zip(*tl)]
    # the timed host path must reproduce the device-resident plane bit for bit (same kernels, same
    # per-output summation order -- float32 too); tests/ tie that plane to the oracle
    plan.execute(x, out)
    torch.cuda.synchronize()
    out_host = out.cpu()
    e2e_verified = all(bool(torch.equal(h_, out_host)) for h_ in h_outs)
    del out_host
    if not e2e_verified:
        raise SystemExit("bench.py: dd_execute_host_async output differs from dd_execute output")
    plan_b.destroy()
    del h_outs

    # ---- time-major input: transpose pre-step + the same path
    tm = None
    if rank == 0:
        if cfg.in_dtype == W.U4:
            # repack along channels (reading R16): unpack, transpose, pack pairs of channels
            v = torch.stack((x & 15, x >> 4), dim=2).reshape(cfg.nchans, cfg.nsamps).t().contiguous()
            x_tm = (v[:, 0::2] | (v[:, 1::2] << 4)).contiguous()
            del v
        else:
            x_tm = x.t().contiguous()
        x_cm = torch.empty_like(x)
        tms, tot = [], []
        plan.set_timing(True)
        for i in range(4):
            e0.record(stream)
            plan.execute_tm(x_tm, out)          # fused transpose + interleave pre-pass, same main kernel
            e1.record(stream)
            torch.cuda.synchronize()
            if i:
                tot.append(e0.elapsed_time(e1))
            e0.record(stream)
            B.transpose(x_tm, x_cm, cfg.nchans, cfg.nsamps, cfg.in_dtype)   # stand-alone transpose
            e1.record(stream)
            torch.cuda.synchronize()
            if i:
                tms.append(e0.elapsed_time(e1))
        il_tm, _ = plan.kernel_times(3)
        plan.set_timing(False)
        # end to end from a time-major pinned host block (contiguous chunk copies)
        h_tm = torch.empty(x_tm.shape, dtype=x_tm.dtype).pin_memory()
        h_tm.copy_(x_tm)
        del x_tm, x_cm
        plan.execute_host_tm(h_tm, h_out)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(3):
            plan.execute_host_tm(h_tm, h_out)
        e1.record(stream)
        torch.cuda.synchronize()
        ms_e2e_tm = e0.elapsed_time(e1) / 3
        del h_tm
        tbytes = 2.0 * cfg.nchans * cfg.nsamps * W.ELEM_BYTES[cfg.in_dtype]
        tm = {"api": "dd_execute_tm (fused pre-pass); roofline = stand-alone dd_transpose",
              "fused_prepass_ms": float(np.mean(il_tm)), "transpose_kernel_ms": float(np.mean(tms)),
              "step_ms": float(np.mean(tot)), "value": adds / (float(np.mean(tot)) * 1e-3), "unit": UNIT,
              "e2e": {"api": "dd_execute_host_tm (pinned host buffers)", "ms_per_step": ms_e2e_tm,
                      "value": adds / (ms_e2e_tm * 1e-3), "unit": UNIT},
              "roofline": {"bound": "hbm", "achieved": tbytes / (float(np.mean(tms)) * 1e-3) / 1e9,
                           "peak": hbm_gbs, "unit": "GB/s",
                           "frac": tbytes / (float(np.mean(tms)) * 1e-3) / 1e9 / hbm_gbs,
                           "algorithmic_bytes": tbytes}}

    # ---- time binning by 2 of the same block: HBM-bound pre-step
    binning = None
    if rank == 0 and cfg.in_dtype != W.U16:
        nout = cfg.nsamps // 2
        bdt = {W.U8: torch.int16, W.U4: torch.uint8, W.F32: torch.float32}[cfg.in_dtype]
        xb = torch.empty((cfg.nchans, nout), dtype=bdt, device="cuda")
        ts = []
        for i in range(4):
            e0.record(stream)
            B.bin_time(x, xb, cfg.nchans, cfg.nsamps, 2, cfg.in_dtype)
            e1.record(stream)
            torch.cuda.synchronize()
            if i:
                ts.append(e0.elapsed_time(e1))
        bbytes = x.numel() * x.element_size() + xb.numel() * xb.element_size()
        binning = {"api": "dd_bin_time", "factor": 2, "kernel_ms": float(np.mean(ts)),
                   "roofline": {"bound": "hbm", "achieved": bbytes / (float(np.mean(ts)) * 1e-3) / 1e9,
                                "peak": hbm_gbs, "unit": "GB/s",
                                "frac": bbytes / (float(np.mean(ts)) * 1e-3) / 1e9 / hbm_gbs,
                                "algorithmic_bytes": bbytes}}
        del xb

    if rank != 0:
        plan.destroy()
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    # ---- rooflines of the dominant kernel (dedisperse_kernel), from its own CUDA events
    main_s = float(np.mean(main_ms)) * 1e-3
    il_s = float(np.mean(il_ms)) * 1e-3
    kadds = adds / main_s
    # measured on this device by the library's own probes (dd_probe): bytes per clock per SM read
    # from shared memory (best of LDS.32/.64/.128), IADD3 lane-instructions per clock per SM, and
    # the SM clock during the probes; the derived figures (paper Eq. 8) are reported beside them
    n_sm = int(probed["SM_COUNT"])
    int_peak_derived = N_SM * INT_LANES_PER_SM_CLK * sm_max_mhz * 1e6
    in_b = W.ELEM_BYTES[cfg.in_dtype]                   # bytes a sample occupies in shared memory (4-bit: 0.5)
    hbm_alg_bytes = int(cfg.nchans * cfg.nsamps * in_b) + plan.ndm * plan.out_len * 4
    overridden = (cfg.nsamps, cfg.ndm, cfg.dm_step) != W.ALL_CONFIGS_SHAPE.get(cfg.name)
    share = main_s / (main_s + il_s)
    run_mhz = clocks.get("sm_mhz") if clocks else None
    # The dominant kernel reads one sample from shared memory per add: `roofline` is the shared-memory
    # pipe for EVERY input type (the paper's own accounting, Eq. 8; ncu: 90-99 % of peak wavefronts for
    # u8 / u16 / f32), reported in bytes, with the peak at the clock sampled during the timed region.
    roofline = _smem_roofline(cfg.name, adds, in_b, hbm_alg_bytes, main_s, share, probed, run_mhz, overridden)
    alu_mhz = run_mhz if run_mhz else probed["SM_CLOCK_MHZ"]
    int_peak = n_sm * probed["IADD3"] * alu_mhz * 1e6
    roofline_alu = {"bound": "alu", "achieved": kadds / 1e12, "peak": int_peak / 1e12, "unit": "Tadd/s",
                    "frac": kadds / int_peak,
                    "peak_kind": "measured (dd_probe): %.1f IADD3 lanes/clk/SM x %d SMs x %.0f MHz; derived %.2f Tadd/s"
                                 % (probed["IADD3"], n_sm, alu_mhz, int_peak_derived / 1e12),
                    "note": "sample-adds against one-add-per-lane integer peak (BASELINE.json's metric); "
                            "a packed add performs 8 (u4) / 4 (u8) / 2 (u16) sample-adds, so frac may exceed 1"}
    roofline_alu_pipe = None
    if cfg.in_dtype == W.U4:
        # Secondary view for the 4-bit kernel, which sits nearer its alu-pipe limit than its shared-memory
        # one (ncu, profiles/r02_headline_u4_dedisperse_details.txt: alu 83 % busy,
        # shared-memory wavefronts 76 %): per 32-bit word (8 sample-adds) the odd nibbles cost one LOP3 and
        # one LEA.HI on that pipe.  A builder-defined instruction count, so not comparable across types:
        # it explains the shared-memory fraction above, it does not replace it.
        alu_ops = adds * 2.0 / 8.0
        roofline_alu_pipe = {"bound": "alu", "kernel": "dedisperse_kernel", "achieved": alu_ops / main_s / 1e12,
                             "peak": int_peak / 1e12, "unit": "T lane-instructions/s",
                             "frac": alu_ops / main_s / int_peak,
                             "algorithmic_alu_instructions_per_add": 0.25,
                             "note": "alu-pipe lane-instructions (LOP3 + LEA.HI per 8 adds) against the measured "
                                     "IADD3 issue rate; secondary to `roofline`"}
    roofline_hbm = {"bound": "hbm", "achieved": hbm_alg_bytes / (ms_step * 1e-3) / 1e9, "peak": hbm_gbs,
                    "unit": "GB/s", "frac": hbm_alg_bytes / (ms_step * 1e-3) / 1e9 / hbm_gbs,
                    "peak_kind": peak_kind + " copy bandwidth",
                    "staged_l2_to_smem_bytes": plan.info("STAGE_BYTES")}

    x_host = h_in.numpy() if cfg.in_dtype != W.U16 else h_in.view(torch.int16).numpy().view(np.uint16)
    cpu_base, _ = time_oracle(cfg, 1, 1, x=x_host)
    cpu_tiled = time_tiled(cfg, x_host)
    gpu_launches = args.steps * plan.info("LAUNCHES")
    tile_string, config_dict = _tile_string(plan), _config_dict(cfg, plan)
    realtime = {"t_obs_over_t": cfg.nsamps * cfg.tsamp / (ms_step * 1e-3),
                "out_len_tsamp_over_t": plan.out_len * cfg.tsamp / (ms_step * 1e-3)}
    # ---- the other workloads, device-resident, in the same line (default run of the headline at N = 1):
    # BASELINE.json's other configs and the section 8(f) workloads, each with its own clocks and roofline
    configs = None
    if cfg.name == "headline" and not overridden and world == 1 and not args.no_configs:
        plan.destroy()
        del x, out, h_in, x_host, h_out
        torch.cuda.empty_cache()
        configs = {}
        sampler2 = ClockSampler(local_rank)
        sampler2.start()
        time.sleep(0.3)
        t_cfg0 = time.perf_counter()
        for name in EXTRA_LINE_CONFIGS:
            configs[name] = _time_config(B, name, sampler2, probed)
            torch.cuda.empty_cache()
        for name in EXTRA_LINE_SURVEYS:
            configs[name] = _time_survey(B, name, sampler2)
            torch.cuda.empty_cache()
        sampler2.close()
        configs["_note"] = ("device-resident dd_execute (surveys: dd_survey_execute_tm) per workload, CUDA events, "
                            ">= 5 timed steps after 2 warm-ups, clocks sampled per workload; %.0f s in all; "
                            "their launches are not in the line's gpu_launches" % (time.perf_counter() - t_cfg0))
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": _dtype_name(cfg),
            "data": "synthetic", "config": config_dict, "tile": tile_string,
            "realtime_factor": realtime,
            "value_nominal": world * cfg.ndm * cfg.nsamps * cfg.nchans / (ms_step * 1e-3),
            "kernels_ms": {"interleave_kernel": il_s * 1e3, "dedisperse_kernel": main_s * 1e3},
            "roofline": roofline, "roofline_alu": roofline_alu, "roofline_alu_pipe": roofline_alu_pipe,
            "roofline_hbm": roofline_hbm,
            "measured_peaks": probed,
            "cpu_baseline": cpu_base, "cpu_baseline_tiled": cpu_tiled,
            "time_major": tm, "time_binning": binning,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e,
                    "steps": e2e_steps, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "api": "dd_execute_host_async, two plans / two blocks in flight (pinned host buffers, default "
                           "chunk schedule): every step copies its input in and its output plane out",
                    "single_call_ms": ms_single,
                    "single_call_note": "dd_execute_host alone (synchronous, one block in flight); its timeline below",
                    "e2e_verified": e2e_verified, "timeline": e2e_timeline},
            "gpu_launches": gpu_launches,
            "clocks": clocks, "configs": configs}
    sys.stdout.flush()
    os.dup2(saved_stdout, 1)
    print(json.dumps(line), flush=True)
    plan.destroy()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------- survey pipeline
def run_survey(args):
    """--config survey52: a multi-range plan over one time-major block through dd_survey_execute_tm
    (transpose + time binning + dedispersion of every range, all in the library).  Reports the
    paper's real-time factor R = t_obs / t_c (Eq. 10: t_c includes transpose and
    binning, not the host->device copy) beside adds/s; `e2e` adds the copies."""
    import torch
    rank, local_rank, world = _dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    sys.stdout.flush()
    saved_stdout = os.dup(1)
    os.dup2(2, 1)
    dist = None
    if world > 1 or "TORCHELASTIC_RUN_ID" in os.environ:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2311_05341_b200 import binding as B, build, shard
    if rank == 0:
        build.build()
    if dist is not None:
        dist.barrier()
    sc = W.SURVEYS[args.config]
    hbm_gbs, _, peak_kind = _peaks()
    import dataclasses
    gen = W.Config(sc.name, sc.nchans, sc.nsamps, sc.in_dtype, sc.f_high, sc.chan_bw, sc.tsamp, 1, 0.0,
                   seed=sc.seed + 1000 * rank, mean=sc.mean, sd=sc.sd)
    x_tm = W.noise_torch(gen, "cuda").t().contiguous()      # [nsamps][nchans], resident in HBM
    sv = B.Survey(sc.nchans, sc.nsamps, sc.f_high, sc.chan_bw, sc.tsamp, sc.ranges, sc.in_dtype)
    adds = sum(n * ol * sc.nchans for n, ol in zip(sv.ndm, sv.out_len))
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        sv.execute_tm(x_tm)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_host0 = time.perf_counter()
    e0.record(stream)
    for _ in range(args.steps):
        sv.execute_tm(x_tm)
    e1.record(stream)
    barrier()
    t_host1 = time.perf_counter()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop(t_host0, t_host1) if rank == 0 else None
    value, ms_total = shard.job_throughput(float(adds) * args.steps, ms_total, dist, "cuda")
    ms_step = ms_total / args.steps

    # pre-steps alone: the transpose and each binning (HBM-bound; algorithmic bytes = read + write)
    def timed(fn, n=3):
        ts = []
        for i in range(n + 1):
            e0.record(stream)
            fn()
            e1.record(stream)
            torch.cuda.synchronize()
            if i:
                ts.append(e0.elapsed_time(e1))
        return float(np.mean(ts))
    x_cm = torch.empty((sc.nchans, sc.nsamps), dtype=x_tm.dtype, device="cuda")
    pre = {"transpose_ms": timed(lambda: B.transpose(x_tm, x_cm, sc.nchans, sc.nsamps, sc.in_dtype))}
    in_bytes = x_tm.numel() * x_tm.element_size()
    pre["transpose_frac_of_hbm"] = 2.0 * in_bytes / (pre["transpose_ms"] * 1e-3) / 1e9 / hbm_gbs
    bdt = {W.U8: torch.int16, W.U4: torch.uint8, W.F32: torch.float32}[sc.in_dtype]
    for f in sorted({r[3] for r in sc.ranges if r[3] > 1}):
        xb = torch.empty((sc.nchans, sc.nsamps // f), dtype=bdt, device="cuda")
        ms = timed(lambda: B.bin_time(x_cm, xb, sc.nchans, sc.nsamps, f, sc.in_dtype))
        pre["bin%d_ms" % f] = ms
        pre["bin%d_frac_of_hbm" % f] = (in_bytes + xb.numel() * xb.element_size()) / (ms * 1e-3) / 1e9 / hbm_gbs
        del xb
    del x_cm

    # end to end: pinned time-major host block -> device, the survey, every output plane -> host; two
    # blocks in flight (two surveys on two streams), so that the copies of one block overlap the kernels
    # of the other; every block copies its whole input in and all its output planes out
    h_in = torch.empty(x_tm.shape, dtype=x_tm.dtype).pin_memory()
    h_in.copy_(x_tm)
    sv_b = B.Survey(sc.nchans, sc.nsamps, sc.f_high, sc.chan_bw, sc.tsamp, sc.ranges, sc.in_dtype)
    pipe = [sv, sv_b]
    side = [torch.cuda.Stream(), torch.cuda.Stream()]
    d_ins = [torch.empty_like(x_tm) for _ in pipe]
    h_outs2 = [[torch.empty(o.shape, dtype=o.dtype).pin_memory() for o in s_.outs] for s_ in pipe]
    h_outs = h_outs2[0]

    def e2e_step(i):
        with torch.cuda.stream(side[i]):
            d_ins[i].copy_(h_in, non_blocking=True)
            outs = pipe[i].execute_tm(d_ins[i], side[i])
            for h, o in zip(h_outs2[i], outs):
                h.copy_(o, non_blocking=True)
    e2e_step(0)
    e2e_step(1)
    barrier()
    nblk = 6
    e0.record(stream)
    for s_ in side:
        s_.wait_event(e0)
    for k in range(nblk):
        e2e_step(k % 2)
    for s_ in side:
        stream.wait_stream(s_)
    e1.record(stream)
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    e2e_value, ms_e2e = shard.job_throughput(float(adds) * nblk, ms_e2e, dist, "cuda")
    ms_e2e /= nblk
    ref_outs = [o.cpu() for o in sv.execute_tm(x_tm)]
    torch.cuda.synchronize()
    e2e_verified = all(bool(torch.equal(h, r)) for hs in h_outs2 for h, r in zip(hs, ref_outs))
    sv_b.destroy()
    if rank != 0:
        sv.destroy()
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0
    ranges = [{"dm_start": a, "dm_step": b, "count": n, "bin_factor": f, "out_len": ol, "max_shift": mx,
               "plan_in_dtype": W.DTYPE_NAME[dt]}
              for (a, b, n, f), ol, mx, dt in zip(sc.ranges, sv.out_len, sv.max_shift, sv.dtype)]
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None,
            "dtype": "u8 in; unbinned range: packed u16/u32 integer accumulate; binned ranges: u16 in, u32 accumulate; u32 out",
            "data": "synthetic",
            "config": {"workload": sc.name, "nchans": sc.nchans, "nsamps": sc.nsamps, "layout": "time-major",
                       "f_high_MHz": sc.f_high, "chan_bw_MHz": sc.chan_bw, "tsamp_s": sc.tsamp,
                       "in_dtype": W.DTYPE_NAME[sc.in_dtype], "ranges": ranges, "adds_per_step": adds,
                       "l2": "input (%.2f GiB) and outputs exceed the 126 MB L2; no flush needed" % (in_bytes / 2 ** 30)},
            "api": "dd_survey_execute_tm (transpose + time binning + dedispersion of every range)",
            "realtime_factor": {"R_eq10": sc.t_obs / (ms_step * 1e-3), "t_obs_s": sc.t_obs, "t_c_ms": ms_step,
                                "note": "t_c includes transpose and binning, not the host copy (PAPER.md:366-370)"},
            "pre_steps": pre,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e, "steps": nblk,
                    "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": sum(h.numel() * 4 for h in h_outs),
                    "api": "pinned host block -> device copy, dd_survey_execute_tm, every output plane -> pinned host; "
                           "two blocks in flight on two surveys and two streams",
                    "R_eq10_with_copies": sc.t_obs / (ms_e2e * 1e-3), "e2e_verified": e2e_verified},
            "gpu_launches": args.steps * (1 + len({r[3] for r in sc.ranges if r[3] > 1}) + 2 * len(sc.ranges)),
            "clocks": clocks}
    sys.stdout.flush()
    os.dup2(saved_stdout, 1)
    print(json.dumps(line), flush=True)
    sv.destroy()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def _apply_overrides(args):
    import dataclasses
    if args.config not in W.ALL_CONFIGS:
        return
    if args.nsamps:
        base = W.ALL_CONFIGS[args.config]
        W.ALL_CONFIGS[args.config] = dataclasses.replace(base, nsamps=args.nsamps, name=base.name)
    if args.dm_step or args.ndm:   # (single-range configs only)
        base = W.ALL_CONFIGS[args.config]
        W.ALL_CONFIGS[args.config] = dataclasses.replace(base, dm_step=args.dm_step or base.dm_step,
                                                         ndm=args.ndm or base.ndm, name=base.name)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="headline", choices=list(W.ALL_CONFIGS) + list(W.SURVEYS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--probe-peaks", action="store_true",
                    help="only run the library's on-chip peak probes (dd_probe) and print them")
    ap.add_argument("--no-configs", action="store_true",
                    help="headline only: leave out the `configs` block (the other workloads, about a minute)")
    ap.add_argument("--quick", action="store_true",
                    help="device-resident region only (for profiler captures); the line says so")
    ap.add_argument("--nsamps", type=int, default=0,
                    help="override the config's block length (sanity check: adds/s should not depend "
                         "on the observation length, PAPER.md:287); the line's config says so")
    ap.add_argument("--dm-step", type=float, default=0.0,
                    help="override the config's DM step (walks down the DM-block ladder: the ladder table in profiles/r02_summary.md)")
    ap.add_argument("--ndm", type=int, default=0, help="override the config's number of DM trials")
    args = ap.parse_args()
    _apply_overrides(args)
    if args.config in W.SURVEYS:
        if args.impl == "reference":   # the oracle arm times single plans only
            print(json.dumps({"impl": "reference", "unavailable": "survey workloads have no oracle timing arm"}))
            return 0
        return run_survey(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.probe_peaks:
        return run_probe_peaks(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
