"""Seeded synthetic workloads: the five BASELINE.json configs and their input generators.

This module serves BOTH the CUDA path (tests, bench.py) and the CPU oracle (tests), so it
holds none of the method's arithmetic: no dispersion law, no shift computation, no sums.
Where a generator needs integer shifts (to inject a dispersed pulse) the caller passes the
shift row in -- from the oracle in oracle tests, from ``dd_plan_shift_table`` elsewhere.

The paper measured on SIGPROC ``fake`` filterbank files, which
are not available; these Gaussian-noise generators take the shapes, bit depths, bands and
sampling times of those workloads and stand in for them (recipe in DESIGN.md "Inputs").
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

U8, U16, F32, U4 = 0, 1, 2, 3   # U4: packed 4-bit, two samples per byte, earlier one in the low nibble
NP_DTYPE = {U8: np.uint8, U16: np.uint16, F32: np.float32, U4: np.uint8}
DTYPE_NAME = {U8: "u8", U16: "u16", F32: "f32", U4: "u4"}
ELEM_BYTES = {U8: 1, U16: 2, F32: 4, U4: 0.5}


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config.  Frequencies in MHz, tsamp in seconds."""
    name: str
    nchans: int
    nsamps: int
    in_dtype: int
    f_high: float
    chan_bw: float
    tsamp: float
    ndm: int
    dm_step: float
    seed: int
    mean: float
    sd: float
    # injected boxcar pulses: (dm_index or None = drawn from the seed, amplitude, width)
    pulse_dm_index: int | None = None
    pulse_amp: float = 0.0
    pulse_width: int = 0
    npulses: int = 0
    # multi-range plan (Table 2): ((dm_start, dm_step, count), ...); overrides dm_step
    dm_ranges: tuple = ()
    note: str = field(default="", compare=False)

    @property
    def dm_list(self) -> np.ndarray:
        # one multiply per entry, never a running sum
        if self.dm_ranges:
            return np.concatenate([start + np.arange(n, dtype=np.float64) * step
                                   for start, step, n in self.dm_ranges])
        return np.arange(self.ndm, dtype=np.float64) * self.dm_step

    @property
    def np_dtype(self):
        return NP_DTYPE[self.in_dtype]

    @property
    def t_obs(self) -> float:
        return self.nsamps * self.tsamp


CONFIGS = {
    "tiny": Config("tiny", 64, 4096, U8, 1500.0, -1.5625, 64e-6, 32, 1.0, seed=0,
                   mean=128.0, sd=16.0, pulse_dm_index=17, pulse_amp=20.0, pulse_width=4,
                   npulses=1, note="configs[0]"),
    "c2": Config("c2", 1024, 1 << 18, U8, 1550.0, -0.390625, 64e-6, 1000, 1.0, seed=1,
                 mean=128.0, sd=16.0, note="configs[1]"),
    "c3": Config("c3", 4096, 1 << 18, F32, 1700.0, -0.1953125, 54.61333e-6, 2048, 0.5, seed=2,
                 mean=0.0, sd=1.0, pulse_dm_index=None, pulse_amp=0.5, pulse_width=4,
                 npulses=8, note="configs[2]"),
    "headline": Config("headline", 8192, 1 << 18, U8, 1500.0, -300.0 / 8192, 64e-6, 1024, 2.0,
                       seed=3, mean=128.0, sd=16.0,
                       note="configs[3]; chan_bw is the exact double -300/8192"),
    "lowfreq": Config("lowfreq", 4096, 1 << 20, U16, 190.0, -0.01953125, 655.36e-6, 512, 0.1,
                      seed=4, mean=32768.0, sd=2048.0, note="configs[4]"),
}

# Workloads beyond BASELINE.json's five; bench.py accepts both sets.
EXTRA_CONFIGS = {
    # The paper's own section 5.2 workload at its largest channel count: 8-bit,
    # 64 us, 10 s, 1400 MHz centre, 300 MHz band, Table 2's three DM ranges without binning
    # (3050 trials, DM 0-500).  The paper's figure for it (~5 T adds/s on A100, ~4.5 T on V100,
    # PAPER.md:424) is an average over 512-8192 channels: context, not a like-for-like baseline.
    "paper52": Config("paper52", 8192, 156250, U8, 1550.0, -300.0 / 8192, 64e-6, 3050, 0.0,
                      seed=6, mean=128.0, sd=16.0,
                      dm_ranges=((0.0, 0.1, 1500), (150.0, 0.2, 750), (300.0, 0.25, 800)),
                      note="PAPER.md section 5.2 / Table 2 at 8192 channels"),
    # The large-shift regime (where the paper falls back to its "cache
    # kernel", up to 4x slower): a 300-400 MHz band at 64 us with a coarse DM step -- the shift
    # grows by up to 630 samples per trial, so dd_plan_create goes down its DM-block ladder
    # (3 trials per block, 4 channels per stage instead of 12 and 16).
    "largeshift": Config("largeshift", 4096, 1 << 18, U8, 400.0, -100.0 / 4096, 64e-6, 264, 2.0,
                         seed=8, mean=128.0, sd=16.0,
                         note="large-shift regime, SURVEY.md 8(f) rank 3; not in BASELINE.json"),
    "headline_u4": Config("headline_u4", 8192, 1 << 18, U4, 1500.0, -300.0 / 8192, 64e-6, 1024, 2.0,
                          seed=5, mean=7.5, sd=2.0,
                          note="the headline shape at the paper's 4-bit precision (PAPER.md:295, 424); "
                               "not in BASELINE.json: SURVEY.md 8(f) rank 2"),
}
ALL_CONFIGS = {**CONFIGS, **EXTRA_CONFIGS}


@dataclass(frozen=True)
class SurveyConfig:
    """A multi-range survey plan over one TIME-MAJOR block (dd_survey_*): the pipeline whose time
    the paper's real-time factor counts (transpose + binning + dedispersion)."""
    name: str
    nchans: int
    nsamps: int
    in_dtype: int
    f_high: float
    chan_bw: float
    tsamp: float
    ranges: tuple          # ((dm_start, dm_step, count, bin_factor), ...)
    seed: int
    mean: float
    sd: float
    note: str = field(default="", compare=False)

    @property
    def t_obs(self) -> float:
        return self.nsamps * self.tsamp


SURVEYS = {
    # The paper's section 5.2 block (8-bit, 8192 channels, 64 us, 10 s, 1250-1550 MHz) delivered
    # time-major, with a DDplan-style plan: Table 2's three ranges (the paper
    # runs them without binning) followed by one coarser range, each range binned in time by the
    # factor its DM step has grown by.  The telescope plans of the paper's section 5.5 (DDplan.py
    # output) are not printed in it; this plan stands in for them.
    "survey52": SurveyConfig("survey52", 8192, 156250, U8, 1550.0, -300.0 / 8192, 64e-6,
                             ((0.0, 0.1, 1500, 1), (150.0, 0.2, 750, 2), (300.0, 0.25, 800, 2),
                              (500.0, 0.5, 1000, 4)),
                             seed=7, mean=128.0, sd=16.0,
                             note="PAPER.md section 5.2 block, Table 2 ranges + one, DDplan-style binning"),
}
ALL_CONFIGS_NSAMPS = {k: v.nsamps for k, v in ALL_CONFIGS.items()}
ALL_CONFIGS_SHAPE = {k: (v.nsamps, v.ndm, v.dm_step) for k, v in ALL_CONFIGS.items()}

TINY_PULSE_T0 = 1000


def _quantise(a: np.ndarray, in_dtype: int) -> np.ndarray:
    if in_dtype == F32:
        return a.astype(np.float32)
    if in_dtype == U4:
        return pack_u4(np.clip(np.rint(a), 0, 15).astype(np.uint8))
    hi = 255 if in_dtype == U8 else 65535
    return np.clip(np.rint(a), 0, hi).astype(NP_DTYPE[in_dtype])


def pack_u4(x8: np.ndarray) -> np.ndarray:
    """[nchans, nsamps] values 0..15 -> [nchans, nsamps/2] bytes, sample 2i in the low nibble
    of byte i, sample 2i+1 in the high nibble (data layout only, no method arithmetic)."""
    assert x8.shape[1] % 2 == 0
    return (x8[:, 0::2] | (x8[:, 1::2] << 4)).astype(np.uint8)


def _noise_float_numpy(cfg: Config, nchans: int, nsamps: int) -> np.ndarray:
    """float64 Gaussian noise, before quantisation.  ``tiny`` draws one block from
    ``default_rng(seed)`` (SURVEY.md 8d recipe); the large configs draw one generator per
    channel (``default_rng([seed, c])``) so that any sub-shape is a prefix of the full array."""
    if cfg.name == "tiny":
        return np.random.default_rng(cfg.seed).normal(cfg.mean, cfg.sd, (nchans, nsamps))
    out = np.empty((nchans, nsamps), dtype=np.float64)
    for c in range(nchans):
        out[c] = np.random.default_rng([cfg.seed, c]).normal(cfg.mean, cfg.sd, nsamps)
    return out


def noise_numpy(cfg: Config, nchans: int | None = None, nsamps: int | None = None) -> np.ndarray:
    """Quantised Gaussian noise [nchans, nsamps] of the config's dtype (no pulses)."""
    nchans = cfg.nchans if nchans is None else nchans
    nsamps = cfg.nsamps if nsamps is None else nsamps
    return _quantise(_noise_float_numpy(cfg, nchans, nsamps), cfg.in_dtype)


def noise_torch(cfg: Config, device, nchans: int | None = None, nsamps: int | None = None):
    """The same distribution generated on ``device`` with a seeded torch generator, in
    channel chunks (the 2-8 GiB configs take seconds instead of minutes).  Values differ
    from ``noise_numpy``; whichever array is made is the one handed to both sides."""
    import torch
    nchans = cfg.nchans if nchans is None else nchans
    nsamps = cfg.nsamps if nsamps is None else nsamps
    tdt = {U8: torch.uint8, U16: torch.uint16, F32: torch.float32, U4: torch.uint8}[cfg.in_dtype]
    g = torch.Generator(device=device)
    g.manual_seed(cfg.seed)
    out = torch.empty((nchans, nsamps // 2 if cfg.in_dtype == U4 else nsamps), dtype=tdt, device=device)
    step = max(1, (1 << 26) // nsamps)
    for c0 in range(0, nchans, step):
        c1 = min(nchans, c0 + step)
        a = torch.randn((c1 - c0, nsamps), generator=g, device=device, dtype=torch.float32)
        a.mul_(cfg.sd).add_(cfg.mean)
        if cfg.in_dtype == F32:
            out[c0:c1] = a
        elif cfg.in_dtype == U4:
            b = a.round_().clamp_(0, 15).to(torch.uint8)
            out[c0:c1] = b[:, 0::2] | (b[:, 1::2] << 4)
        else:
            hi = 255 if cfg.in_dtype == U8 else 65535
            a.round_().clamp_(0, hi)
            if cfg.in_dtype == U8:
                out[c0:c1] = a.to(torch.uint8)
            else:
                out[c0:c1].view(torch.int16).copy_(a.to(torch.int32).to(torch.int16))
    return out


def pulse_plan(cfg: Config, out_len: int):
    """(dm_index, t0) of each injected pulse -- drawn from the seed where the config leaves
    them open (c3), fixed for tiny (DM index 17 at t0 = 1000)."""
    if cfg.npulses == 0:
        return []
    if cfg.pulse_dm_index is not None:
        return [(cfg.pulse_dm_index, TINY_PULSE_T0)]
    rng = np.random.default_rng([cfg.seed, 1 << 20])
    dms = rng.integers(0, cfg.ndm, cfg.npulses)
    t0s = rng.integers(0, max(1, out_len - cfg.pulse_width), cfg.npulses)
    return [(int(d), int(t)) for d, t in zip(dms, t0s)]


def inject_pulse_numpy(x: np.ndarray, shift_row: np.ndarray, t0: int, width: int,
                       amp: float) -> None:
    """Add ``amp`` to the FLOAT array x[c, t0 + shift_row[c] + k], k < width, in place
    (before quantisation).  ``shift_row`` is the caller's integer shift row for the pulse's DM."""
    for c in range(x.shape[0]):
        a = t0 + int(shift_row[c])
        x[c, a:a + width] += amp


def inject_pulse_torch(x, shift_row, t0: int, width: int, amp: float, in_dtype: int) -> None:
    import torch
    nchans = x.shape[0]
    rows = torch.arange(nchans, device=x.device).unsqueeze(1)
    cols = (torch.as_tensor(np.asarray(shift_row, dtype=np.int64), device=x.device).unsqueeze(1)
            + t0 + torch.arange(width, device=x.device).unsqueeze(0))
    if in_dtype == F32:
        x[rows, cols] = x[rows, cols] + amp
    elif in_dtype == U8:
        v = x[rows, cols].to(torch.float32) + amp
        x[rows, cols] = v.round().clamp(0, 255).to(torch.uint8)
    else:
        xv = x.view(torch.int16)
        v = (xv[rows, cols].to(torch.int32) & 0xFFFF).to(torch.float32) + amp
        xv[rows, cols] = v.round().clamp(0, 65535).to(torch.int32).to(torch.int16)


def make_input_numpy(cfg: Config, table: np.ndarray | None, out_len: int | None,
                     nchans: int | None = None, nsamps: int | None = None,
                     noise: bool = True) -> np.ndarray:
    """Noise + the config's pulses, then rint / clip to the input dtype.  ``table``
    ([ndm, nchans] int32 from the caller) is only needed when the config injects pulses.
    ``noise=False`` gives the noise-free variant (every sample = mean) used by pulse pins."""
    nchans = cfg.nchans if nchans is None else nchans
    nsamps = cfg.nsamps if nsamps is None else nsamps
    if noise:
        x = _noise_float_numpy(cfg, nchans, nsamps)
    else:
        x = np.full((nchans, nsamps), cfg.mean, dtype=np.float64)
    if cfg.npulses:
        assert table is not None and out_len is not None
        for d, t0 in pulse_plan(cfg, out_len):
            inject_pulse_numpy(x, table[d], t0, cfg.pulse_width, cfg.pulse_amp)
    return _quantise(x, cfg.in_dtype)


def make_input_torch(cfg: Config, device, table: np.ndarray | None, out_len: int | None):
    x = noise_torch(cfg, device)
    if cfg.npulses:
        assert table is not None and out_len is not None
        for d, t0 in pulse_plan(cfg, out_len):
            inject_pulse_torch(x, table[d], t0, cfg.pulse_width, cfg.pulse_amp, cfg.in_dtype)
    return x
