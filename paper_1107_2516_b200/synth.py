"""Seeded synthetic filterbank inputs and the five BASELINE.json workload descriptions.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no delay formula, no shift computation, no de-dispersion.  Pulse injection
takes the integer shift row of the pulse's DM trial as an ARGUMENT (tests pass the oracle's
table, bench.py passes the library's; the two are bit-identical by test).

The paper's inputs were SIGPROC ``fake`` filterbanks -- per-channel N(0,1) noise plus a square
pulse along the dispersion curve -- and constant-valued buffers
(PAPER.md:191).  Neither SIGPROC nor its files exist here, so these seeded stand-ins reproduce
the shapes and statistics.
"""
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field
import os

import numpy as np

BASE_SEED = 11072516


@dataclass
class Config:
    name: str
    nchans: int
    f_top_mhz: float       # frequency of channel 0 (highest), MHz
    df_mhz: float          # channel width magnitude, MHz (channels descend)
    t_samp_ms: float
    n_out: int             # output samples per DM trial (per chunk for streaming)
    ndm: int
    dm_step: float
    dtype: str = "f32"     # "f32" (float in / float out) or "u8" (uint8 in / int32 out)
    nsub: int = 0          # >0: subband two-stage plan
    nfine: int = 0
    nbeams: int = 1
    nchunks: int = 1
    npulses: int = 0
    pulse_width_ms: tuple = (0.5, 5.0)
    pulse_amp: tuple = (0.5, 2.0)
    seed: int = 0
    fixed_pulses: list = field(default_factory=list)   # [(trial, t_start, width_samples, amp)]

    @property
    def dm_list(self):
        # built as d*step (one multiply), never by accumulation (reading R4)
        return np.arange(self.ndm, dtype=np.float64) * self.dm_step

    def plan_args(self):
        return dict(nchans=self.nchans, f_top_mhz=self.f_top_mhz, df_mhz=self.df_mhz,
                    t_samp_ms=self.t_samp_ms, dm_list=self.dm_list, nsub=self.nsub, nfine=self.nfine)


def span(lo_mhz, hi_mhz, nchans):
    """A band "spanning lo-hi MHz": f_top = hi, df = (hi-lo)/nchans (reading R2)."""
    return float(hi_mhz), (float(hi_mhz) - float(lo_mhz)) / nchans


def configs():
    c = {}
    c[1] = Config("cfg1_tiny", 128, 150.0, 0.05, 0.1, 8192, 64, 0.1, seed=BASE_SEED + 1,
                  fixed_pulses=[(30, 3000, 10, 3.0)])
    ft, df = span(137.0, 143.0, 1024)
    c[2] = Config("cfg2_lofar", 1024, ft, df, 0.0512, 65536, 2048, 0.05, seed=BASE_SEED + 2,
                  npulses=5, pulse_width_ms=(0.5, 5.0), pulse_amp=(0.5, 2.0))
    ft, df = span(1182.0, 1582.0, 1024)
    c[3] = Config("cfg3_lband", 1024, ft, df, 0.064, 262144, 4096, 0.5, seed=BASE_SEED + 3,
                  npulses=10, pulse_width_ms=(0.5, 10.0), pulse_amp=(0.25, 2.0))
    ft, df = span(120.0, 150.0, 4096)
    c[4] = Config("cfg4_subband", 4096, ft, df, 0.05, 131072, 4096, 0.05, seed=BASE_SEED + 4,
                  nsub=32, nfine=32, npulses=8, pulse_width_ms=(2.0, 10.0), pulse_amp=(0.25, 1.0))
    ft, df = span(1200.0, 1500.0, 2048)
    c[5] = Config("cfg5_stream_u8", 2048, ft, df, 0.064, 65536, 3072, 0.5, dtype="u8",
                  seed=BASE_SEED + 5, nbeams=4, nchunks=16, npulses=8,
                  pulse_width_ms=(0.5, 5.0), pulse_amp=(0.5, 2.0))
    return c


def scaled(cfg, **kw):
    """A copy of cfg with some fields replaced (smaller parity-test variants)."""
    d = dict(cfg.__dict__)
    d.update(kw)
    d["fixed_pulses"] = list(d["fixed_pulses"])
    return Config(**d)


def _chan_rng(seed, beam, c):
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(seed), int(beam), int(c)])))


def draw_pulses(cfg, n_out, beam=0):
    """Pulse parameters: trial index uniform over the DM list, start uniform in [0, n_out-w),
    width and per-channel amplitude uniform in cfg's ranges.  Returns [(trial, t, w, amp)]."""
    out = list(cfg.fixed_pulses)
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(cfg.seed) + 1000, beam])))
    for _ in range(cfg.npulses):
        trial = int(rng.integers(0, cfg.ndm))
        w = max(1, int(round(rng.uniform(*cfg.pulse_width_ms) / cfg.t_samp_ms)))
        amp = float(rng.uniform(*cfg.pulse_amp))
        t0 = int(rng.integers(0, max(1, n_out - w)))
        out.append((trial, t0, w, amp))
    return out


def make_input(cfg, n_in, pulses=(), shift_rows=None, beam=0, out=None, threads=None):
    """[nchans][n_in] array: float32 N(0,1) (cfg.dtype f32) or uint8
    round(128 + 16*(N(0,1) + pulse)) clipped to 0..255 (cfg.dtype u8).

    pulses: [(trial, t_start, width, amp)]; shift_rows: {trial: int array [nchans]} -- the integer
    shift of every channel at that trial, supplied by the caller.  The pulse adds amp to
    x[c][t_start + shift_rows[trial][c] + j], j in [0, width) (clipped to the array)."""
    nch = cfg.nchans
    is_u8 = cfg.dtype == "u8"
    if out is None:
        out = np.empty((nch, n_in), dtype=np.uint8 if is_u8 else np.float32)
    assert out.shape == (nch, n_in)

    def one(c):
        g = _chan_rng(cfg.seed, beam, c).standard_normal(n_in, dtype=np.float32)
        for (trial, t0, w, amp) in pulses:
            a = t0 + int(shift_rows[trial][c])
            lo, hi = max(0, a), min(n_in, a + w)
            if hi > lo:
                g[lo:hi] += np.float32(amp)
        if is_u8:
            v = np.rint(np.float32(128.0) + np.float32(16.0) * g)
            np.clip(v, 0, 255, out=v)
            out[c] = v.astype(np.uint8)
        else:
            out[c] = g

    nthr = threads or min(32, os.cpu_count() or 1)
    if nthr > 1 and nch >= 8:
        with ThreadPoolExecutor(nthr) as ex:
            list(ex.map(one, range(nch), chunksize=max(1, nch // (nthr * 4))))
    else:
        for c in range(nch):
            one(c)
    return out
