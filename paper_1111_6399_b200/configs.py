"""The five BASELINE.json:configs as data (c1..c5), plus shrunken variants for tests.

Holds shapes, band, sampling, DM plan and the noise/pulse recipe only — none of
the method's arithmetic (no delay formula lives here; pulse injection in
``synth.py`` takes the integer shift table as an argument).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Tuple

import numpy as np

SEED0 = 11116399  # seed_i = 11116399 + i


@dataclass(frozen=True)
class SurveyConfig:
    name: str
    nchans: int
    fch1: float            # MHz, centre of channel 0 (highest frequency)
    foff: float            # MHz, negative
    tsamp: float           # s
    nsamp_out: int
    dm_segments: Tuple[Tuple[float, float, int], ...]  # (start, step, count); DM = start + i*step
    dtype: str             # "u8" | "f16" | "f32"
    noise_mean: float
    noise_sigma: float
    pulse_amp: float
    npulses: int
    seed: int
    nbeams: int = 1
    nchunks: int = 1       # streaming: consecutive chunks of nsamp_out samples
    fixed_pulses: Tuple[Tuple[int, int], ...] = ()  # (dm index, t0); else seeded positions

    def dm_list(self) -> np.ndarray:
        parts = [start + np.arange(n, dtype=np.float64) * step for start, step, n in self.dm_segments]
        return np.concatenate(parts)

    @property
    def ndm(self) -> int:
        return sum(n for _, _, n in self.dm_segments)

    @property
    def np_dtype(self):
        return {"u8": np.uint8, "f16": np.float16, "f32": np.float32}[self.dtype]

    @property
    def esize(self) -> int:
        return {"u8": 1, "f16": 2, "f32": 4}[self.dtype]

    @property
    def adds(self) -> int:
        """One add per (DM, channel, sample) — the metric's unit (BASELINE.json:metric)."""
        return self.ndm * self.nchans * self.nsamp_out * self.nbeams * self.nchunks


C1 = SurveyConfig("c1_tiny_f32", 64, 1500.0, -1.0, 64e-6, 4096, ((0.0, 1.0, 64),),
                  "f32", 0.0, 1.0, 5.0, 1, SEED0 + 1, fixed_pulses=((30, 1000),))
C2 = SurveyConfig("c2_lofar_u8", 496, 159.0, -32.0 / 496.0, 327.68e-6, 65536, ((0.0, 0.05, 2000),),
                  "u8", 128.0, 16.0, 20.0, 3, SEED0 + 2)
C3 = SurveyConfig("c3_meerkat_f32", 4096, 1712.0, -856.0 / 4096.0, 64e-6, 131072, ((0.0, 0.5, 4096),),
                  "f32", 0.0, 1.0, 0.5, 5, SEED0 + 3)
C4 = SurveyConfig("c4_f16_nonuniform", 8192, 600.0, -300.0 / 8192.0, 81.92e-6, 65536,
                  ((0.0, 0.1, 2000), (200.0, 0.25, 1200), (500.0, 0.5, 1000)),
                  "f16", 0.0, 1.0, 0.5, 5, SEED0 + 4)
C5 = SurveyConfig("c5_stream_u8", 1024, 1530.0, -0.3125, 64e-6, 32768, ((0.0, 1.0, 1024),),
                  "u8", 128.0, 12.0, 20.0, 4, SEED0 + 5, nbeams=32, nchunks=60)

CONFIGS = {"c1": C1, "c2": C2, "c3": C3, "c4": C4, "c5": C5}


def shrink(cfg: SurveyConfig, nchans=None, nsamp_out=None, ndm_stride: int = 1,
           nbeams=None, nchunks=None) -> SurveyConfig:
    """A smaller plan with the same band edges / DM range, for oracle-sized parity tests.

    ``nchans`` fewer, wider channels over the same band; ``ndm_stride`` keeps every
    k-th DM trial of each segment; ``nsamp_out`` shorter output.
    """
    out = cfg
    if nchans is not None and nchans != cfg.nchans:
        out = replace(out, nchans=nchans, foff=cfg.foff * cfg.nchans / nchans)
    if nsamp_out is not None:
        out = replace(out, nsamp_out=nsamp_out)
    if ndm_stride != 1:
        segs = tuple((s, st * ndm_stride, (n + ndm_stride - 1) // ndm_stride) for s, st, n in cfg.dm_segments)
        out = replace(out, dm_segments=segs)
    if nbeams is not None:
        out = replace(out, nbeams=nbeams)
    if nchunks is not None:
        out = replace(out, nchunks=nchunks)
    if out is not cfg:
        out = replace(out, name=cfg.name + "_shrunk")
    return out


def paper_sweep(nchans: int, max_dm: float = 200.0, ndm: int | None = None, nsamp_out: int = 65536) -> SurveyConfig:
    """The paper's own experiment regime (Fig. 4): ``ndm = nchans`` equally spaced
    trials up to ``max_dm`` ("to ensure that we do not sub-sample the data"); left panel sweeps
    nchans at max DM 200, right panel sweeps max DM at nchans = ndm = 2000. The paper gives neither
    band nor sampling time for these runs: c2's LOFAR-like band and tsamp are used."""
    ndm = nchans if ndm is None else ndm
    return SurveyConfig(f"paper_nchan{nchans}_ndm{ndm}_dm{max_dm:g}", nchans, 159.0, -32.0 / nchans, 327.68e-6, nsamp_out,
                        ((0.0, max_dm / max(ndm - 1, 1), ndm),), "u8", 128.0, 16.0, 20.0, 3, SEED0 + 100 + nchans)
