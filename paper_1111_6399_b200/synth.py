"""Seeded synthetic filterbank input — the one module that serves both the oracle
tests and the CUDA path. It stands in for the paper's sigproc-simulated data
(noise plus a dispersed pulse), which is not available.

No method arithmetic lives here: the integer delays used to lay a pulse along a
trial dispersion curve are passed in as ``shifts[nchans][ndm]`` by the caller
(tests pass the oracle's table; bench.py passes ``Plan.shifts()``).

Recipe:
  f32 : N(mean, sigma) + amp on the pulse samples
  f16 : half( N(mean, sigma) + amp*[pulse] )
  u8  : clip( round(N(mean, sigma)) + amp*[pulse], 0, 255 )   (add, then clip)
A pulse (d_inj, t0) touches exactly one sample per channel: in[c][t0 + s(c, d_inj)].
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np
import torch

from .configs import SurveyConfig

_TORCH_DTYPE = {"u8": torch.uint8, "f16": torch.float16, "f32": torch.float32}


def pulse_positions(cfg: SurveyConfig, seed: int | None = None, t_span: int | None = None) -> List[Tuple[int, int]]:
    """Seeded (d_inj, t0) pairs: d_inj in [ndm/8, ndm), t0 in [0, t_span)."""
    if cfg.fixed_pulses:
        return [tuple(p) for p in cfg.fixed_pulses]
    rng = np.random.default_rng(cfg.seed if seed is None else seed)
    t_span = cfg.nsamp_out if t_span is None else t_span
    lo = min(cfg.ndm // 8, cfg.ndm - 1)
    return [(int(rng.integers(lo, cfg.ndm)), int(rng.integers(0, t_span))) for _ in range(cfg.npulses)]


def make_input(cfg: SurveyConfig, shifts, nsamp_in: int, device="cpu", seed: int | None = None,
               pulses: Sequence[Tuple[int, int]] | None = None, noise: bool = True,
               t_origin: int = 0, chan_block: int = 256) -> Tuple[torch.Tensor, List[Tuple[int, int]]]:
    """One beam of ``in[nchans][nsamp_in]`` on ``device``; returns (tensor, pulses).

    ``shifts``: integer array-like ``[nchans][ndm]``. ``t_origin``: global time of
    column 0 (streaming: pulses are placed in global stream time and only the
    samples that fall inside this block are written). ``noise=False`` gives the
    noise-free variant (background = noise_mean) used by the peak pins.
    """
    seed = cfg.seed if seed is None else seed
    pulses = pulse_positions(cfg, seed) if pulses is None else list(pulses)
    shifts_t = torch.as_tensor(np.asarray(shifts), dtype=torch.int64, device=device)
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    out = torch.empty((cfg.nchans, nsamp_in), dtype=_TORCH_DTYPE[cfg.dtype], device=device)
    for c0 in range(0, cfg.nchans, chan_block):
        c1 = min(cfg.nchans, c0 + chan_block)
        if noise:
            blk = torch.randn((c1 - c0, nsamp_in), generator=gen, device=device, dtype=torch.float32)
            blk.mul_(cfg.noise_sigma).add_(cfg.noise_mean)
        else:
            blk = torch.full((c1 - c0, nsamp_in), float(cfg.noise_mean), device=device, dtype=torch.float32)
        if cfg.dtype == "u8":
            blk.round_()
        rows = torch.arange(c0, c1, device=device)
        for d_inj, t0 in pulses:
            cols = t0 + shifts_t[c0:c1, d_inj] - t_origin
            ok = (cols >= 0) & (cols < nsamp_in)
            blk[(rows - c0)[ok], cols[ok]] += cfg.pulse_amp
        if cfg.dtype == "u8":
            blk.clamp_(0, 255)
        out[c0:c1] = blk.to(out.dtype)
    return out, pulses
