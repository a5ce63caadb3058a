"""Shared helpers for the parity tests: run the oracle, run the CUDA path, compare.

The oracle (``oracle/``) and the CUDA library never see each other; this module feeds the same
seeded input (``paper_1111_6399_b200.synth``) to both and compares per element.
"""
from __future__ import annotations

import os

import numpy as np
import torch

import oracle
import paper_1111_6399_b200 as P
from paper_1111_6399_b200 import synth

FP_RTOL = 1e-5  # BASELINE.json:north_star: |gpu - oracle| <= 1e-5 * sum_c |term|


def oracle_table(cfg):
    return oracle.shift_table(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, cfg.dm_list())


def make_case(cfg, device="cuda", **kw):
    """(input tensor on device, oracle shift table, nsamp_in)."""
    tab = oracle_table(cfg)
    nsamp_in = cfg.nsamp_out + int(tab.max())
    x, pulses = synth.make_input(cfg, tab, nsamp_in, device=device, **kw)
    return x, tab, pulses


def oracle_rows(cfg, x_host: np.ndarray, rows=None, nsamp_out=None):
    """The oracle on the given DM rows. Many rows of a large plan are split over the host cores: the
    oracle itself stays single-threaded and unchanged, it is just called on disjoint row subsets from
    several Python threads (ctypes releases the GIL for the duration of the call)."""
    nout = cfg.nsamp_out if nsamp_out is None else nsamp_out
    call = lambda r: oracle.dedisperse(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, cfg.dm_list(), x_host, nout, rows=r)
    rows_arr = np.arange(cfg.ndm, dtype=np.int32) if rows is None else np.asarray(rows, dtype=np.int32)
    nthreads = min(os.cpu_count() or 1, 32, rows_arr.size)
    if nthreads < 2 or rows_arr.size * cfg.nchans * nout < 2e9:
        return call(rows)
    from concurrent.futures import ThreadPoolExecutor
    parts = np.array_split(rows_arr, nthreads)
    with ThreadPoolExecutor(nthreads) as ex:
        res = list(ex.map(call, parts))
    if cfg.dtype == "u8":
        return np.concatenate(res, axis=0)
    return np.concatenate([r[0] for r in res], axis=0), np.concatenate([r[1] for r in res], axis=0)


def assert_matches_oracle(cfg, gpu_out: torch.Tensor, ref, rows=None, what=""):
    """Bit-exact for u8/int32; |diff| <= 1e-5 * abs_sum for floating point (north_star)."""
    got = gpu_out if rows is None else gpu_out[torch.as_tensor(np.asarray(rows), device=gpu_out.device, dtype=torch.long)]
    got = got.cpu().numpy()
    if cfg.dtype == "u8":
        assert got.dtype == np.int32
        bad = np.nonzero(got != ref)
        assert bad[0].size == 0, f"{what}: {bad[0].size} int mismatches, first at {bad[0][0]},{bad[1][0]}"
    else:
        out64, asum = ref
        err = np.abs(got.astype(np.float64) - out64)
        tol = FP_RTOL * asum
        bad = np.nonzero(err > tol)
        worst = float((err / np.maximum(asum, 1e-300)).max())
        assert bad[0].size == 0, f"{what}: {bad[0].size} fp mismatches, worst rel {worst:.3e}"


def spread_rows(ndm: int, n: int, extra=()):
    rows = set(np.linspace(0, ndm - 1, min(n, ndm)).round().astype(int).tolist()) | {int(e) for e in extra}
    return np.array(sorted(rows), dtype=np.int32)


def run_gpu(cfg, x: torch.Tensor, kernel=P.KERNEL_AUTO, nsamp_out=None, plan=None):
    plan = plan or P.Plan.from_config(cfg)
    plan.set_kernel(kernel)
    out = plan.execute(x, cfg.nsamp_out if nsamp_out is None else nsamp_out)
    torch.cuda.synchronize()
    return out, plan
