"""-m gpu: detection behind the hot path, dedisp_detect vs oracle/detect_oracle.cpp.

Integer blocks: the candidate set and every S/N must be bit-identical (exact integer statistics, explicitly
rounded double operations on both sides). Float blocks: the row sums are taken in another order, so S/N agrees
to 1e-9 and only candidates within 1e-9 of the threshold may differ. The GPU lists candidates in any order.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_1111_6399_b200 as P
from paper_1111_6399_b200 import CONFIGS

from _util import make_case, run_gpu

pytestmark = pytest.mark.gpu


def _sorted(c):
    return np.sort(c, order=["dm_index", "width", "t"])


def _int_block(nrows, n, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    x = torch.randn((nrows, n), generator=g, device="cuda").mul_(40.0).add_(5000.0).round_().to(torch.int32)
    x[1, 100:108] += 90                      # a width-8 pulse
    x[nrows - 1, n - 3:] += 400              # a pulse cut by the end of the row
    return x


@pytest.mark.parametrize("nrows,n,nwidths,thr", [(5, 10000, 6, 3.5), (3, 2048, 8, 3.0), (4, 2049 + 31, 6, 2.5), (2, 7, 4, -1.0), (70, 5000, 1, 3.0)])
def test_detect_int_rows_bit_exact(nrows, n, nwidths, thr):
    x = _int_block(nrows, n, seed=nrows * 1000 + n) if n > 200 else torch.arange(nrows * n, device="cuda", dtype=torch.int32).reshape(nrows, n) % 5
    got, total = P.detect(x, nwidths, thr)
    ref, rtotal = oracle.detect(x.cpu().numpy(), nwidths, thr)
    assert total == rtotal == len(got) == len(ref) and total > 0
    g, r = _sorted(got), _sorted(ref)
    assert np.array_equal(g["dm_index"], r["dm_index"]) and np.array_equal(g["width"], r["width"]) and np.array_equal(g["t"], r["t"])
    assert np.array_equal(g["snr"], r["snr"])                     # bit-identical doubles


def test_detect_constant_rows_and_capacity():
    x = torch.full((3, 4000), 7, dtype=torch.int32, device="cuda")
    x[1] = _int_block(2, 4000, 5)[0]
    got, total = P.detect(x, 4, 2.0, max_cands=10)               # far more than 10 candidates: counted, 10 stored
    ref, rtotal = oracle.detect(x.cpu().numpy(), 4, 2.0)
    assert total == rtotal > 10 and len(got) == 10
    assert set(got["dm_index"]) == {1}                            # the constant rows (no variance) yield nothing
    keys = {(int(c["dm_index"]), int(c["width"]), int(c["t"])): float(c["snr"]) for c in ref}
    assert all(keys[(int(c["dm_index"]), int(c["width"]), int(c["t"]))] == float(c["snr"]) for c in got)


def test_detect_float_rows_within_tolerance():
    g = torch.Generator(device="cuda").manual_seed(99)
    x = torch.randn((6, 30000), generator=g, device="cuda")
    x[2, 777:793] += 1.5
    thr = 4.0
    got, total = P.detect(x, 6, thr)
    ref, rtotal = oracle.detect(x.cpu().numpy(), 6, thr)
    gk = {(int(c["dm_index"]), int(c["width"]), int(c["t"])): float(c["snr"]) for c in got}
    rk = {(int(c["dm_index"]), int(c["width"]), int(c["t"])): float(c["snr"]) for c in ref}
    for k in set(gk) ^ set(rk):                                   # only borderline candidates may differ
        assert abs((gk.get(k) or rk.get(k)) - thr) < 1e-9
    common = set(gk) & set(rk)
    assert len(common) > 5 and max(abs(gk[k] - rk[k]) for k in common) < 1e-9
    best = max(gk, key=gk.get)
    assert best[0] == 2 and best[1] == 16 and 777 - 2 <= best[2] <= 777 + 2


def test_dedisperse_then_detect_finds_the_injected_pulse():
    """c1 (Fig. 3: the injected pulse is recovered at its DM and time), now without the block
    leaving the GPU: the strongest candidate of the de-dispersed block is the injected (DM 30, t 1000)."""
    cfg = CONFIGS["c1"]
    x, tab, pulses = make_case(cfg)
    out, _ = run_gpu(cfg, x)
    got, total = P.detect(out, 4, 6.0)
    assert total > 0
    best = got[np.argmax(got["snr"])]
    assert (int(best["dm_index"]), int(best["t"]), int(best["width"])) == (pulses[0][0], pulses[0][1], 1)
    ref, rtotal = oracle.detect(out.cpu().numpy(), 4, 6.0)
    assert abs(total - rtotal) <= 2
