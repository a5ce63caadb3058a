"""-m gpu: dedisp_detect_static, the entry point that allocates nothing (its scratch is a fixed static __device__
array inside the library), against the existing dedisp_detect path with a caller-provided workspace.

Collected last on purpose (the suite runs with pytest -x). Two calls in a row on DIFFERENT blocks: the array keeps
the previous call's row sums, so a missing clear, or a kernel handed the host-side stand-in of the array instead
of its device address, shows up in the second call at the latest. Integer blocks must agree bit for bit (exact
integer statistics); float blocks within the 1e-9 the detection tests use (atomic double sums in another order).
"""
import numpy as np
import pytest
import torch

import paper_1111_6399_b200 as P
from paper_1111_6399_b200 import api

pytestmark = pytest.mark.gpu


def _sorted(c):
    return np.sort(c, order=["dm_index", "width", "t"])


def _int_block(nrows, n, seed, base):
    g = torch.Generator(device="cuda").manual_seed(seed)
    x = torch.randn((nrows, n), generator=g, device="cuda").mul_(40.0).add_(base).round_().to(torch.int32)
    x[1, 100:108] += 90
    x[nrows - 1, n - 3:] += 400
    return x


def test_detect_static_matches_detect_on_two_calls_in_a_row():
    cands = torch.empty((1 << 16) * P.CAND_DTYPE.itemsize, dtype=torch.uint8, device="cuda")    # the caller's outputs, reused
    count = torch.empty(1, dtype=torch.int64, device="cuda")
    cases = [(_int_block(37, 9000, 1, 5000.0), 6, 3.5),      # second call: fewer rows, other level -> stale sums would show
             (_int_block(9, 20011, 2, -300.0), 8, 3.0),
             (_int_block(37, 9000, 1, 5000.0), 6, 3.5)]      # and the first block again
    for x, nwidths, thr in cases:
        ref, rtotal = P.detect(x, nwidths, thr, max_cands=1 << 16)
        got, total = P.detect_static(x, nwidths, thr, max_cands=1 << 16, cands=cands, count=count)
        assert total == rtotal == len(got) == len(ref) and total > 0
        g, r = _sorted(got), _sorted(ref)
        for k in ("dm_index", "width", "t", "snr"):
            assert np.array_equal(g[k], r[k]), k             # bit-identical, S/N included


def test_detect_static_float_rows_twice():
    gen = torch.Generator(device="cuda").manual_seed(7)
    thr = 4.0
    for rep in range(2):
        x = torch.randn((6 + rep, 30000), generator=gen, device="cuda")
        x[2, 777:793] += 1.5
        ref, _ = P.detect(x, 6, thr)
        got, _ = P.detect_static(x, 6, thr)
        gk = {(int(c["dm_index"]), int(c["width"]), int(c["t"])): float(c["snr"]) for c in got}
        rk = {(int(c["dm_index"]), int(c["width"]), int(c["t"])): float(c["snr"]) for c in ref}
        for k in set(gk) ^ set(rk):                          # only borderline candidates may differ
            assert abs((gk.get(k) or rk.get(k)) - thr) < 1e-9
        common = set(gk) & set(rk)
        assert len(common) > 5 and max(abs(gk[k] - rk[k]) for k in common) < 1e-9


def test_detect_static_limits():
    n = 64
    big = torch.zeros((api.DETECT_STATIC_MAX_NDM + 1, n), dtype=torch.int32, device="cuda")
    with pytest.raises(P.DedispError) as ei:                 # one row more than the static scratch holds
        P.detect_static(big, 2, 3.0, max_cands=16)
    assert ei.value.code == api.ETOOLARGE and "DEDISP_DETECT_STATIC_MAX_NDM" in str(ei.value)
    full = torch.arange(api.DETECT_STATIC_MAX_NDM * n, device="cuda", dtype=torch.int32).reshape(-1, n) % 7
    ref, rtotal = P.detect(full, 2, 1.0, max_cands=1 << 20)
    got, total = P.detect_static(full, 2, 1.0, max_cands=1 << 20)      # exactly the maximum: every row of the array in use
    assert total == rtotal > 0 and np.array_equal(_sorted(got), _sorted(ref))
    count = torch.empty(1, dtype=torch.int64, device="cuda")
    rc = api.lib().dedisp_detect_static(full.data_ptr(), 0, 4, n, n, 2, 1.0, None, 0, count.data_ptr() + 4, None)
    assert rc == api.EINVAL                                   # misaligned d_count
