"""-m gpu: streaming driver (SURVEY.md §8(a) row a-5, §8(b) "Streaming semantics").

Output block k of the driver must equal one-shot de-dispersion of the concatenated stream delayed
by maxshift (zero history before the first chunk) — checked against the ORACLE run on the
zero-prefixed concatenated stream, per beam, bit-exact (u8) / within tolerance (f32).
"""
from dataclasses import replace

import numpy as np
import pytest
import torch

import paper_1111_6399_b200 as P
from paper_1111_6399_b200 import CONFIGS, shrink, synth

from _util import assert_matches_oracle, oracle_rows, oracle_table

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dtype_cfg,nbuf", [("c5", 2), ("c5", 3), ("c3", 2)])
def test_chunked_equals_oneshot_oracle(dtype_cfg, nbuf):
    base = CONFIGS[dtype_cfg]
    nbeams, nchunks, chunk = 3, 5, 1536
    cfg = shrink(base, nchans=96, nsamp_out=chunk, nbeams=nbeams, nchunks=nchunks)
    cfg = replace(cfg, dm_segments=((0.0, 312.0 / 39 if base.dtype == "u8" else 2.0, 40),))  # maxshift ~ 3.4 chunks
    tab = oracle_table(cfg)
    maxshift = int(tab.max())
    assert maxshift > chunk // 2  # the carry must matter (and here even spans chunks when > chunk)
    plan = P.Plan.from_config(cfg)
    assert plan.max_shift == maxshift
    total = nchunks * chunk
    # whole stream per beam in global time, pulses cross chunk boundaries
    beams = []
    for b in range(nbeams):
        x, _ = synth.make_input(cfg, tab, total, device="cpu", seed=cfg.seed * 1000003 + b * 101,
                                pulses=[(cfg.ndm - 1, chunk - 7), (cfg.ndm // 2, 2 * chunk + 11)])
        beams.append(x)
    stream_all = torch.stack(beams)                                   # [beam][chan][total]
    st = P.Stream(plan, nbeams, chunk, nbuf)
    got = []
    for k in range(nchunks):
        h = stream_all[:, :, k * chunk:(k + 1) * chunk].contiguous().pin_memory()
        out_ptr, _ = st.push(h)
        st.sync()                                                     # block k valid; buffer reused later
        got.append(st.out_view(out_ptr).clone())
    st.close()
    got = torch.cat(got, dim=2)                                       # [beam][dm][total], delayed by maxshift
    for b in range(nbeams):
        padded = np.concatenate([np.zeros((cfg.nchans, maxshift), dtype=cfg.np_dtype), beams[b].numpy()], axis=1)
        ref = oracle_rows(cfg, np.ascontiguousarray(padded), nsamp_out=total)
        assert_matches_oracle(cfg, got[b], ref, what=f"stream beam {b}")


def test_stream_overlapped_pushes_match_synced():
    """Pushing without intermediate syncs (copy k+1 overlapping compute k) gives the same blocks."""
    cfg = shrink(CONFIGS["c5"], nchans=64, nsamp_out=4096, ndm_stride=16, nbeams=4, nchunks=6)
    plan = P.Plan.from_config(cfg)
    tab = plan.shifts()
    chunks = []
    for k in range(cfg.nchunks):
        xs = [synth.make_input(cfg, tab, cfg.nsamp_out, device="cpu", seed=9000 + 10 * k + b)[0] for b in range(cfg.nbeams)]
        chunks.append(torch.stack(xs).pin_memory())

    st = P.Stream(plan, cfg.nbeams, cfg.nsamp_out, 2)
    ref = []
    for h in chunks:
        out_ptr, _ = st.push(h)
        st.sync()
        ref.append(st.out_view(out_ptr).clone())
    st.close()
    a = torch.stack(ref)
    st = P.Stream(plan, cfg.nbeams, cfg.nsamp_out, 3)
    ptrs = [st.push(h)[0] for h in chunks[:3]]                        # three pushes in flight, no sync between
    st.sync()
    for k in range(3):
        assert torch.equal(st.out_view(ptrs[k]), a[k])
    st.close()


def test_c5_full_shape_first_chunks_through_the_stream():
    """configs[4] at its real shape through dedisp_stream_push (SURVEY.md §8(d) "parity coverage at
    scale"): 32 beams x 1024 channels x 32768-sample chunks, the first 3 chunks, maxshift carried
    between them; 2 beams x 64 DM rows of every output block against the oracle run on the
    zero-prefixed concatenated stream."""
    cfg = CONFIGS["c5"]
    nchunks, chunk = 3, cfg.nsamp_out
    plan = P.Plan.from_config(cfg)
    tab = oracle_table(cfg)
    maxshift = int(tab.max())
    assert plan.max_shift == maxshift
    total = nchunks * chunk
    beams_checked = (3, 29)
    host = torch.empty((cfg.nbeams, cfg.nchans, total), dtype=torch.uint8).pin_memory()
    for b in range(cfg.nbeams):
        x, _ = synth.make_input(cfg, tab, total, device="cuda", seed=cfg.seed * 1000003 + b * 101,
                                pulses=[(cfg.ndm - 1, chunk - 5), (cfg.ndm // 3, chunk + 77)])
        host[b].copy_(x)
    st = P.Stream(plan, cfg.nbeams, chunk, 2)
    rows = np.linspace(0, cfg.ndm - 1, 64).round().astype(np.int32)
    ridx = torch.as_tensor(rows, device="cuda", dtype=torch.long)
    got = {b: [] for b in beams_checked}
    for k in range(nchunks):
        h = host[:, :, k * chunk:(k + 1) * chunk].contiguous().pin_memory()
        out_ptr, _ = st.push(h)
        st.sync()
        view = st.out_view(out_ptr)
        for b in beams_checked:
            got[b].append(view[b][ridx].clone())
    st.close()
    for b in beams_checked:
        padded = np.concatenate([np.zeros((cfg.nchans, maxshift), dtype=np.uint8), host[b].numpy()], axis=1)
        ref = oracle_rows(cfg, np.ascontiguousarray(padded), rows=rows, nsamp_out=total)
        assert_matches_oracle(cfg, torch.cat(got[b], dim=1), ref, what=f"c5 stream beam {b}")
