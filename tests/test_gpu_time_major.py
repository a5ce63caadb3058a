"""-m gpu: fused corner turn + low-bit unpack, dedisp_execute_time_major.

The oracle side is oracle.unpack_time_major (oracle/corner_turn_oracle.cpp, pinned in
tests/test_oracle_pins.py) feeding the unchanged de-dispersion oracle; the packing of the test input is
done here with numpy, by neither side.
"""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1111_6399_b200 as P
from paper_1111_6399_b200 import CONFIGS, shrink, synth

from _util import assert_matches_oracle, oracle_rows, oracle_table, spread_rows

pytestmark = pytest.mark.gpu


def pack_time_major(x_cm: np.ndarray, nbits: int, pad_bytes: int = 0, fill: int = 0xA5) -> np.ndarray:
    """channel-major values [c][t] (< 2**nbits) -> time-major rows, first channel in the low bits, rows
    padded with `fill` bytes to a multiple of 16 bytes plus pad_bytes."""
    nchans, nsamp = x_cm.shape
    bits = ((x_cm.T[:, :, None] >> np.arange(nbits)) & 1).astype(np.uint8).reshape(nsamp, nchans * nbits)
    packed = np.packbits(bits, axis=1, bitorder="little")
    row = (packed.shape[1] + 15) // 16 * 16 + pad_bytes
    out = np.full((nsamp, row), fill, dtype=np.uint8)
    out[:, :packed.shape[1]] = packed
    return out


def quantised_case(cfg, nbits, seed=None):
    tab = oracle_table(cfg)
    nsamp_in = cfg.nsamp_out + int(tab.max())
    x, _ = synth.make_input(cfg, tab, nsamp_in, device="cpu", seed=seed)
    return (x.numpy() >> (8 - nbits)).astype(np.uint8), nsamp_in


# Oracle-sized plans that keep the configs' channel width and DM step (so that sub-bands stay >= 16 channels
# wide, which time-major plans need) but cover a short stretch of high DMs and few output samples.
SMALL_TM = {
    "c2tm": replace(CONFIGS["c2"], name="c2_tm_small", nsamp_out=3000, dm_segments=((80.0, 0.05, 150),)),
    "c5tm": replace(CONFIGS["c5"], name="c5_tm_small", nsamp_out=2049, dm_segments=((600.0, 1.0, 100),), nbeams=1, nchunks=1),
    "lowdm": replace(CONFIGS["c2"], name="c2_tm_lowdm", nsamp_out=1777, dm_segments=((0.0, 0.05, 61),)),
}


@pytest.mark.parametrize("nbits", [1, 2, 4, 8])
@pytest.mark.parametrize("name", list(SMALL_TM))
def test_time_major_full_output_vs_oracle(name, nbits):
    cfg = SMALL_TM[name]
    plan = P.Plan.from_config(cfg, time_major=True)
    q, nsamp_in = quantised_case(cfg, nbits)
    raw = pack_time_major(q, nbits, pad_bytes=16 if nbits == 4 else 0)
    cm = oracle.unpack_time_major(raw, cfg.nchans, nbits)            # the oracle's own view of the packed block
    assert np.array_equal(cm, q)
    ref = oracle_rows(cfg, cm)
    for rep in range(2):
        out = plan.execute_time_major(torch.from_numpy(raw).cuda(), nbits, cfg.nsamp_out)
        torch.cuda.synchronize()
        assert_matches_oracle(cfg, out, ref, what=f"{name}/{nbits}-bit time-major")
    # the same plan still takes channel-major input
    out_cm = plan.execute(torch.from_numpy(cm).cuda(), cfg.nsamp_out)
    torch.cuda.synchronize()
    assert torch.equal(out, out_cm)


def test_time_major_errors():
    cfg = SMALL_TM["lowdm"]
    q, nsamp_in = quantised_case(cfg, 8)
    raw = torch.from_numpy(pack_time_major(q, 8)).cuda()
    plain = P.Plan.from_config(cfg)
    with pytest.raises(P.DedispError) as ei:                         # plan not created for time-major input
        plain.execute_time_major(raw, 8, cfg.nsamp_out)
    assert ei.value.code == 4
    plan = P.Plan.from_config(cfg, time_major=True)
    with pytest.raises(P.DedispError) as ei:
        plan.execute_time_major(raw, 3, cfg.nsamp_out)
    assert ei.value.code == 1
    odd = torch.zeros((nsamp_in, raw.shape[1] + 8), dtype=torch.uint8, device="cuda")     # row pitch not a multiple of 16
    with pytest.raises(P.DedispError) as ei:
        plan.execute_time_major(odd, 8, cfg.nsamp_out)
    assert ei.value.code == 1
    with pytest.raises(P.DedispError) as ei:                         # nchans must be a multiple of 16
        P.Plan(100, 1500.0, -1.0, 64e-6, [0.0, 1.0], "u8", time_major=True)
    assert ei.value.code == 1
    with pytest.raises(P.DedispError):
        P.Plan(128, 1500.0, -1.0, 64e-6, [0.0, 1.0], "f32", time_major=True)


@pytest.mark.parametrize("nbits", [8, 2])
def test_time_major_c2_full_size(nbits):
    """configs[1] (LOFAR-like, 496 channels, 2000 DMs, 65536 samples) fed time-major: 48 oracle rows, and the
    whole output against the channel-major path of the same library on the unpacked data."""
    cfg = CONFIGS["c2"]
    plan = P.Plan.from_config(cfg, time_major=True)
    assert plan.kernel == P.KERNEL_SUBBAND
    q, nsamp_in = quantised_case(cfg, nbits)
    raw = pack_time_major(q, nbits)
    rows = spread_rows(cfg.ndm, 48)
    ref = oracle_rows(cfg, oracle.unpack_time_major(raw, cfg.nchans, nbits), rows=rows)
    out = plan.execute_time_major(torch.from_numpy(raw).cuda(), nbits, cfg.nsamp_out)
    torch.cuda.synchronize()
    assert_matches_oracle(cfg, out, ref, rows=rows, what=f"c2 {nbits}-bit time-major")
    out_cm = plan.execute(torch.from_numpy(q).cuda(), cfg.nsamp_out)
    torch.cuda.synchronize()
    assert torch.equal(out, out_cm)
