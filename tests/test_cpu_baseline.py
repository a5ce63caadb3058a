"""-m "not gpu": the stronger CPU baseline of bench.py (baseline_cpu/) against the oracle.
It is a reporting baseline only; this test keeps its numbers honest (bit-exact on u8, 1e-5*sum|terms| on f32)."""
import numpy as np

import baseline_cpu
import oracle
from paper_1111_6399_b200 import CONFIGS, shrink, synth


def _case(cfg):
    dm = cfg.dm_list()
    tab = oracle.shift_table(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm)
    x, _ = synth.make_input(cfg, tab, cfg.nsamp_out + int(tab.max()), device="cpu")
    return dm, x.numpy()


def test_vectorised_cpu_baseline_matches_oracle_u8():
    cfg = shrink(CONFIGS["c2"], nchans=62, nsamp_out=9000, ndm_stride=50)      # several 8192-sample tiles, ragged tail
    dm, x = _case(cfg)
    got = baseline_cpu.dedisperse(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm, x, cfg.nsamp_out, nthreads=3)
    assert np.array_equal(got, oracle.dedisperse(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm, x, cfg.nsamp_out))


def test_vectorised_cpu_baseline_matches_oracle_f32():
    cfg = CONFIGS["c1"]
    dm, x = _case(cfg)
    got = baseline_cpu.dedisperse(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm, x, cfg.nsamp_out)
    ref, asum = oracle.dedisperse(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm, x, cfg.nsamp_out)
    assert (np.abs(got - ref) <= 1e-5 * asum).all()
