"""Pins for the oracle against what the paper and the mathematics fix — not against itself.

Each test names the mistake it would catch. No GPU, no CUDA library.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1111_6399_b200.configs import CONFIGS, C1, C2, shrink
from paper_1111_6399_b200 import synth

PLAN = (16, 1500.0, -4.0, 64e-6)  # nchans, fch1, foff, tsamp — a small plan used by several pins
DMS = np.arange(0.0, 40.0, 2.5)


def plan_of(cfg):
    return (cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp)


# ---------------------------------------------------------------- shift formula
def test_textbook_delay_ms_ghz_form():
    """Lorimer & Kramer 2005 (cited PAPER.md:66): dt = 4.148808 ms * DM * (f_lo^-2 - f_hi^-2), f in GHz.
    Catches a wrong constant, wrong exponent, swapped frequencies, tsamp multiplied instead of divided."""
    tab = oracle.shift_table(*plan_of(C1), C1.dm_list())
    # hand-worked (SURVEY.md §8(c) pin v): DM 63, 1.437 vs 1.5 GHz -> 10.41 ms -> 162.6 samples -> 163
    dt_ms = 4.148808 * 63.0 * (1.0 / 1.437 ** 2 - 1.0 / 1.5 ** 2)
    assert abs(dt_ms - 10.41) < 0.01
    assert tab[63, 63] == 163 == round(dt_ms * 1e-3 / 64e-6)
    # every entry is within half a sample of the un-rounded GHz/ms form
    f_ghz = (1500.0 - np.arange(64)) / 1e3
    dt_samples = 4.148808e-3 * np.outer(f_ghz ** -2 - 1.5 ** -2, np.arange(64.0)) / 64e-6
    assert np.all(np.abs(tab - dt_samples) <= 0.5 + 1e-9)


def test_round_half_up_not_truncate_or_ceil():
    """floor(x+0.5): catches floor(x), ceil(x). With truncation s(63,63) would be 162."""
    tab = oracle.shift_table(*plan_of(C1), C1.dm_list())
    assert tab[63, 63] == 163      # x = 162.65
    assert tab[63, 1] == 3         # x = 2.58 -> 3, floor would give 2
    assert tab[31, 30] == 37       # x = 37.27 -> 37, ceil would give 38


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4", "c5"])
def test_shift_table_regression_pins(golden, name):
    """tests/golden/shift_pins.txt: maxshift, sum of all entries, three spot values."""
    pins, dm30, nsamp_in = golden
    cfg = CONFIGS[name]
    if name in ("c3", "c4"):
        pytest.importorskip("numpy")
    tab = oracle.shift_table(*plan_of(cfg), cfg.dm_list())
    maxshift, total, s_last_1, s_mid_mid, s_1_last = pins[name]
    assert tab.max() == maxshift == tab[-1, -1]
    assert oracle.max_shift(*plan_of(cfg), cfg.dm_list()) == maxshift
    assert int(tab.sum()) == total
    assert tab[cfg.nchans - 1, 1] == s_last_1
    assert tab[cfg.nchans // 2, cfg.ndm // 2] == s_mid_mid
    assert tab[1, cfg.ndm - 1] == s_1_last
    assert cfg.nsamp_out + maxshift == nsamp_in[name]
    if name == "c1":
        for c, s in dm30.items():
            assert tab[c, 30] == s


def test_table_structure():
    """s(0,d)=0 (reference = channel 0), s(c,0)=0 for DM 0, non-decreasing in c and d, all >= 0.
    Catches a wrong reference frequency or sign (ascending band would give negative shifts)."""
    for cfg in (C1, C2, CONFIGS["c5"]):
        tab = oracle.shift_table(*plan_of(cfg), cfg.dm_list())
        assert np.all(tab[0] == 0) and np.all(tab[:, 0] == 0) and tab.min() == 0
        assert np.all(np.diff(tab, axis=0) >= 0) and np.all(np.diff(tab, axis=1) >= 0)


# ---------------------------------------------------------------- whole oracle
@pytest.mark.parametrize("dtype", [np.uint8, np.float32, np.float16])
def test_dm0_row_is_plain_channel_sum(dtype):
    """north_star check 1: at DM=0 all shifts are 0, out[d0] = sum_c in[c][t] (numpy sum, independent)."""
    rng = np.random.default_rng(1)
    dms = np.array([0.0, 7.0, 0.0])
    ms = oracle.max_shift(*PLAN, dms)
    nout = 300
    if dtype == np.uint8:
        x = rng.integers(0, 256, size=(16, nout + ms), dtype=np.uint8)
        out = oracle.dedisperse(*PLAN, dms, x, nout)
        want = x[:, :nout].astype(np.int64).sum(axis=0)
        assert out.dtype == np.int32
        assert np.array_equal(out[0], want) and np.array_equal(out[2], want)
        assert not np.array_equal(out[1], want)
    else:
        x = rng.standard_normal((16, nout + ms)).astype(dtype)
        out, asum = oracle.dedisperse(*PLAN, dms, x, nout)
        want = x[:, :nout].astype(np.float64).sum(axis=0)
        np.testing.assert_allclose(out[0], want, rtol=0, atol=1e-12)
        np.testing.assert_allclose(asum[0], np.abs(x[:, :nout].astype(np.float64)).sum(axis=0), atol=1e-12)


def test_unit_impulse_response():
    """Pin iv: impulse at (c0,u0) -> out[d][u0 - s(c0,d)] = 1, zero elsewhere.
    Catches the shift applied with the wrong sign (t - s), a transposed table, a wrong channel."""
    tab_expected_dir = 4.148808e3 * DMS * ((1500.0 - 4.0 * 11) ** -2 - 1500.0 ** -2) / 64e-6
    ms = oracle.max_shift(*PLAN, DMS)
    nout = 200
    c0, u0 = 11, 150
    x = np.zeros((16, nout + ms), dtype=np.float32)
    x[c0, u0] = 1.0
    out, _ = oracle.dedisperse(*PLAN, DMS, x, nout)
    for d in range(DMS.size):
        s = int(math.floor(tab_expected_dir[d] + 0.5))
        row = np.zeros(nout)
        if 0 <= u0 - s < nout:
            row[u0 - s] = 1.0
        assert np.array_equal(out[d], row), d
    # lower frequencies arrive later: the impulse moves to EARLIER output time as DM grows
    peaks = [int(np.argmax(out[d])) for d in range(DMS.size) if out[d].max() > 0]
    assert peaks == sorted(peaks, reverse=True) and peaks[0] == u0


@pytest.mark.parametrize("cfg", [C1, shrink(C2, nchans=62, nsamp_out=2048, ndm_stride=40)])
def test_noise_free_pulse_recovered(cfg):
    """north_star check 2 / PAPER.md:52 (Fig. 3): a pulse laid along a trial curve is recovered at the
    injected DM and time with peak = nchans*amp; every channel's pulse lands once per row."""
    dms = cfg.dm_list()
    tab = oracle.shift_table(*plan_of(cfg), dms)
    nin = cfg.nsamp_out + int(tab.max())
    d_inj, t0 = (30, 1000) if cfg is C1 else (cfg.ndm - 3, 777)
    x, _ = synth.make_input(cfg, tab, nin, noise=False, pulses=[(d_inj, t0)])
    x = x.numpy()
    res = oracle.dedisperse(*plan_of(cfg), dms, x, cfg.nsamp_out)
    out = res if cfg.dtype == "u8" else res[0]
    bg = cfg.nchans * cfg.noise_mean
    excess = out.astype(np.float64) - bg
    assert excess[d_inj, t0] == cfg.nchans * cfg.pulse_amp
    if cfg is C1:
        assert excess[d_inj, t0] == 320.0      # 64 * 5
    d_max, t_max = np.unravel_index(np.argmax(excess), excess.shape)
    assert (d_max, t_max) == (d_inj, t0)
    assert np.sum(excess == excess.max()) == 1
    # invariant: each channel's pulse sample lands exactly once in every row whose curve stays in range
    for d in range(cfg.ndm):
        lo = t0 + tab[:, d_inj] - tab[:, d]
        if np.all((lo >= 0) & (lo < cfg.nsamp_out)):
            assert excess[d].sum() == cfg.nchans * cfg.pulse_amp


def test_tiny_brute_force_per_output():
    """north_star check 3: per-(d,t) recomputation, delay recomputed inline per term, other loop order."""
    nch, fch1, foff, tsamp = 7, 400.0, -3.0, 1e-3
    dms = np.array([0.0, 1.5, 3.0, 9.0, 9.0, 20.0])
    nout = 29
    ms = oracle.max_shift(nch, fch1, foff, tsamp, dms)
    rng = np.random.default_rng(5)
    x8 = rng.integers(0, 256, size=(nch, nout + ms), dtype=np.uint8)
    xf = rng.standard_normal((nch, nout + ms)).astype(np.float32)
    xh = (3.0 * rng.standard_normal((nch, nout + ms))).astype(np.float16)   # oracle_dedisperse_f16 at non-zero shift
    o8 = oracle.dedisperse(nch, fch1, foff, tsamp, dms, x8, nout)
    of, oa = oracle.dedisperse(nch, fch1, foff, tsamp, dms, xf, nout)
    oh, oha = oracle.dedisperse(nch, fch1, foff, tsamp, dms, xh, nout)
    for t in range(nout):
        for d in range(dms.size):
            tot8, totf, tota, toth, totha = 0, 0.0, 0.0, 0.0, 0.0
            for c in reversed(range(nch)):
                f = fch1 + c * foff
                s = math.floor(4.148808e3 * dms[d] * (f ** -2 - fch1 ** -2) / tsamp + 0.5)
                tot8 += int(x8[c, t + s])
                totf += float(xf[c, t + s])
                tota += abs(float(xf[c, t + s]))
                toth += float(xh[c, t + s])          # numpy's own half -> double conversion
                totha += abs(float(xh[c, t + s]))
            assert o8[d, t] == tot8
            assert abs(of[d, t] - totf) < 1e-12 and abs(oa[d, t] - tota) < 1e-12
            assert abs(oh[d, t] - toth) < 1e-12 and abs(oha[d, t] - totha) < 1e-12
    assert ms > 20  # the plan actually shifts


def test_row_subset_and_identity_and_invariants():
    """nchans=1 -> identity; constant input -> nchans*v; linearity on ints; time translation;
    rows= subset equals the same rows of the full run."""
    rng = np.random.default_rng(9)
    ms = oracle.max_shift(*PLAN, DMS)
    nout = 128
    a = rng.integers(0, 100, size=(16, nout + ms + 5), dtype=np.uint8)
    b = rng.integers(0, 100, size=(16, nout + ms + 5), dtype=np.uint8)
    full = oracle.dedisperse(*PLAN, DMS, a, nout)
    sub = oracle.dedisperse(*PLAN, DMS, a, nout, rows=[3, 15, 0])
    assert np.array_equal(sub, full[[3, 15, 0]])
    assert np.array_equal(oracle.dedisperse(*PLAN, DMS, (a + b).astype(np.uint8), nout),
                          full + oracle.dedisperse(*PLAN, DMS, b, nout))
    shifted = oracle.dedisperse(*PLAN, DMS, np.ascontiguousarray(a[:, 5:]), nout - 0)
    assert np.array_equal(shifted[:, : nout - 5], full[:, 5:])
    const = np.full((16, nout + ms), 3, dtype=np.uint8)
    assert np.all(oracle.dedisperse(*PLAN, DMS, const, nout) == 48)
    one = rng.standard_normal((1, nout)).astype(np.float32)
    o, _ = oracle.dedisperse(1, 1500.0, -4.0, 64e-6, DMS, one, nout)
    assert np.array_equal(o, np.broadcast_to(one.astype(np.float64), (DMS.size, nout)))


def test_input_too_short_is_refused():
    x = np.zeros((16, 100), dtype=np.uint8)
    with pytest.raises(ValueError):
        oracle.dedisperse(*PLAN, DMS, x, 100)   # needs 100 + maxshift columns


def test_half_conversion_exact_all_finite_patterns():
    """The oracle's own binary16 decoder vs numpy's, on every finite bit pattern (nchans=1, DM=0)."""
    bits = np.arange(65536, dtype=np.uint16)
    h = bits.view(np.float16)
    h = h[np.isfinite(h)].reshape(1, -1).copy()
    out, _ = oracle.dedisperse(1, 1500.0, -1.0, 64e-6, np.array([0.0]), h, h.shape[1])
    assert np.array_equal(out[0], h[0].astype(np.float64))


def test_float_sequential_diagnostic_inside_tolerance():
    """fp path sanity: a float32 sequential sum differs from the double result by << 1e-5 * sum|terms|."""
    rng = np.random.default_rng(3)
    cfg = shrink(C1, nsamp_out=512)
    dms = cfg.dm_list()
    ms = oracle.max_shift(*plan_of(cfg), dms)
    x = rng.standard_normal((cfg.nchans, 512 + ms)).astype(np.float32)
    o, a = oracle.dedisperse(*plan_of(cfg), dms, x, 512)
    s = oracle.dedisperse(*plan_of(cfg), dms, x, 512, seq_f32=True)
    assert np.max(np.abs(s - o) / a) < 1e-6


# ---- corner turn + unpack in front of the hot path (oracle/corner_turn_oracle.cpp)
def test_unpack_time_major_hand_packed_bytes():
    """Hand-packed rows, reading R15: first channel in the least significant bits."""
    # 4-bit, 4 channels, 2 time samples: t0 = (1, 2, 3, 4) -> bytes 0x21 0x43; t1 = (15, 0, 9, 6) -> 0x0F 0x69
    raw = np.array([[0x21, 0x43], [0x0F, 0x69]], dtype=np.uint8)
    assert oracle.unpack_time_major(raw, 4, 4).tolist() == [[1, 15], [2, 0], [3, 9], [4, 6]]
    # 2-bit, 4 channels per byte: (3, 0, 1, 2) -> 0b10_01_00_11 = 0x93
    assert oracle.unpack_time_major(np.array([[0x93]], dtype=np.uint8), 4, 2).tolist() == [[3], [0], [1], [2]]
    # 1-bit, 8 channels per byte: channels 0, 3, 7 set -> 0b1000_1001 = 0x89; a pad byte is ignored
    assert oracle.unpack_time_major(np.array([[0x89, 0xFF]], dtype=np.uint8), 8, 1).ravel().tolist() == [1, 0, 0, 1, 0, 0, 0, 1]
    # 8-bit is a plain transpose
    raw = np.arange(12, dtype=np.uint8).reshape(3, 4)
    assert np.array_equal(oracle.unpack_time_major(raw, 4, 8), raw.T)


@pytest.mark.parametrize("nbits", [1, 2, 4, 8])
def test_unpack_time_major_vs_numpy_and_round_trip(nbits):
    """Independent statement with numpy: unpackbits(bitorder='little') regrouped nbits at a time; and a
    pack -> unpack round trip from known channel-major values, with padded rows."""
    rng = np.random.default_rng(40 + nbits)
    nchans, nsamp, pad = 48, 37, 5
    row_bytes = nchans * nbits // 8 + pad
    raw = rng.integers(0, 256, size=(nsamp, row_bytes), dtype=np.uint8)
    bits = np.unpackbits(raw[:, : nchans * nbits // 8], axis=1, bitorder="little").reshape(nsamp, nchans, nbits)
    want = (bits * (1 << np.arange(nbits))).sum(axis=2).astype(np.uint8).T
    assert np.array_equal(oracle.unpack_time_major(raw, nchans, nbits), want)
    vals = rng.integers(0, 1 << nbits, size=(nchans, nsamp), dtype=np.uint8)          # [c][t]
    vbits = ((vals.T[:, :, None] >> np.arange(nbits)) & 1).astype(np.uint8).reshape(nsamp, nchans * nbits)
    packed = np.packbits(vbits, axis=1, bitorder="little")
    packed = np.concatenate([packed, np.full((nsamp, pad), 0xAA, dtype=np.uint8)], axis=1)
    assert np.array_equal(oracle.unpack_time_major(np.ascontiguousarray(packed), nchans, nbits), vals)


# ---- detection behind the hot path (oracle/detect_oracle.cpp, reading R16)
def test_detect_closed_forms():
    # alternating +-1: mu = 0, var = 1; width 1: snr = x; width 2: every window sums to 0
    n = 64
    x = np.where(np.arange(n) % 2 == 0, 1, -1).astype(np.int32)[None, :]
    c, cnt = oracle.detect(x, 2, 0.5)
    assert cnt == n // 2 and set(c["width"]) == {1} and np.all(c["t"] % 2 == 0) and np.allclose(c["snr"], 1.0)
    # a lone pulse of width 4 and height a on a zero row of length n: mu = 4a/n, var = 4a^2/n - mu^2;
    # the matched window (w = 4 at the pulse start) has snr = (4a - 4 mu) / (sd * 2), the largest of all
    n, a, t0 = 1000, 7, 123
    x = np.zeros((1, n), dtype=np.int32)
    x[0, t0:t0 + 4] = a
    mu = 4 * a / n
    sd = math.sqrt(4 * a * a / n - mu * mu)
    c, cnt = oracle.detect(x, 5, 0.0)
    best = c[np.argmax(c["snr"])]
    assert (best["width"], best["t"]) == (4, t0)
    assert best["snr"] == ((4 * a - 4 * mu) * (1.0 / (sd * math.sqrt(4.0))))
    w8 = c[(c["width"] == 8) & (c["t"] == t0 - 2)][0]          # a width-8 window around the pulse sees the same sum
    assert abs(w8["snr"] - (4 * a - 8 * mu) / (sd * math.sqrt(8.0))) < 1e-12
    # constant rows have no variance and yield nothing; float rows likewise
    assert oracle.detect(np.full((2, 50), 5, dtype=np.int32), 3, -1e9)[1] == 0
    assert oracle.detect(np.full((2, 50), 0.25, dtype=np.float32), 3, -1e9)[1] == 0


@pytest.mark.parametrize("dtype", [np.int32, np.float32])
def test_detect_vs_numpy_brute_force(dtype):
    """Every (row, w, t) recomputed with direct window sums (no doubling) in numpy; integer rows must agree
    exactly, float rows to 1e-6 (fp32 window sums in another order)."""
    rng = np.random.default_rng(77)
    nrows, n, nwidths, thr = 3, 257, 4, 1.5
    x = rng.integers(-50, 200, size=(nrows, n)).astype(dtype) if dtype == np.int32 else rng.standard_normal((nrows, n)).astype(dtype)
    c, cnt = oracle.detect(x, nwidths, thr)
    assert cnt == len(c) > 0
    got = {(int(r["dm_index"]), int(r["width"]), int(r["t"])): float(r["snr"]) for r in c}
    want = {}
    for r in range(nrows):
        row = x[r].astype(np.float64)
        mu, var = row.mean(), (row * row).mean() - row.mean() ** 2
        for k in range(nwidths):
            w = 1 << k
            for t in range(n - w + 1):
                snr = (row[t:t + w].sum() - w * mu) / (math.sqrt(var) * math.sqrt(w))
                if snr >= thr + 1e-6 or (snr >= thr - 1e-6 and (r, w, t) in got):
                    want[(r, w, t)] = snr
    assert set(got) == set(want)
    tol = 0.0 if dtype == np.int32 else 1e-6
    assert max(abs(got[k] - want[k]) for k in got) <= max(tol, 1e-12)
