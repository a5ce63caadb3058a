"""-m gpu: CUDA path vs oracle, element by element, through the C ABI (include/dedisp.h).

Chain of trust: oracle => every kernel on oracle-sized cases (full outputs) and on
row subsets of the full-size configs; optimised kernels == NAIVE kernel on the FULL output of every
full-size config (NAIVE is itself oracle-checked; it is a cross-check, never the oracle).
"""
import numpy as np
import pytest
import torch

import paper_1111_6399_b200 as P
from paper_1111_6399_b200 import CONFIGS, paper_sweep, shrink
from paper_1111_6399_b200.configs import SurveyConfig

from _util import assert_matches_oracle, make_case, oracle_table, oracle_rows, run_gpu, spread_rows

pytestmark = pytest.mark.gpu

KERNELS = [P.KERNEL_NAIVE, P.KERNEL_TILED, P.KERNEL_SUBBAND]
KNAME = {P.KERNEL_NAIVE: "naive", P.KERNEL_TILED: "tiled", P.KERNEL_SUBBAND: "subband"}


def _plan_with(cfg, kernel):
    plan = P.Plan.from_config(cfg)
    try:
        plan.set_kernel(kernel)
    except P.DedispError as e:
        assert e.code == 4
        pytest.skip(f"{KNAME[kernel]} kernel not admitted by plan {cfg.name}")
    return plan


# ---- oracle-sized cases: full outputs, several tiles plus ragged tails in both d and t
SMALL = {
    "c1": CONFIGS["c1"],
    "c2s": shrink(CONFIGS["c2"], nsamp_out=5000, ndm_stride=9),          # 223 DMs, u8, shifts to 28k
    "c3s": shrink(CONFIGS["c3"], nchans=300, nsamp_out=4500, ndm_stride=31),
    "c4s": shrink(CONFIGS["c4"], nchans=257, nsamp_out=3100, ndm_stride=29),
    "c5s": shrink(CONFIGS["c5"], nchans=128, nsamp_out=2049, ndm_stride=5),
    "paper": paper_sweep(250, 200.0, nsamp_out=3000),                     # PAPER.md:56-58 regime, ndm = nchans
    "fine": SurveyConfig("fine_dm_u8", 200, 159.0, -32.0 / 200.0, 327.68e-6, 3000, ((0.0, 0.01, 333),),
                         "u8", 128.0, 16.0, 20.0, 2, 77),                  # paper regime: adjacent-DM delta <= 1
}


@pytest.mark.parametrize("kernel", KERNELS, ids=[KNAME[k] for k in KERNELS])
@pytest.mark.parametrize("name", list(SMALL))
def test_small_full_output_vs_oracle(name, kernel):
    cfg = SMALL[name]
    plan = _plan_with(cfg, kernel)
    x, tab, _ = make_case(cfg)
    assert plan.max_shift == int(tab.max())
    out, _ = run_gpu(cfg, x, kernel, plan=plan)
    ref = oracle_rows(cfg, x.cpu().numpy())
    assert_matches_oracle(cfg, out, ref, what=f"{name}/{KNAME[kernel]}")


def test_c1_pulse_recovered():
    """PAPER.md:52 (Fig. 3): the injected pulse is recovered at its DM and time."""
    cfg = CONFIGS["c1"]
    x, tab, pulses = make_case(cfg, noise=False)
    out, _ = run_gpu(cfg, x)
    d_inj, t0 = pulses[0]
    assert out[d_inj, t0].item() == cfg.nchans * cfg.pulse_amp
    assert int(out.argmax()) == d_inj * cfg.nsamp_out + t0


# ---- edge shapes
EDGE = [
    dict(nchans=1, ndm_seg=((0.0, 1.0, 5),), nsamp_out=100),
    dict(nchans=7, ndm_seg=((3.0, 1.0, 1),), nsamp_out=1),
    dict(nchans=33, ndm_seg=((0.0, 0.0, 9),), nsamp_out=513),            # all-zero DM list
    dict(nchans=33, ndm_seg=((5.0, 0.0, 3), (5.0, 0.0, 2), (9.0, 2.0, 4)), nsamp_out=1025),  # duplicates
    dict(nchans=64, ndm_seg=((0.0, 40.0, 17),), nsamp_out=777),          # coarse plan, wide windows
]


@pytest.mark.parametrize("dtype", ["u8", "f16", "f32"])
@pytest.mark.parametrize("case", range(len(EDGE)))
@pytest.mark.parametrize("kernel", KERNELS, ids=[KNAME[k] for k in KERNELS])
def test_edge_shapes(case, dtype, kernel):
    e = EDGE[case]
    mean, sig = (128.0, 16.0) if dtype == "u8" else (0.0, 1.0)
    cfg = SurveyConfig(f"edge{case}_{dtype}", e["nchans"], 400.0, -100.0 / max(e["nchans"], 2), 256e-6, e["nsamp_out"],
                       e["ndm_seg"], dtype, mean, sig, 3.0, 1, 1000 + case)
    plan = _plan_with(cfg, kernel)
    x, tab, _ = make_case(cfg)
    out, _ = run_gpu(cfg, x, kernel, plan=plan)
    assert_matches_oracle(cfg, out, oracle_rows(cfg, x.cpu().numpy()), what=cfg.name)


@pytest.mark.parametrize("kernel", KERNELS, ids=[KNAME[k] for k in KERNELS])
def test_strided_and_batched(kernel):
    """dedisp_execute_strided / _batched: padded pitches, 3 beams in one launch == per-beam oracle."""
    cfg = SMALL["c5s"]
    plan = _plan_with(cfg, kernel)
    nsamp_in = cfg.nsamp_out + plan.max_shift
    pitch = nsamp_in + 13
    xs = torch.zeros((3, cfg.nchans + 1, pitch), dtype=torch.uint8, device="cuda")
    outs = torch.full((3, cfg.ndm + 2, cfg.nsamp_out + 5), -7, dtype=torch.int32, device="cuda")
    hosts = []
    for b in range(3):
        x, _, _ = make_case(cfg, seed=500 + b)
        xs[b, :cfg.nchans, :nsamp_in] = x
        hosts.append(x.cpu().numpy())
    plan.execute(xs[:, :cfg.nchans], cfg.nsamp_out, outs[:, :cfg.ndm])
    torch.cuda.synchronize()
    for b in range(3):
        assert_matches_oracle(cfg, outs[b, :cfg.ndm, :cfg.nsamp_out], oracle_rows(cfg, hosts[b]), what=f"beam {b}")
    assert bool((outs[:, cfg.ndm:] == -7).all()) and bool((outs[:, :, cfg.nsamp_out:] == -7).all())


def test_concurrent_executes_on_two_streams():
    """§8(b) ownership: dedisp_execute allocates nothing and leaves the plan read-only for every dtype, so
    two calls on ONE plan may run concurrently on different streams (u8 input: the raw path converts
    inside the kernel, there is no shared scratch)."""
    cfg = SMALL["c2s"]
    plan = _plan_with(cfg, P.KERNEL_SUBBAND)
    xs = [make_case(cfg, seed=700 + i)[0] for i in range(2)]
    outs = [plan.alloc_out(cfg.nsamp_out) for _ in range(2)]
    streams = [torch.cuda.Stream() for _ in range(2)]
    torch.cuda.synchronize()
    for rep in range(3):
        for i in range(2):
            plan.execute(xs[i], cfg.nsamp_out, outs[i], stream=streams[i])
    torch.cuda.synchronize()
    for i in range(2):
        assert_matches_oracle(cfg, outs[i], oracle_rows(cfg, xs[i].cpu().numpy()), what=f"stream {i}")


def test_unaligned_fp32_rows_take_the_raw_path():
    """fp32 rows whose base / pitch are not 16-byte aligned: SUBBAND realigns them in its raw path (no
    silent drop to the NAIVE kernel)."""
    cfg = SMALL["c3s"]
    plan = _plan_with(cfg, P.KERNEL_SUBBAND)
    x, tab, _ = make_case(cfg)
    nsamp_in = cfg.nsamp_out + plan.max_shift
    pitch = nsamp_in + 3 - (nsamp_in % 2)                       # odd pitch: rows start at every 4-byte phase
    buf = torch.zeros(cfg.nchans * pitch + 5, dtype=torch.float32, device="cuda")
    view = buf[1:1 + cfg.nchans * pitch].view(cfg.nchans, pitch)[:, :nsamp_in]    # base off by 4 bytes
    view.copy_(x)
    out = plan.execute(view, cfg.nsamp_out)
    torch.cuda.synchronize()
    assert plan.kernel == P.KERNEL_SUBBAND
    assert_matches_oracle(cfg, out, oracle_rows(cfg, x.cpu().numpy()), what="unaligned fp32 rows")


@pytest.mark.parametrize("kernel", KERNELS, ids=[KNAME[k] for k in KERNELS])
@pytest.mark.parametrize("name,lead", [("c3s", 0), ("c3s", 3), ("c2s", 0), ("c2s", 5), ("c4s", 1)])
def test_guard_bands_are_never_summed(name, lead, kernel):
    """compute-sanitizer is closed on this pool, so out-of-bounds reads are hunted with poison instead:
    the input rows sit in a larger buffer whose every other element (in front of the first row, in the
    pitch padding between rows, behind the last row) holds a value that would wreck any sum it entered
    (NaN for fp, 255 for u8 with the oracle run on the clean rows); `lead` elements in front make the base
    unaligned. The output must still equal the oracle's, and the canaries around out must survive."""
    cfg = SMALL[name]
    plan = _plan_with(cfg, kernel)
    x, tab, _ = make_case(cfg)
    nsamp_in = cfg.nsamp_out + plan.max_shift
    per16 = 16 // x.element_size()
    pitch = (nsamp_in + 2 * per16 + per16 - 1) // per16 * per16 + (1 if lead else 0) * 0
    poison = 255 if cfg.dtype == "u8" else float("nan")
    buf = torch.full((64 + lead + cfg.nchans * pitch + 64,), poison, dtype=x.dtype, device="cuda")
    view = buf[64 + lead: 64 + lead + cfg.nchans * pitch].view(cfg.nchans, pitch)[:, :nsamp_in]
    view.copy_(x)
    obuf = torch.full((cfg.ndm + 2, cfg.nsamp_out + 8), -7, dtype=torch.int32 if cfg.dtype == "u8" else torch.float32, device="cuda")
    out = obuf[1:cfg.ndm + 1, 4:4 + cfg.nsamp_out]
    if kernel == P.KERNEL_TILED and (view.data_ptr() & 15):
        with pytest.raises(P.DedispError) as ei:      # TILED, when forced, wants a 16-byte-aligned base (dedisp.h)
            plan.execute(view, cfg.nsamp_out, out)
        assert ei.value.code == 1
        return
    plan.execute(view, cfg.nsamp_out, out)
    torch.cuda.synchronize()
    assert_matches_oracle(cfg, out, oracle_rows(cfg, x.cpu().numpy()), what=f"{name}/{KNAME[kernel]} lead {lead}")
    assert bool((obuf[0] == -7).all()) and bool((obuf[-1] == -7).all())
    assert bool((obuf[:, :4] == -7).all()) and bool((obuf[:, 4 + cfg.nsamp_out:] == -7).all())


def test_errors():
    cfg = CONFIGS["c1"]
    plan = P.Plan.from_config(cfg)
    x = torch.zeros((cfg.nchans, cfg.nsamp_out + plan.max_shift - 1), device="cuda")
    with pytest.raises(P.DedispError) as ei:
        plan.execute(x, cfg.nsamp_out)     # row too short
    assert ei.value.code == 1
    with pytest.raises(P.DedispError):
        plan.set_kernel(99)
    with pytest.raises(P.DedispError):
        P.Plan(4, 100.0, +1.0, 1e-3, [0.0, 1.0], "f32")       # ascending band rejected (DESIGN R11)
    with pytest.raises(P.DedispError):
        P.Plan(4, 100.0, -1.0, 1e-3, [1.0, 0.5], "f32")       # decreasing DMs rejected


# ---- full-size configs, in the launch configuration bench.py times
def _full(name, nrows):
    cfg = CONFIGS[name]
    x, tab, pulses = make_case(cfg)
    rows = spread_rows(cfg.ndm, nrows, extra=[p[0] for p in pulses])
    return cfg, x, rows


def _boundary_rows(cfg):
    """Rows on both sides of every DM-segment boundary of the plan (c4: 1999/2000, 3199/3200) and of the
    48-row CTA blocks of the SUBBAND kernel next to them."""
    rows, start = [], 0
    for _, _, n in cfg.dm_segments[:-1]:
        start += n
        blk = (start // 48) * 48
        rows += [start - 1, start, blk - 1, blk, blk + 47, blk + 48]
    return [r for r in rows if 0 <= r < cfg.ndm]


@pytest.mark.parametrize("name,nrows", [("c2", 48), ("c3", 64), ("c4", 64)])
def test_full_size_rows_vs_oracle_and_naive(name, nrows):
    """Full-size configs in the launch configuration bench.py times: 64 oracle rows (SURVEY.md §8(d)
    "parity coverage at scale") at the north_star tolerance, and the WHOLE output against the
    oracle-checked NAIVE kernel: bit-equal for u8; for fp every element within 2e-5 * sum|terms| of
    NAIVE (each side is within 1e-5 * sum|terms| of the exact sum), with sum|terms| for the whole
    output obtained by running NAIVE on |x| and that run itself checked against the oracle's abs_sum."""
    cfg, x, rows = _full(name, nrows)
    rows = np.array(sorted(set(rows.tolist()) | set(_boundary_rows(cfg))), dtype=np.int32)
    ref = oracle_rows(cfg, x.cpu().numpy(), rows=rows)
    out_naive, plan = run_gpu(cfg, x, P.KERNEL_NAIVE)
    assert_matches_oracle(cfg, out_naive, ref, rows=rows, what=f"{name}/naive")
    asum = None
    if cfg.dtype != "u8":
        asum = plan.execute(x.abs(), cfg.nsamp_out)
        torch.cuda.synchronize()
        ridx = torch.as_tensor(rows, device="cuda", dtype=torch.long)
        got_asum = asum[ridx].cpu().numpy().astype(np.float64)
        assert (np.abs(got_asum - ref[1]) <= 1e-5 * ref[1]).all(), f"{name}: NAIVE sum|terms| differs from the oracle's"
    for k in (P.KERNEL_TILED, P.KERNEL_SUBBAND, P.KERNEL_AUTO):
        try:
            plan.set_kernel(k)
        except P.DedispError:
            continue
        out = plan.execute(x, cfg.nsamp_out)
        torch.cuda.synchronize()
        assert_matches_oracle(cfg, out, ref, rows=rows, what=f"{name}/kernel{k}")
        if cfg.dtype == "u8":
            assert torch.equal(out, out_naive)
        else:
            nbad = 0
            for d0 in range(0, cfg.ndm, 256):      # row slabs: no full-size temporaries
                sl = slice(d0, min(cfg.ndm, d0 + 256))
                nbad += int(((out[sl] - out_naive[sl]).abs() > 2e-5 * asum[sl]).sum())
            assert nbad == 0, f"{name}/kernel{k}: {nbad} elements further than 2e-5*sum|terms| from NAIVE"
        del out
    del out_naive, asum
    torch.cuda.empty_cache()


def test_c5_one_chunk_batched_rows_vs_oracle():
    """c5 launch shape: 32 beams x 1024 chans x (32768 + maxshift) u8 in one batched launch."""
    cfg = CONFIGS["c5"]
    plan = P.Plan.from_config(cfg)
    nsamp_in = cfg.nsamp_out + plan.max_shift
    tab = oracle_table(cfg)
    assert plan.max_shift == int(tab.max())
    xs = torch.empty((cfg.nbeams, cfg.nchans, nsamp_in), dtype=torch.uint8, device="cuda")
    from paper_1111_6399_b200 import synth
    for b in range(cfg.nbeams):
        xs[b], _ = synth.make_input(cfg, tab, nsamp_in, device="cuda", seed=cfg.seed * 1000003 + b * 101)
    out = plan.execute(xs, cfg.nsamp_out)
    torch.cuda.synchronize()
    rows = spread_rows(cfg.ndm, 24)
    for b in (0, 17, 31):
        ref = oracle_rows(cfg, xs[b].cpu().numpy(), rows=rows)
        assert_matches_oracle(cfg, out[b], ref, rows=rows, what=f"c5 beam {b}")
    plan.set_kernel(P.KERNEL_NAIVE)
    out2 = plan.execute(xs, cfg.nsamp_out)
    torch.cuda.synchronize()
    assert torch.equal(out, out2)


@pytest.mark.parametrize("name", ["c3s", "c2s", "c4s"])
def test_execute_host_matches_oracle(name):
    """dedisp_execute_host (the e2e call bench.py times): host buffers in and out. For aligned fp32
    rows the H2D copy is split per sub-band pass on a second stream; the result must not depend on
    that, nor on calling twice in a row with different data (scratch and events are reused)."""
    cfg = SMALL[name]
    if name == "c3s":   # make nsamp_in a multiple of 4 so that the per-pass overlap path is taken
        tab = oracle_table(cfg)
        cfg = shrink(cfg, nsamp_out=cfg.nsamp_out + (-(cfg.nsamp_out + int(tab.max())) % 4))
    plan = P.Plan.from_config(cfg)
    try:
        plan.set_kernel(P.KERNEL_SUBBAND)     # the overlapped copies belong to SUBBAND (AUTO may prefer TILED for coarse plans)
    except P.DedispError:
        pass
    for seed in (11, 12):
        x, tab, _ = make_case(cfg, device="cpu", seed=seed)
        h_in = x.pin_memory()
        out = plan.execute_host(h_in, cfg.nsamp_out)
        assert_matches_oracle(cfg, out, oracle_rows(cfg, x.numpy()), what=f"{name}/execute_host seed {seed}")
    if name == "c4s":   # fp16, three DM ranges: launches in reverse order, each range's last sub-band stores; 4 DM blocks = 4 slabs
        assert plan.kernel == P.KERNEL_SUBBAND and plan.geometry()["nranges"] == 3 and plan.last_host_slabs == 4
    if name == "c3s":
        assert plan.num_subbands() > 1 and (cfg.nsamp_out + plan.max_shift) % 4 == 0


def test_execute_host_slab_branch_matches_oracle():
    """The branch bench.py's e2e figure times on c3: aligned fp32 rows, > 1 pass, >= 4 DM blocks, so
    that the per-pass H2D overlap AND the last two passes in DM slabs (one per DM block here, at most 8) with
    overlapped D2H both run (plan.cu dedisp_execute_host). Full output vs the oracle, twice with different data."""
    cfg = shrink(CONFIGS["c3"], nchans=300, nsamp_out=4500, ndm_stride=16)      # 256 DMs -> 6 DM blocks
    tab = oracle_table(cfg)
    cfg = shrink(cfg, nsamp_out=cfg.nsamp_out + (-(cfg.nsamp_out + int(tab.max())) % 4))
    plan = P.Plan.from_config(cfg)
    plan.set_kernel(P.KERNEL_SUBBAND)     # (AUTO would pick TILED for a plan this coarse: passes of a few channels)
    assert plan.num_subbands() > 1 and (cfg.nsamp_out + plan.max_shift) % 4 == 0
    for seed in (21, 22):
        x, _, _ = make_case(cfg, device="cpu", seed=seed)
        out = plan.execute_host(x.pin_memory(), cfg.nsamp_out)
        assert plan.last_host_slabs == 6, "the slab branch was not taken"
        assert_matches_oracle(cfg, out, oracle_rows(cfg, x.numpy()), what=f"execute_host slabs seed {seed}")


def test_execute_host_multi_range_without_slabs():
    """Three DM ranges in three DM blocks (< 4: no slab overlap): the launches still run last sub-band first with
    the H2D copy ordered to match, and every range's LAST sub-band stores. Full output vs the oracle, twice."""
    cfg = shrink(CONFIGS["c4"], nchans=257, nsamp_out=3100, ndm_stride=40)       # 105 DMs: 3 blocks, 3 ranges
    plan = P.Plan.from_config(cfg)
    plan.set_kernel(P.KERNEL_SUBBAND)
    g = plan.geometry()
    assert g["nblk"] == 3 and g["nranges"] == 3 and plan.launches_per_execute > 1
    for seed in (41, 42):
        x, _, _ = make_case(cfg, device="cpu", seed=seed)
        out = plan.execute_host(x.pin_memory(), cfg.nsamp_out)
        assert plan.last_host_slabs == 0
        assert_matches_oracle(cfg, out, oracle_rows(cfg, x.numpy()), what=f"execute_host 3 ranges seed {seed}")
        dev = plan.execute(x.cuda(), cfg.nsamp_out)                                # forward order, resident input
        torch.cuda.synchronize()
        assert_matches_oracle(cfg, dev, oracle_rows(cfg, x.numpy()), what=f"execute 3 ranges seed {seed}")


def test_execute_host_slab_branch_u8_unmerged_passes():
    """The same branch for a u8 plan whose passes are launched one by one (packed 16-bit sums, raw path): the
    channels arrive in the order the launches need them, the last two launches run slab by slab, and every slab's
    rows are converted to int32 before their D2H copy. Bit-exact against the oracle, twice."""
    cfg = SurveyConfig("host_u8", 700, 1500.0, -0.4, 64e-6, 3000, ((0.0, 2.0, 240),), "u8", 128.0, 16.0, 20.0, 1, 9)
    plan = P.Plan.from_config(cfg)
    assert plan.kernel == P.KERNEL_SUBBAND and plan.launches_per_execute == plan.num_subbands() + 1 == 7    # 6 passes + the conversion
    for seed in (31, 32):
        x, _, _ = make_case(cfg, device="cpu", seed=seed)
        out = plan.execute_host(x.pin_memory(), cfg.nsamp_out)
        assert plan.last_host_slabs == 5, "the slab branch was not taken"
        assert_matches_oracle(cfg, out, oracle_rows(cfg, x.numpy()), what=f"execute_host u8 slabs seed {seed}")


def test_execute_host_with_merged_passes():
    """A merged launch reads every channel at once, so dedisp_execute_host must not split the H2D copy
    per pass behind it: result still equals the oracle."""
    cfg = SMALL["c3s"]
    tab = oracle_table(cfg)
    cfg = shrink(cfg, nsamp_out=cfg.nsamp_out + (-(cfg.nsamp_out + int(tab.max())) % 4))
    plan = P.Plan.from_config(cfg)
    plan.set_kernel(P.KERNEL_SUBBAND)
    plan.set_pass_merge(True)
    x, _, _ = make_case(cfg, device="cpu", seed=31)
    out = plan.execute_host(x.pin_memory(), cfg.nsamp_out)
    assert plan.last_host_slabs == 0
    assert_matches_oracle(cfg, out, oracle_rows(cfg, x.numpy()), what="execute_host merged")


@pytest.mark.parametrize("name", ["c3s", "c4s", "paper"])
def test_merged_passes_match_oracle(name):
    """dedisp_plan_set_pass_merge: all SUBBAND passes in one launch, partial sums added with L2
    reductions in any order. fp plans stay within the tolerance; u8 plans ("paper" merges on its own:
    many short passes) stay bit-exact because their fp32 partial sums are exact integers."""
    cfg = SMALL[name]
    plan = _plan_with(cfg, P.KERNEL_SUBBAND)
    plan.set_pass_merge(True)
    assert plan.num_subbands() > 1
    x, tab, _ = make_case(cfg)
    ref = oracle_rows(cfg, x.cpu().numpy())
    for _ in range(2):                       # twice: the merged path zeroes out itself
        out = plan.execute(x, cfg.nsamp_out)
        torch.cuda.synchronize()
        assert_matches_oracle(cfg, out, ref, what=f"{name}/merged")


# ---- u8 plans: packed 16-bit sums on the integer pipes (SubbandGeom::i16) vs. the fp32 sums of DEDISP_PLAN_NO_PACKED
@pytest.mark.parametrize("name", ["c2s", "c5s", "paper", "fine"])
def test_packed_and_fp32_u8_plans_both_match_oracle(name):
    cfg = SMALL[name]
    x, tab, _ = make_case(cfg)
    ref = oracle_rows(cfg, x.cpu().numpy())
    outs = []
    for packed in (True, False):
        plan = P.Plan.from_config(cfg, packed=packed)
        plan.set_kernel(P.KERNEL_SUBBAND)
        out = plan.execute(x, cfg.nsamp_out)
        torch.cuda.synchronize()
        assert_matches_oracle(cfg, out, ref, what=f"{name}/packed={packed}")
        outs.append(out)
    assert torch.equal(outs[0], outs[1])


@pytest.mark.parametrize("value", [255, "random"])
def test_packed_sums_do_not_overflow_a_16_bit_lane(value):
    """The worst case of the packed path: a DM plan so fine that only the 257-channel cap cuts the sub-bands,
    and input that is 255 everywhere (every 16-bit lane of a full pass ends at 65535 = 257 * 255 exactly) or
    uniform over 0..255."""
    cfg = SurveyConfig("packed_overflow", 700, 1500.0, -0.1, 64e-6, 3500, ((0.0, 0.02, 101),), "u8", 128.0, 16.0, 20.0, 0, 5)
    plan = P.Plan.from_config(cfg)
    plan.set_kernel(P.KERNEL_SUBBAND)
    assert plan.verify_records() == 0
    sb = plan.subbands()
    assert int(np.diff(sb).max()) == 257                       # a full-width pass exists
    tab = oracle_table(cfg)
    nsamp_in = cfg.nsamp_out + int(tab.max())
    if value == "random":
        x = np.random.default_rng(11).integers(0, 256, size=(cfg.nchans, nsamp_in), dtype=np.uint8)
    else:
        x = np.full((cfg.nchans, nsamp_in), 255, dtype=np.uint8)
    out = plan.execute(torch.from_numpy(x).cuda(), cfg.nsamp_out)
    torch.cuda.synchronize()
    assert_matches_oracle(cfg, out, oracle_rows(cfg, x), what=f"packed overflow {value}")
    if value == 255:
        assert int(out.min()) == int(out.max()) == 700 * 255
