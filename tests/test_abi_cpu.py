"""CPU-only checks of the C-ABI library: it loads without a GPU, exports every symbol that
include/dedisp.h declares, its host shift-table builder agrees with the ORACLE's independent
table on every entry of all five configs, and host-side validation returns the documented codes.
No compute call is made here.
"""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
import paper_1111_6399_b200 as P
from paper_1111_6399_b200 import CONFIGS, api

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "dedisp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dedisp_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    declared = _declared_symbols()
    assert len(declared) >= 20
    L = api.lib()
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/dedisp.h but not exported"
    assert sorted(api.SYMBOLS) == declared, "binding's symbol list out of sync with the header"


@pytest.mark.parametrize("name", list(CONFIGS))
def test_library_shift_table_equals_oracle_table(name, golden):
    cfg = CONFIGS[name]
    tab, mx = P.shift_table_host(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, cfg.dm_list())
    ref = oracle.shift_table(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, cfg.dm_list())
    assert np.array_equal(tab.astype(np.int64), ref)
    pins, _, _ = golden
    assert mx == pins[name][0]                       # maxshift regression value (tests/golden/shift_pins.txt)


def test_host_only_plan_inspection_and_refusal():
    cfg = CONFIGS["c2"]
    plan = P.Plan.from_config(cfg, host_only=True)
    assert (plan.nchans, plan.ndm, plan.max_shift) == (496, 2000, 28324)
    assert np.array_equal(plan.shifts().astype(np.int64),
                          oracle.shift_table(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, cfg.dm_list()))
    assert plan.kernel in (P.KERNEL_TILED, P.KERNEL_SUBBAND, P.KERNEL_NAIVE)
    assert plan.launches_per_execute >= 1
    # a host-only plan never executes, and there is no CPU fallback
    rc = api.lib().dedisp_execute(plan._h, ctypes.c_void_p(16), 10, ctypes.c_void_p(16), None)
    assert rc == api.EUNSUPPORTED


def test_validation_codes():
    L = api.lib()
    dm = (ctypes.c_double * 3)(0.0, 1.0, 2.0)
    tab = (ctypes.c_int * 12)()
    mx = ctypes.c_longlong()
    ok = lambda *a: L.dedisp_shift_table_host(*a, tab, ctypes.byref(mx))
    assert ok(4, 100.0, -1.0, 1e-3, dm, 3) == api.OK
    assert ok(0, 100.0, -1.0, 1e-3, dm, 3) == api.EINVAL
    assert ok(4, 100.0, +1.0, 1e-3, dm, 3) == api.EINVAL      # ascending band
    assert ok(4, 100.0, -1.0, 0.0, dm, 3) == api.EINVAL       # tsamp
    assert ok(4, 3.0, -1.0, 1e-3, dm, 3) == api.EINVAL        # lowest channel <= 0 MHz
    bad = (ctypes.c_double * 3)(0.0, 2.0, 1.0)
    assert ok(4, 100.0, -1.0, 1e-3, bad, 3) == api.EINVAL     # decreasing DMs
    nan = (ctypes.c_double * 3)(0.0, float("nan"), 1.0)
    assert ok(4, 100.0, -1.0, 1e-3, nan, 3) == api.EINVAL
    huge = (ctypes.c_double * 3)(0.0, 1.0, 1e9)
    assert ok(4, 100.0, -20.0, 1e-9, huge, 3) == api.EUNSUPPORTED  # shift >= 2^31
    h = ctypes.c_void_p()
    assert L.dedisp_plan_create_ex(ctypes.byref(h), 4, 100.0, -1.0, 1e-3, dm, 3, 7, 1) == api.EINVAL  # dtype
    assert L.dedisp_plan_destroy(None) == api.OK
    assert L.dedisp_plan_max_shift(None) == -1
    assert L.dedisp_error_string(api.ECUDA) == b"CUDA error"


def test_no_gpu_means_loud_failure():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(P.DedispError):
        P.Plan.from_config(CONFIGS["c1"])


@pytest.mark.parametrize("name", list(CONFIGS))
def test_subband_records_encode_exactly_the_shift_table(name):
    """The SUBBAND kernel only ever sees packed records (+ window bases + per-pass skews); rebuilding
    s(c,d) from them on the host must give back the plan's table, and every channel must belong to
    exactly one pass (dedisp_plan_verify_records == 0 mismatches)."""
    plan = P.Plan.from_config(CONFIGS[name], host_only=True)
    g = plan.num_subbands()
    assert g >= 1
    sb = plan.subbands()
    assert sb[0] == 0 and sb[-1] == CONFIGS[name].nchans and np.all(np.diff(sb) > 0)
    assert plan.verify_records() == 0


def test_generated_channel_body_is_up_to_date():
    """subband_rows.inc is committed generated code: it must equal what gen_subband_rows.py emits for
    its default (= plan.h) tile constants, so that the file and its generator cannot drift apart."""
    import importlib.util
    import os
    csrc = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_1111_6399_b200", "csrc")
    spec = importlib.util.spec_from_file_location("gen_subband_rows", os.path.join(csrc, "gen_subband_rows.py"))
    gen = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(gen)
    with open(os.path.join(csrc, "subband_rows.inc")) as f:
        committed = f.read()
    d, k, sp, g, stride = (int(x) for x in committed.splitlines()[0].split("gen_subband_rows.py")[1].split("-")[0].split())
    assert committed == gen.generate(d, k, sp, g, stride)
    with open(os.path.join(csrc, "plan.h")) as f:
        plan_h = f.read()
    assert f"#define SB_D_CFG {d}" in plan_h and f"#define SB_K_CFG {k}" in plan_h
    assert f"#define SB_S_CFG {sp}" in plan_h and f"#define SB_G_CFG {g}" in plan_h
    # the packed 16-bit variant of u8 plans
    with open(os.path.join(csrc, "subband_rows_i16.inc")) as f:
        committed = f.read()
    d16, k16, omax, stride16 = (int(x) for x in committed.splitlines()[0].split("generate_i16")[1].split(")")[0].split())
    assert (d16, k16, stride16) == (d, k, stride) and (d16, k16, omax, stride16) == gen.DEFAULT_I16
    assert committed == gen.generate_i16(d16, k16, omax, stride16)
    assert f"#define SB16_OMAX_CFG {omax}" in plan_h


@pytest.mark.parametrize("name", ["c2", "c5"])
def test_u8_plans_are_packed_with_at_most_257_channels_per_pass(name):
    """u8 plans sum packed 16-bit pairs: 257 channels x 255 is the most a 16-bit lane holds, so no pass may be
    wider; DEDISP_PLAN_NO_PACKED plans keep the fp32 geometry. Both encode the shift table exactly."""
    cfg = CONFIGS[name]
    packed = P.Plan.from_config(cfg, host_only=True)
    plain = P.Plan.from_config(cfg, host_only=True, packed=False)
    assert packed.verify_records() == 0 and plain.verify_records() == 0      # includes the 257-channel check
    assert packed.num_subbands() * 257 >= cfg.nchans
    assert packed.geometry() != plain.geometry()


def test_kernel_selection_falls_back_when_subband_is_not_admitted():
    """AUTO resolves to SUBBAND only when the plan admits it: u8 sums must stay exact in fp32
    (nchans*255 < 2^24), otherwise the int32 TILED kernel is used; forcing SUBBAND is refused."""
    import paper_1111_6399_b200 as P
    ok = P.Plan(512, 1500.0, -0.5, 64e-6, [0.0, 1.0, 2.0, 3.0], "u8", host_only=True)
    assert ok.kernel == P.KERNEL_SUBBAND and ok.num_subbands() >= 1 and ok.verify_records() == 0
    big = P.Plan(70000, 1500.0, -0.01, 64e-6, [0.0, 1.0], "u8", host_only=True)   # 70000*255 > 2^24
    assert big.kernel == P.KERNEL_TILED and big.num_subbands() == 0
    with pytest.raises(P.DedispError) as ei:
        big.set_kernel(P.KERNEL_SUBBAND)
    assert ei.value.code == 4
    f32 = P.Plan(70000, 1500.0, -0.01, 64e-6, [0.0, 1.0], "f32", host_only=True)   # no exactness bound for fp32
    assert f32.kernel == P.KERNEL_SUBBAND
