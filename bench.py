#!/usr/bin/env python
"""bench.py — one JSON line per run (contract in the task statement).

A step = one pass of the whole hot path (shifted accumulate over all channels for every DM trial
of the plan; the shift table is built once per plan, outside the timed region, as the method
does) over one synthetic batch of the workload. Default workload: c3, the MeerKAT-like fp32 config
that carries BASELINE.json's roofline target. Metric: Gadds/s, one add per (DM, channel, sample).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c3] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
from dataclasses import replace
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "dedispersion Gadds/s (DM x chan x sample)"
UNIT = "Gadds/s"
N_SM, LANES_PER_SM = 148, 128          # B200: 148 SMs x 128 FP32/INT32 add lanes


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p.get("hbm_gbs", 6650.0)), float(p.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


def beam_seed(cfg_seed: int, rank: int) -> int:
    """Each rank de-disperses its own synthetic beam (independent problems: DESIGN.md section 9)."""
    return cfg_seed + 7919 * rank


def max_over_ranks(x: float, world: int, device="cuda") -> float:
    """Slowest rank's time: the whole-job time of a sharded run (contract: max over ranks)."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(adds_per_rank: int, steps: int, world: int, slowest_seconds: float) -> float:
    """Whole-job Gadds/s: every rank did adds_per_rank*steps adds in the slowest rank's time."""
    return world * adds_per_rank * steps / slowest_seconds / 1e9


class ClockSampler:
    """nvidia-smi clocks/throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=fd, stderr=subprocess.DEVNULL)
            os.close(fd)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        with open(self.path) as f:
            for line in f:
                tok = [t.strip() for t in line.split(",")]
                if len(tok) < 9:
                    continue
                try:
                    sm.append(float(tok[1])); mx.append(float(tok[2])); pw.append(float(tok[3]))
                except ValueError:
                    continue
                for n, v in zip(names, tok[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        os.unlink(self.path)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def oracle_sample(cfg, per_call_s: float = 3.0):
    """The oracle, as it stands, on a bounded row subset of the workload: returns run(rows) -> seconds,
    the row list sized for about per_call_s of one core, and the adds per row."""
    import numpy as np
    import oracle
    from paper_1111_6399_b200 import synth
    dm = cfg.dm_list()
    tab = oracle.shift_table(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm)
    nsamp_in = cfg.nsamp_out + int(tab.max())
    x, _ = synth.make_input(cfg, tab, nsamp_in, device="cpu")
    x = x.numpy()
    rate_guess = {"f32": 1.0e9, "u8": 2.0e9, "f16": 0.12e9}[cfg.dtype]
    per_row = cfg.nchans * cfg.nsamp_out
    nrows = int(max(1, min(cfg.ndm, round(per_call_s * rate_guess / per_row))))

    def rows_for(n):
        return np.linspace(0, cfg.ndm - 1, min(cfg.ndm, n)).round().astype(np.int32)

    def run(rows):
        t0 = time.perf_counter()
        oracle.dedisperse(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm, x, cfg.nsamp_out, rows=rows)
        return time.perf_counter() - t0

    return run, rows_for, nrows, per_row


def cpu_oracle_baseline(cfg, per_call_s: float = 3.0, repeats: int = 3):
    """cpu_baseline: one warm-up call, then the median of `repeats` calls, (1) on one core and (2) on all
    host cores - the unchanged single-threaded oracle entry point called on disjoint DM-row subsets from
    one Python thread per core (ctypes releases the GIL), SURVEY.md section 8(d) "Oracle timing"."""
    import numpy as np
    from concurrent.futures import ThreadPoolExecutor
    run, rows_for, nrows, per_row = oracle_sample(cfg, per_call_s)
    rows = rows_for(nrows)
    run(rows_for(1))                                     # warm-up: page in the input, build the oracle .so
    t1 = sorted(run(rows) for _ in range(repeats))[repeats // 2]
    cores = os.cpu_count() or 1
    all_rows = rows_for(min(cfg.ndm, nrows * cores))
    parts = [p for p in np.array_split(all_rows, cores) if p.size]

    def run_all():
        t0 = time.perf_counter()
        with ThreadPoolExecutor(len(parts)) as ex:
            list(ex.map(run, parts))
        return time.perf_counter() - t0

    run_all()
    tn = sorted(run_all() for _ in range(repeats))[repeats // 2]
    sample = (f"{rows.size} of {cfg.ndm} DM rows (evenly spread) x all {cfg.nchans} channels x all {cfg.nsamp_out} samples "
              f"of {cfg.name}; 1 warm-up + median of {repeats} calls")
    vec = None
    if cfg.dtype in ("u8", "f32"):
        # the threaded, time-blocked, compiler-vectorised CPU kernel of baseline_cpu/
        # (the modern counterpart of the paper's SSE/AVX kernel) on a larger row sample
        import baseline_cpu
        import oracle
        from paper_1111_6399_b200 import synth
        dm = cfg.dm_list()
        tab = oracle.shift_table(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm)
        x, _ = synth.make_input(cfg, tab, cfg.nsamp_out + int(tab.max()), device="cpu")
        x = x.numpy()
        vrows = rows_for(min(cfg.ndm, max(cores, nrows * cores * 4)))

        def run_vec():
            t0 = time.perf_counter()
            baseline_cpu.dedisperse(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, dm[vrows], x, cfg.nsamp_out, cores)
            return time.perf_counter() - t0

        run_vec()
        tv = sorted(run_vec() for _ in range(repeats))[repeats // 2]
        vec = {"value": vrows.size * per_row / tv / 1e9, "unit": UNIT, "cores": cores, "rows": int(vrows.size),
               "seconds_per_call": tv, "kind": "baseline_cpu/: threaded over DM rows, 8192-sample accumulator tiles, "
               "compiler-vectorised inner loop (-O3 -march=native); checked against the oracle in tests/test_cpu_baseline.py"}
    return {"value": rows.size * per_row / t1 / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
            "seconds_per_call": t1,
            "all_cores": {"value": all_rows.size * per_row / tn / 1e9, "unit": UNIT, "cores": len(parts),
                          "rows": int(all_rows.size), "seconds_per_call": tn,
                          "how": "same oracle entry point, one Python thread per core on disjoint DM rows"},
            "vectorised": vec}


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    run, rows_for, nrows, per_row = oracle_sample(cfg, per_call_s=3.0)
    rows = rows_for(nrows)
    for _ in range(max(1, args.warmup)):
        run(rows)
    times = [run(rows) for _ in range(args.steps)]
    tot = sum(times)
    adds = rows.size * per_row
    val = adds * args.steps / tot / 1e9
    sample = (f"{rows.size} of {cfg.ndm} DM rows (evenly spread) x all {cfg.nchans} channels x all {cfg.nsamp_out} samples "
              f"of {cfg.name}, single thread; each step = this sample")
    line = {"metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic", "impl": "reference",
            "config": {"workload": cfg.name, "nchans": cfg.nchans, "ndm": cfg.ndm, "nsamp_out": cfg.nsamp_out,
                       "note": "oracle/ (plain C++ triple loop) on the host; each step = the bounded sample"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# dram__bytes_read.sum + dram__bytes_write.sum per dedisp_execute, summed over the launches of one
# execute, from the committed ncu captures (profiles/r2_dram_<config>.csv), keyed by (workload, kernel)
NCU_TRAFFIC_BYTES = {}
_traffic_file = os.path.join(ROOT, "profiles", "r2_traffic.json")
if os.path.exists(_traffic_file):
    with open(_traffic_file) as _f:
        NCU_TRAFFIC_BYTES = {tuple(k.split("/")): float(v) for k, v in json.load(_f).items()}


def add_peak(sm_mhz: float) -> float:
    return N_SM * LANES_PER_SM * sm_mhz * 1e6 / 1e9


def resident_steps(plan, x, nsamp_out, out, steps, warmup):
    """`steps` executes with the input resident in HBM, each bracketed by CUDA events on the launching
    stream; returns the per-step device times (ms) and the time from the first to the last event."""
    import torch
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        plan.execute(x, nsamp_out, out)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    torch.cuda.synchronize()
    for a, b in evs:
        a.record(stream)
        plan.execute(x, nsamp_out, out)
        b.record(stream)
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs], evs[0][0].elapsed_time(evs[-1][1])


def other_configs(sm_max_mhz: float, steps: int = 3, warmup: int = 3):
    """The other full-size configs (c2, c4, c5-one-chunk-of-32-beams), resident inputs, a few steps each, so
    that the driver-run default line records them too (they are parity-test cases, not the headline)."""
    import torch
    import paper_1111_6399_b200 as P
    from paper_1111_6399_b200 import CONFIGS, synth
    res = {}
    for name in ("c2", "c4", "c5"):
        cfg = CONFIGS[name]
        plan = P.Plan.from_config(cfg)
        nsamp_in = cfg.nsamp_out + plan.max_shift
        tab = plan.shifts()
        if cfg.nbeams > 1:
            x = torch.empty((cfg.nbeams, cfg.nchans, nsamp_in), dtype=torch.uint8, device="cuda")
            for b in range(cfg.nbeams):
                x[b], _ = synth.make_input(cfg, tab, nsamp_in, device="cuda", seed=cfg.seed * 1000003 + b * 101)
            out = plan.alloc_out(cfg.nsamp_out, cfg.nbeams)
        else:
            x, _ = synth.make_input(cfg, tab, nsamp_in, device="cuda")
            out = plan.alloc_out(cfg.nsamp_out)
        ms, _ = resident_steps(plan, x, cfg.nsamp_out, out, steps, warmup)
        adds = cfg.nbeams * cfg.ndm * cfg.nchans * cfg.nsamp_out
        med = sorted(ms)[len(ms) // 2]
        kname = {1: "naive", 2: "tiled", 3: "subband"}[plan.kernel]
        res[cfg.name] = {"ms_per_step": med, "value": adds / med / 1e6, "frac": adds / med / 1e6 / add_peak(sm_max_mhz),
                         "kernel": kname, "launches_per_step": plan.launches_per_execute, "steps": steps,
                         "beams": cfg.nbeams, "traffic": NCU_TRAFFIC_BYTES.get((cfg.name, kname))}
        del x, out, plan
        torch.cuda.empty_cache()
    return res


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist

    import paper_1111_6399_b200 as P
    from paper_1111_6399_b200 import synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a GPU: the product has no CPU path"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over(x: float) -> float:
        return max_over_ranks(x, world)

    hbm_gbs, sm_max_mhz, peak_src = _peaks()
    plan = P.Plan.from_config(cfg)                      # table build + upload: once per plan, not per step
    if args.kernel:
        plan.set_kernel({"naive": 1, "tiled": 2, "subband": 3}[args.kernel])
    if args.merge_passes:
        plan.set_pass_merge(True)
    nsamp_in = cfg.nsamp_out + plan.max_shift
    # each rank de-disperses its own beam (independent problems, no data-path collective): weak scaling
    x, _ = synth.make_input(cfg, plan.shifts(), nsamp_in, device="cuda", seed=beam_seed(cfg.seed, rank))
    out = plan.alloc_out(cfg.nsamp_out)
    adds = cfg.ndm * cfg.nchans * cfg.nsamp_out
    launches = plan.launches_per_execute
    stream = torch.cuda.current_stream()

    for _ in range(args.warmup):
        plan.execute(x, cfg.nsamp_out, out)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    for a, b in evs:                                    # input (4.4 GB for c3) >> 126 MB L2: no flush needed
        a.record(stream)
        plan.execute(x, cfg.nsamp_out, out)
        b.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over(evs[0][0].elapsed_time(evs[-1][1]))
    step_list = sorted(a.elapsed_time(b) for a, b in evs)
    step_ms = sum(step_list) / args.steps                                # device time of one execute (mean)
    value = job_value(adds, args.steps, world, total_ms * 1e-3)

    # ---- e2e: the host-buffer C-ABI call; H2D + kernels + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        esteps = max(1, min(args.steps, args.e2e_steps))
        h_in = torch.empty((cfg.nchans, nsamp_in), dtype=x.dtype, pin_memory=True)
        h_in.copy_(x)
        h_out = torch.empty((cfg.ndm, cfg.nsamp_out), dtype=out.dtype, pin_memory=True)
        plan.execute_host(h_in, cfg.nsamp_out, h_out)   # warm-up: allocates the scratch
        barrier()
        t0 = time.perf_counter()
        for _ in range(esteps):
            plan.execute_host(h_in, cfg.nsamp_out, h_out)
        barrier()
        et = max_over(time.perf_counter() - t0)
        # outside the timed region: the host result of the LAST timed call against the device-resident
        # `out` of the timed loop above (same input). The host call runs the passes in another order, so
        # fp sums may differ in their last bits: |diff| <= 2e-5 * sum|terms| (each side within 1e-5 of the
        # exact sum), with sum|terms| taken as nchans * mean|x|; integer outputs must be equal.
        rows = torch.linspace(0, cfg.ndm - 1, min(cfg.ndm, 97)).round().long()
        host_rows, dev_rows = h_out[rows], out[rows.cuda()].cpu()
        if cfg.dtype == "u8":
            e2e_ok, e2e_err = bool(torch.equal(host_rows, dev_rows)), 0.0
        else:
            bound = 2e-5 * cfg.nchans * float(x[:: max(1, cfg.nchans // 64)].float().abs().mean())
            e2e_err = float((host_rows - dev_rows).abs().max())
            e2e_ok = e2e_err <= bound
        e2e = {"value": job_value(adds, esteps, world, et), "unit": UNIT,
               "h2d_bytes_per_step": h_in.numel() * h_in.element_size(),
               "d2h_bytes_per_step": h_out.numel() * h_out.element_size(), "steps": esteps,
               "ms_per_step": 1e3 * et / esteps, "api": "dedisp_execute_host (pinned host buffers)",
               "e2e_checked": e2e_ok, "e2e_check": f"{rows.numel()} rows of the last timed call's host output vs the "
               f"device-resident output, max |diff| {e2e_err:.3g}", "host_slabs": plan.last_host_slabs}
        assert e2e_ok, e2e["e2e_check"]
        del h_in, h_out

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak = add_peak(sm_max_mhz)                                     # Gadds/s at the max SM clock
    achieved = adds / (step_ms * 1e-3) / 1e9
    esize = cfg.esize
    bytes_once = cfg.nchans * nsamp_in * esize + cfg.ndm * cfg.nsamp_out * 4
    kname = {1: "naive", 2: "tiled", 3: "subband"}[plan.kernel]
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": UNIT, "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_BYTES.get((cfg.name, kname)),
                "kernel": f"dedisp_{kname}_kernel", "launches_per_step": launches,
                "peak_source": f"148 SMs x 128 lanes x sm_max_mhz ({peak_src} MEASURED_PEAKS.json clock)",
                "hbm_bytes_once": bytes_once, "hbm_time_ms_at_peak": bytes_once / (hbm_gbs * 1e9) * 1e3,
                "hbm_achieved_gbs": bytes_once / (step_ms * 1e-3) / 1e9, "hbm_peak_gbs": hbm_gbs,
                "ms_mean": step_ms, "ms_median": step_list[len(step_list) // 2], "ms_best": step_list[0],
                "frac_median": adds / (step_list[len(step_list) // 2] * 1e-3) / 1e9 / peak,
                "frac_best": adds / (step_list[0] * 1e-3) / 1e9 / peak}
    if clocks and clocks.get("sm_mhz"):
        roofline["frac_at_sampled_clock"] = achieved / add_peak(clocks["sm_mhz"])

    del x, out
    torch.cuda.empty_cache()
    others = None
    if world == 1 and args.config == "c3" and not args.no_others and not args.kernel:
        others = other_configs(sm_max_mhz)

    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline = cpu_oracle_baseline(cfg, per_call_s=args.cpu_seconds)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "i32" if cfg.dtype == "u8" else "f32",
            "data": "synthetic",
            "config": {"workload": cfg.name, "nchans": cfg.nchans, "ndm": cfg.ndm, "nsamp_out": cfg.nsamp_out,
                       "nsamp_in": nsamp_in, "in_dtype": cfg.dtype, "beams_per_gpu": 1,
                       "l2": "input larger than L2, no flush", "kernel": kname,
                       "parallelism": f"{world} independent beams, one per GPU, no collective"},
            "real_time_factor": cfg.nsamp_out * cfg.tsamp / (total_ms / args.steps * 1e-3),
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches * args.steps,
            "roofline": roofline, "cpu_baseline": cpu_baseline, "others": others}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_c5_stream(args, cfg):
    """c5 (configs[4]): 32 beams x 1024 ch u8, consecutive 32768-sample chunks through the streaming
    driver. value = one chunk of all beams, inputs resident (dedisp_execute_batched); e2e = chunks
    pushed from pinned host memory through dedisp_stream_push (H2D overlapped with compute, maxshift
    carry on the device), reading back the per-(beam, DM) maximum of every block. 1 GPU only."""
    import torch

    import paper_1111_6399_b200 as P
    from paper_1111_6399_b200 import synth

    assert torch.cuda.is_available(), "bench.py needs a GPU: the product has no CPU path"
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    hbm_gbs, sm_max_mhz, peak_src = _peaks()
    plan = P.Plan.from_config(cfg)
    nb, chunk = cfg.nbeams, cfg.nsamp_out
    nsamp_in = chunk + plan.max_shift
    tab = plan.shifts()
    xs = torch.empty((nb, cfg.nchans, nsamp_in), dtype=torch.uint8, device="cuda")
    for b in range(nb):
        xs[b], _ = synth.make_input(cfg, tab, nsamp_in, device="cuda", seed=cfg.seed * 1000003 + b * 101)
    out = plan.alloc_out(chunk, nb)
    adds = nb * cfg.ndm * cfg.nchans * chunk
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        plan.execute(xs, chunk, out)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(0)
    torch.cuda.synchronize()
    sampler.start()
    for a, b in evs:
        a.record(stream)
        plan.execute(xs, chunk, out)
        b.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    total_ms = evs[0][0].elapsed_time(evs[-1][1])
    step_ms = sum(a.elapsed_time(b) for a, b in evs) / args.steps
    value = adds * args.steps / (total_ms * 1e-3) / 1e9
    del out
    if args.no_e2e:
        e2e = None
        del xs
    else:
        e2e = _c5_stream_e2e(args, cfg, plan, xs, adds)
    return _c5_line(args, cfg, plan, hbm_gbs, sm_max_mhz, peak_src, value, total_ms, step_ms, clocks, e2e, adds, nsamp_in)


def _c5_stream_e2e(args, cfg, plan, xs, adds):
    import torch
    import paper_1111_6399_b200 as P
    nb, chunk = cfg.nbeams, cfg.nsamp_out
    # ---- e2e: configs[4]'s stream of 60 consecutive chunks through the streaming driver. The chunks cycle
    # through a pool of 3 distinct pinned host chunks (generating 60 x 1 GB is outside the method); the
    # first chunk's block is checked against the oracle outside the timed region.
    pool = [xs[:, :, plan.max_shift - k * 4096: plan.max_shift - k * 4096 + chunk].contiguous().cpu().pin_memory() for k in range(3)]
    del xs
    torch.cuda.empty_cache()
    st = P.Stream(plan, nb, chunk, 3)                     # 3 buffers: block k-1 is still being read while k+1 is enqueued
    nchunks = cfg.nchunks if not args.stream_chunks else args.stream_chunks
    h_max = torch.empty((nchunks, nb, cfg.ndm), dtype=torch.int32, pin_memory=True)
    read_done = [torch.cuda.Event() for _ in range(3)]

    def read_block(k, ptr, ev):                           # the consumer: per-(beam, DM) maxima of block k
        st.wait_event(ev)
        h_max[k].copy_(st.out_view(ptr).amax(dim=2), non_blocking=True)
        read_done[k % 3].record()
        st.release_after(read_done[k % 3])                # the driver may overwrite the block only after this read

    torch.cuda.synchronize()
    t0 = time.perf_counter()
    prev = None
    for k in range(nchunks):
        ptr, ev = st.push(pool[k % 3])
        if prev is not None:                             # read block k-1's metric while block k computes
            read_block(k - 1, *prev)
        prev = (ptr, ev)
    read_block(nchunks - 1, *prev)
    torch.cuda.synchronize()
    et = time.perf_counter() - t0
    st.close()
    # check (outside the timed region): block 0 = the first chunk after maxshift zeros; maxima of a few
    # beams / DM rows from the oracle on exactly that input
    import numpy as np
    import oracle
    rows = np.linspace(0, cfg.ndm - 1, 16).round().astype(np.int32)
    e2e_ok = True
    for b in (0, nb - 1):
        padded = np.concatenate([np.zeros((cfg.nchans, plan.max_shift), dtype=np.uint8), pool[0][b].numpy()], axis=1)
        ref = oracle.dedisperse(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, cfg.dm_list(), np.ascontiguousarray(padded), chunk, rows=rows)
        e2e_ok = e2e_ok and bool((ref.max(axis=1) == h_max[0, b].numpy()[rows]).all())
    assert e2e_ok, "streamed block 0 maxima differ from the oracle"
    e2e = {"value": adds * nchunks / et / 1e9, "unit": UNIT, "h2d_bytes_per_step": pool[0].numel(),
           "d2h_bytes_per_step": nb * cfg.ndm * 4, "steps": nchunks, "ms_per_step": 1e3 * et / nchunks,
           "real_time_factor": chunk * cfg.tsamp / (et / nchunks), "e2e_checked": e2e_ok,
           "api": f"dedisp_stream_push: {nchunks} consecutive chunks (pool of 3 pinned host chunks cycled, 3 device buffers); "
                  "D2H = per-(beam, DM) maxima of each block, read on a second stream and handed back with dedisp_stream_release_after"}
    return e2e


def _c5_line(args, cfg, plan, hbm_gbs, sm_max_mhz, peak_src, value, total_ms, step_ms, clocks, e2e, adds, nsamp_in):
    nb, chunk = cfg.nbeams, cfg.nsamp_out
    peak = add_peak(sm_max_mhz)
    achieved = adds / (step_ms * 1e-3) / 1e9
    kname = {1: "naive", 2: "tiled", 3: "subband"}[plan.kernel]
    bytes_once = nb * (cfg.nchans * nsamp_in + cfg.ndm * chunk * 4)
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": UNIT, "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_BYTES.get((cfg.name, kname)), "kernel": f"dedisp_{kname}_kernel",
                "launches_per_step": plan.launches_per_execute,
                "peak_source": f"148 SMs x 128 lanes x sm_max_mhz ({peak_src} MEASURED_PEAKS.json clock)",
                "hbm_bytes_once": bytes_once, "hbm_time_ms_at_peak": bytes_once / (hbm_gbs * 1e9) * 1e3}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "i32", "data": "synthetic",
            "config": {"workload": cfg.name, "nchans": cfg.nchans, "ndm": cfg.ndm, "nsamp_out": chunk, "nbeams": nb,
                       "in_dtype": "u8", "l2": "input larger than L2, no flush", "kernel": kname,
                       "note": "step = one 32768-sample chunk of all 32 beams"},
            "real_time_factor": chunk * cfg.tsamp / (total_ms / args.steps * 1e-3),
            "clocks": clocks, "e2e": e2e, "gpu_launches": plan.launches_per_execute * args.steps,
            "roofline": roofline, "cpu_baseline": None}
    print(json.dumps(line), flush=True)


def run_time_major(args, cfg):
    """the same workload fed TIME-major with nbits-bit packed samples through
    dedisp_execute_time_major (corner turn + unpack fused into the staging step). value: input resident;
    e2e: pinned host block -> H2D -> execute -> D2H of the result. 1 GPU, one beam."""
    import torch

    import paper_1111_6399_b200 as P
    from paper_1111_6399_b200 import synth

    assert torch.cuda.is_available(), "bench.py needs a GPU: the product has no CPU path"
    assert cfg.dtype == "u8", "time-major input is integer data: use --config c2 or c5"
    nbits = args.time_major
    hbm_gbs, sm_max_mhz, peak_src = _peaks()
    plan = P.Plan.from_config(cfg, time_major=True)
    nsamp_in = cfg.nsamp_out + plan.max_shift
    x, _ = synth.make_input(cfg, plan.shifts(), nsamp_in, device="cuda")          # [c][t] u8
    q = (x >> (8 - nbits)).t().contiguous()                                       # [t][c], values < 2**nbits
    per = 8 // nbits
    packed = (q.view(nsamp_in, cfg.nchans // per, per).to(torch.int32) << (nbits * torch.arange(per, device="cuda", dtype=torch.int32))).sum(dim=2).to(torch.uint8)
    row = (packed.shape[1] + 15) // 16 * 16
    raw = torch.zeros((nsamp_in, row), dtype=torch.uint8, device="cuda")
    raw[:, :packed.shape[1]] = packed
    del x, q, packed
    out = plan.alloc_out(cfg.nsamp_out)
    adds = cfg.ndm * cfg.nchans * cfg.nsamp_out
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        plan.execute_time_major(raw, nbits, cfg.nsamp_out, out)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(0)
    torch.cuda.synchronize()
    sampler.start()
    for a, b in evs:
        a.record(stream)
        plan.execute_time_major(raw, nbits, cfg.nsamp_out, out)
        b.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    total_ms = evs[0][0].elapsed_time(evs[-1][1])
    steps = sorted(a.elapsed_time(b) for a, b in evs)
    step_ms = sum(steps) / len(steps)
    e2e = None
    if not args.no_e2e:
        h_raw = raw.cpu().pin_memory()
        h_out = torch.empty((cfg.ndm, cfg.nsamp_out), dtype=torch.int32, pin_memory=True)
        esteps = max(1, min(args.steps, args.e2e_steps))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(esteps):
            raw.copy_(h_raw, non_blocking=True)
            plan.execute_time_major(raw, nbits, cfg.nsamp_out, out)
            h_out.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        et = time.perf_counter() - t0
        e2e = {"value": adds * esteps / et / 1e9, "unit": UNIT, "h2d_bytes_per_step": h_raw.numel(),
               "d2h_bytes_per_step": h_out.numel() * 4, "steps": esteps, "ms_per_step": 1e3 * et / esteps,
               "api": "pinned host block -> H2D -> dedisp_execute_time_major -> D2H"}
    peak = add_peak(sm_max_mhz)
    achieved = adds / (step_ms * 1e-3) / 1e9
    bytes_once = raw.numel() + cfg.ndm * cfg.nsamp_out * 4
    line = {"metric": METRIC, "value": adds * args.steps / (total_ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "i32", "data": "synthetic",
            "config": {"workload": cfg.name + f"_time_major_{nbits}bit", "nchans": cfg.nchans, "ndm": cfg.ndm, "nsamp_out": cfg.nsamp_out,
                       "nsamp_in": nsamp_in, "in_dtype": f"u{nbits} packed, time-major [t][c], row {row} bytes", "kernel": "subband",
                       "passes": plan.num_subbands(), "l2": "out larger than L2, no flush"},
            "real_time_factor": cfg.nsamp_out * cfg.tsamp / (total_ms / args.steps * 1e-3),
            "clocks": clocks, "e2e": e2e, "gpu_launches": plan.launches_per_execute * args.steps,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": UNIT, "frac": achieved / peak, "traffic": None,
                         "kernel": "dedisp_subband_kernel (time-major staging)", "launches_per_step": plan.launches_per_execute,
                         "peak_source": f"148 SMs x 128 lanes x sm_max_mhz ({peak_src} MEASURED_PEAKS.json clock)",
                         "hbm_bytes_once": bytes_once, "ms_median": steps[len(steps) // 2], "ms_best": steps[0]},
            "cpu_baseline": None}
    print(json.dumps(line), flush=True)


def run_detect(args, cfg):
    """dedisp_detect on the de-dispersed block of the config (c5: 32 beams x 1024 DMs x
    32768 samples int32 = 4.3 GB; c3: 4096 x 131072 fp32 = 2.1 GB), which stays on the GPU. HBM-bound: the block is
    read twice (row statistics, then boxcar + threshold); roofline = 2 x block bytes / measured HBM bandwidth."""
    import ctypes
    import torch

    import paper_1111_6399_b200 as P
    from paper_1111_6399_b200 import synth

    assert torch.cuda.is_available(), "bench.py needs a GPU: the product has no CPU path"
    hbm_gbs, _, _ = _peaks()
    plan = P.Plan.from_config(cfg)
    nsamp_in = cfg.nsamp_out + plan.max_shift
    tab = plan.shifts()
    if cfg.nbeams > 1:
        x = torch.empty((cfg.nbeams, cfg.nchans, nsamp_in), dtype=torch.uint8, device="cuda")
        for b in range(cfg.nbeams):
            x[b], _ = synth.make_input(cfg, tab, nsamp_in, device="cuda", seed=cfg.seed * 1000003 + b * 101)
        out = plan.execute(x, cfg.nsamp_out)
    else:
        x, _ = synth.make_input(cfg, tab, nsamp_in, device="cuda")
        out = plan.execute(x, cfg.nsamp_out)
    torch.cuda.synchronize()
    del x
    block = out.view(-1, cfg.nsamp_out)
    rows, n = block.shape
    nwidths, thr, max_cands = 6, 7.0, 1 << 20
    L = P.lib()
    work = torch.empty(int(L.dedisp_detect_workspace_bytes(rows)) // 8 + 1, dtype=torch.int64, device="cuda")
    cands = torch.empty(max_cands * P.CAND_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def call():
        rc = L.dedisp_detect(block.data_ptr(), int(block.dtype == torch.float32), rows, n, block.stride(0), nwidths, thr,
                             cands.data_ptr(), max_cands, work.data_ptr(), ctypes.c_void_p(stream.cuda_stream))
        assert rc == 0

    for _ in range(args.warmup):
        call()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(0)
    torch.cuda.synchronize()
    sampler.start()
    for a, b in evs:
        a.record(stream)
        call()
        b.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    steps = sorted(a.elapsed_time(b) for a, b in evs)
    step_ms = sum(steps) / len(steps)
    total = int(work[0].item())
    t0 = time.perf_counter()
    esteps = max(1, min(args.steps, args.e2e_steps))
    for _ in range(esteps):
        got, tot = P.detect(block, nwidths, thr, max_cands)       # call + sync + candidates copied to the host
    et = (time.perf_counter() - t0) / esteps
    nbytes = rows * n * 4
    algo = 2 * nbytes
    line = {"metric": "detection throughput (de-dispersed samples/s)", "value": rows * n / (step_ms * 1e-3) / 1e9, "unit": "Gsamples/s",
            "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "i32" if block.dtype == torch.int32 else "f32", "data": "synthetic",
            "config": {"workload": cfg.name + "_detect", "rows": rows, "nsamp": n, "nwidths": nwidths, "threshold_sigma": thr,
                       "candidates": total, "l2": "block larger than L2, no flush"},
            "clocks": clocks,
            "e2e": {"value": rows * n / et / 1e9, "unit": "Gsamples/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 8 + len(got) * P.CAND_DTYPE.itemsize, "ms_per_step": 1e3 * et,
                    "api": "dedisp_detect on the resident block + D2H of the count and the candidate list"},
            "gpu_launches": 2 * args.steps,
            "roofline": {"bound": "hbm", "achieved": algo / (step_ms * 1e-3) / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                         "frac": algo / (step_ms * 1e-3) / 1e9 / hbm_gbs, "traffic": None,
                         "kernel": "dedisp_detect_stats_kernel + dedisp_detect_boxcar_kernel", "algorithmic_bytes": algo,
                         "ms_median": steps[len(steps) // 2], "ms_best": steps[0]},
            "cpu_baseline": None}
    print(json.dumps(line), flush=True)


def run_paper_sweep(args):
    """the paper's Fig. 4 regime (ndm = nchans) as a second workload; one
    JSON line per point, with the paper's own axis ("execution time as percentage of real-time")."""
    import torch

    import paper_1111_6399_b200 as P
    from paper_1111_6399_b200 import paper_sweep, synth

    assert torch.cuda.is_available(), "bench.py needs a GPU: the product has no CPU path"
    _, sm_max_mhz, _ = _peaks()
    peak = N_SM * LANES_PER_SM * sm_max_mhz * 1e6 / 1e9
    points = [(n, 200.0) for n in (250, 500, 1000, 2000, 4000)] + [(2000, dm) for dm in (50.0, 100.0, 400.0, 800.0)]
    for nchans, max_dm in points:
        cfg = paper_sweep(nchans, max_dm)
        plan = P.Plan.from_config(cfg)
        if args.kernel:
            try:
                plan.set_kernel({"naive": 1, "tiled": 2, "subband": 3}[args.kernel])
            except P.DedispError:
                continue
        x, _ = synth.make_input(cfg, plan.shifts(), cfg.nsamp_out + plan.max_shift, device="cuda")
        out = plan.alloc_out(cfg.nsamp_out)
        for _ in range(args.warmup):
            plan.execute(x, cfg.nsamp_out, out)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            plan.execute(x, cfg.nsamp_out, out)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        adds = cfg.ndm * cfg.nchans * cfg.nsamp_out
        print(json.dumps({"workload": cfg.name, "nchans": nchans, "ndm": cfg.ndm, "max_dm": max_dm, "nsamp_out": cfg.nsamp_out,
                          "passes": plan.num_subbands(), "kernel": plan.kernel, "ms_per_step": ms,
                          "pct_of_real_time": 100.0 * ms * 1e-3 / (cfg.nsamp_out * cfg.tsamp),
                          "gadds_per_s": adds / ms / 1e6, "frac_of_add_peak": adds / ms / 1e6 / peak}), flush=True)
        del x, out, plan
        torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--sweep", default=None, choices=["paper"])
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c3", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--kernel", default=None, choices=["naive", "tiled", "subband"])
    ap.add_argument("--merge-passes", action="store_true", help="fp plans: all SUBBAND passes in one launch (not bit-reproducible)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-seconds", type=float, default=3.0, help="cpu_baseline: oracle seconds per timed call")
    ap.add_argument("--no-others", action="store_true", help="skip the c2/c4/c5 block of the default line")
    ap.add_argument("--time-major", type=int, default=0, choices=[0, 1, 2, 4, 8],
                    help="feed the (u8) config time-major with this many bits per sample (dedisp_execute_time_major)")
    ap.add_argument("--detect", action="store_true", help="time dedisp_detect on the config's de-dispersed block (c3 or c5)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--stream-chunks", type=int, default=0, help="c5 e2e: chunks pushed (default: the config's 60)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    world_env = os.environ.get("WORLD_SIZE")
    if args.gpus > 1 and world_env is None and args.impl == "ours":
        # plain `python bench.py --gpus N`: start the N ranks ourselves, one process per GPU
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if world_env is not None and args.impl == "ours" and int(world_env) != args.gpus:
        sys.exit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world_env}")
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    from paper_1111_6399_b200 import CONFIGS
    cfg = CONFIGS[args.config]
    if args.sweep:
        run_paper_sweep(args)
    elif args.impl == "reference":
        run_reference(args, cfg)
    elif args.detect:
        run_detect(args, cfg)
    elif args.time_major:
        run_time_major(args, replace(cfg, nbeams=1, nchunks=1))
    elif args.config == "c5":
        run_c5_stream(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
