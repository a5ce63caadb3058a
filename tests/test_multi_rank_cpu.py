"""-m "not gpu": the N>1 host logic of bench.py on CPU, 2 ranks over gloo.

The path shards by beam with no data-path collective; what N>1 adds is (1) a distinct seeded beam
per rank, (2) the max-over-ranks time and (3) the whole-job aggregate. Two real processes
rendezvous on 127.0.0.1 and check each of them; the per-rank work is a host-only plan (table build,
sub-band records) so the plan layer is exercised in every rank without a GPU.
"""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        import paper_1111_6399_b200 as P
        from paper_1111_6399_b200 import CONFIGS, synth

        cfg = CONFIGS["c1"]
        plan = P.Plan.from_config(cfg, host_only=True)          # every rank builds the same plan
        x, _ = synth.make_input(cfg, plan.shifts(), cfg.nsamp_out + plan.max_shift, device="cpu",
                                seed=bench.beam_seed(cfg.seed, rank))
        # (1) beams differ between ranks, plans do not
        sums = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(sums, x.double().sum().reshape(1))
        shifts = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(shifts, torch.tensor([int(plan.shifts().sum())]))
        # (2) max over ranks: rank r "took" (r + 1) seconds
        slowest = bench.max_over_ranks(float(rank + 1), world, device="cpu")
        # (3) whole-job value
        val = bench.job_value(1_000_000_000, 2, world, slowest)
        dist.barrier()
        out.put((rank, [float(s) for s in sums], [int(s) for s in shifts], slowest, val))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_host_logic():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, sums, shifts, slowest, val in res:
        assert sums[0] != sums[1], "each rank must de-disperse its own beam"
        assert shifts[0] == shifts[1], "every rank builds the same shift table"
        assert slowest == 2.0                                    # the slowest rank's time, on every rank
        assert val == world * 1e9 * 2 / 2.0 / 1e9                # 2 ranks x 2 steps x 1e9 adds in 2 s = 2 Gadds/s
