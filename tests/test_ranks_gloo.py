"""N > 1 host logic of bench.py on CPU: two gloo ranks (world_size 2, 127.0.0.1).

The path does not shard (replicas only), so the only multi-rank logic is the
aggregation "time = max over ranks, units = sum over ranks" and the rule that every rank takes its own
cloud (seed + rank).  No GPU, no CUDA library call.
"""
from __future__ import annotations

import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r measured (10 + 5 r) ms over (100 + r) units
        ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 100.0 + rank, "cpu")
        dist.barrier()
        out.put((rank, ms, units))
    finally:
        dist.destroy_process_group()


def test_time_is_max_and_units_are_summed_over_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, units in got:
        assert ms == 15.0, "time must be the max over ranks"
        assert units == 201.0, "units must be summed over ranks"
    # whole-job throughput from the aggregated pair
    import bench
    assert bench.throughput(201.0, 15.0) == 201.0 / 0.015


def test_single_process_aggregation_is_identity():
    import bench
    assert bench.aggregate_over_ranks(3.5, 7.0) == (3.5, 7.0)


def test_every_rank_rasterises_its_own_cloud():
    # replicas: rank r uses seed + r, so two ranks never time the same point cloud
    from paper_2403_16862_b200.workloads import make_workload
    a = make_workload("tiny", seed=0)
    b = make_workload("tiny", seed=1)
    assert a.pos.shape == b.pos.shape and not (a.pos == b.pos).all()
