"""Host-side logic of bench.py that runs with more than one rank (replicas only, no data-path collective):
the max-over-ranks timing reduction and the whole-job throughput, on the CPU with the gloo backend and world size 2."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms, e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 3.0 - rank], dist)       # rank 1 is the slow one on the first entry
        val = bench.job_value(1000.0, 4, world, ms)
        out.put((rank, ms, e2e, val))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for rank, ms, e2e, val in res:
        assert ms == 15.0 and e2e == 3.0                      # both ranks see the maximum
        assert val == pytest.approx(2 * 1000.0 * 4 / 15.0e-3)   # units of ALL ranks over the slowest rank's time


def test_single_process_passthrough():
    import bench
    assert bench.max_over_ranks([1.5, 2.5], None) == [1.5, 2.5]
    assert bench.job_value(10.0, 3, 1, 2.0) == pytest.approx(10.0 * 3 / 2.0e-3)


def test_reference_arm_runs_only_on_rank_zero(capsys):
    import argparse
    import bench
    args = argparse.Namespace(workload="config0", steps=1, warmup=0, gpus=2)
    bench.run_reference(args, rank=1, world=2)
    assert capsys.readouterr().out == ""
