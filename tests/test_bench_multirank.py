"""CPU-only, world_size 2 over gloo: the only cross-rank step of `bench.py --gpus N` (replicas only) is the
reduction of per-rank timings into the whole-job number - max over ranks for time, sum over ranks for units."""
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
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [120.0, 150.0][rank]            # rank 1 is the slow replica
    units = [24576.0, 6144.0][rank]      # replicas may differ in size
    ms_max = bench.over_ranks(ms, "max", "cpu")
    units_all = bench.over_ranks(units, "sum", "cpu")
    out[rank] = (ms_max, units_all, bench.job_throughput(units_all, 3, ms_max))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_reduction_over_gloo():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        ms_max, units_all, value = res[rank]
        assert ms_max == 150.0 and units_all == 30720.0
        assert abs(value - 30720.0 * 3 / 0.150) < 1e-6


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.over_ranks(3.5, "max", "cpu") == 3.5
    assert bench.job_throughput(100.0, 2, 50.0) == 4000.0
