"""bench.py --gpus N is "replicas only": no data-path collective, the only cross-rank step is the
maximum of the per-rank times.  That host logic is exercised here with two gloo ranks on CPU."""
import os
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _rank(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(dist, 1.5 if rank == 0 else 2.5, "cpu")      # rank 1 is the slow replica
    out[rank] = (ms, bench.aggregate_value(world, 10 ** 9, ms))
    dist.destroy_process_group()


def test_two_ranks_take_the_slowest_time_and_sum_the_bytes():
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_rank, args=(2, 29611, out), nprocs=2, join=True)
        assert out[0] == out[1] == (2.5, 2 * 10 ** 9 / 2.5e-3 / 1e9)


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(None, 3.25, "cpu") == 3.25
    assert bench.aggregate_value(1, 1 << 30, 1.0) == (1 << 30) / 1e-3 / 1e9
