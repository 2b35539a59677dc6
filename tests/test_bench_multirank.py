"""The N > 1 path of bench.py is "replicas only": no data-path collective, timing = max over
ranks, value = sum of the replicas' units / that time.  Covered here with world_size-2 gloo processes on CPU."""
import os
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")       # rank 1 is the slow replica
    dist.barrier()
    out[rank] = ms
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, 29731, out), nprocs=2, join=True)
        assert out[0] == out[1] == 15.0


def test_reference_arm_and_bytes_accounting():
    sys.path.insert(0, ROOT)
    import bench
    # B_mat(N) = 16 N (N + 1) / 2
    assert abs(bench.alg_bytes(98304, 0) - 77.310e9) < 1e7
    assert bench.alg_bytes(16384, 4) == 16.0 * 16384 * 16385 / 2 + 32.0 * 16384 * 4
    assert bench.max_over_ranks(3.0, None, "cpu") == 3.0
