"""N > 1 path of bench.py on CPU: world_size 2, gloo.  The hot path does not shard ("replicas
only"): the only thing that crosses ranks is the timing -- MAX over ranks -- and the whole-job value is the sum of
the replicas' algorithmic bytes over the slowest rank's time.  This test runs that aggregation in two processes."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 3.0 + 2.0 * rank            # rank 1 is the slow replica
        ms = bench.max_over_ranks(dist, ms_local, "cpu")
        by = bench.bytes_iteration((32, 32, 32, 64), 16, 8)
        val = bench.replicas_value(world, by, ms)
        dist.barrier()
        out[rank] = (ms, val, by)
    finally:
        dist.destroy_process_group()


def test_replicas_timing_is_max_over_ranks_and_value_sums():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in (0, 1):
        ms, val, by = res[rank]
        assert ms == 5.0                                  # the slowest rank, on every rank
        assert abs(val - 2 * by / 5.0 * 1e-6) < 1e-9 * val  # two replicas' bytes over the max time


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(None, 1.25, "cpu") == 1.25
    assert bench.replicas_value(1, 2.0e9, 2.0) == 1000.0


def test_reference_arm_other_ranks_exit_without_work(monkeypatch):
    """--impl reference under torchrun: rank 0 alone runs; the other ranks return 0 and print nothing."""
    import bench
    monkeypatch.setenv("RANK", "1")

    class A:
        workload, warmup, steps, gpus = "cfg2", 0, 1, 2
    assert bench.run_reference(A) == 0
