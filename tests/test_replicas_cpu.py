"""The timing protocol of bench.py's N > 1 path on CPU: two gloo processes -- barrier, MAX over
ranks, whole-job rate (paper_2103_12819_b200/replicas.py).  What the ranks run between the barriers
(z-slabs of one grid, tests/test_slabs_cpu.py and test_slabs_gpu.py) is not this file's subject."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2103_12819_b200.replicas import barrier, max_over_ranks, whole_job_rate
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    barrier()
    mine = 10.0 + 5.0 * rank            # rank 1 is the slow one
    slowest = max_over_ranks(mine)
    rate = whole_job_rate(1000, 4, slowest, world)
    barrier()
    q.put((rank, slowest, rate))
    dist.destroy_process_group()


def test_two_ranks_share_the_slowest_time_and_sum_the_work():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slowest, rate in got:
        assert slowest == 15.0                       # MAX over ranks, on every rank
        assert rate == 2 * 1000 * 4 / 15.0           # all ranks' cell updates / slowest time


def test_without_a_process_group_the_helpers_are_identities():
    from paper_2103_12819_b200.replicas import barrier, max_over_ranks, whole_job_rate
    barrier()
    assert max_over_ranks(3.5) == 3.5
    assert whole_job_rate(10, 2, 4.0, 1) == 5.0
