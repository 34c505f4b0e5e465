"""N > 1 is N independent replicas; the cross-rank timing logic of bench.py (barrier, MAX over ranks, whole-job
throughput) is covered here with two CPU processes over gloo."""
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
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2512_20276_b200 import replicas as R
    R.barrier()
    ms = [10.0 + 5.0 * rank, 30.0 - 3.0 * rank]              # rank 1 is slower on the first, faster on the second
    mx = R.max_over_ranks(ms)
    fps = R.whole_job_throughput(steps=20, ms_max=mx[0])
    R.barrier()
    out.put((rank, mx, fps, R.world()))
    dist.destroy_process_group()


def test_two_replicas_report_max_time_and_summed_throughput():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, fps, world in res:
        assert world == 2
        assert mx == [15.0, 30.0]                            # MAX over ranks, identical on every rank
        assert abs(fps - 2 * 20 / 0.015) < 1e-6              # both replicas' frames over the slowest rank's time


def test_single_process_is_a_no_op():
    from paper_2512_20276_b200 import replicas as R
    assert R.world() == 1
    R.barrier()
    assert R.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert R.whole_job_throughput(10, 100.0) == 100.0
