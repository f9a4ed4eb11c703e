"""world_size-2 gloo test (CPU) of the N > 1 bookkeeping bench.py uses: barrier, MAX over ranks of
the timed region, whole-job throughput = units of all ranks / slowest rank's time."""
import os
import socket

import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2403_15773_b200 import dist as d
    d.barrier()
    ms = [12.5, 17.25][rank]                  # rank 1 is the slow one
    units = [1000.0, 1000.0][rank]            # replicas: same units per rank (weak scaling)
    tmax = d.max_over_ranks(ms)
    thr = d.job_throughput(units, ms * 1e-3)
    out.put((rank, d.world(), tmax, thr))
    d.barrier()
    dist.destroy_process_group()


def test_two_rank_timing_protocol():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, world, tmax, thr in res:
        assert world == 2
        assert tmax == 17.25
        assert abs(thr - 2000.0 / 17.25e-3) < 1e-6


def test_single_process_is_identity():
    from paper_2403_15773_b200 import dist as d
    assert d.world() == 1
    assert d.max_over_ranks(3.5) == 3.5
    assert d.job_throughput(10.0, 2.0) == 5.0
