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


# ------------------------------------------------------------------ z-slab plumbing (slabs.py)
def _slab_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2403_15773_b200 import slabs
    res = {}
    for jet in (False, True):
        plan = slabs.neighbor_plan(rank, world, jet)
        z0, z1 = slabs.slab_ranges(21, world)[rank]
        lo, hi = slabs.gather_neighbors(("handle-of-%d" % rank, z1 - z0), plan, dist)
        res[jet] = (plan, (z0, z1), lo, hi)
    out.put((rank, res))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_slab_plan_and_handle_exchange():
    from paper_2403_15773_b200 import tslb
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_slab_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    # periodic z: both faces of both slabs are halo faces and see the other rank
    for r in (0, 1):
        plan, rng, lo, hi = res[r][False]
        assert plan["bc_zlo"] == plan["bc_zhi"] == tslb.BC_HALO and plan["lo"] == plan["hi"] == 1 - r
        assert lo == hi == ("handle-of-%d" % (1 - r), 10 if r == 0 else 11)
        assert rng == ((0, 11), (11, 21))[r]
    # jet: inflow on rank 0's low face, outflow on rank 1's high face, one shared face
    p0, _, lo0, hi0 = res[0][True]
    p1, _, lo1, hi1 = res[1][True]
    assert (p0["bc_zlo"], p0["bc_zhi"]) == (tslb.BC_JET_INFLOW, tslb.BC_HALO) and lo0 is None and hi0 == ("handle-of-1", 10)
    assert (p1["bc_zlo"], p1["bc_zhi"]) == (tslb.BC_HALO, tslb.BC_OUTFLOW) and hi1 is None and lo1 == ("handle-of-0", 11)


def test_slab_ranges_cover_the_domain():
    import pytest
    from paper_2403_15773_b200 import slabs
    for nz, n in ((1536, 8), (23, 3), (8, 4), (800, 7)):
        r = slabs.slab_ranges(nz, n)
        assert r[0][0] == 0 and r[-1][1] == nz and all(a[1] == b[0] for a, b in zip(r, r[1:]))
        w = [b - a for a, b in r]
        assert max(w) - min(w) <= 1 and min(w) >= 2
    with pytest.raises(ValueError):
        slabs.slab_ranges(7, 4)
    one = slabs.neighbor_plan(0, 1, False)          # a single periodic slab is its own neighbour
    assert one["lo"] == one["hi"] == 0
