"""N > 1 is "replicas only": no data-path collective, only the
contract's barrier + max-over-ranks timing.  World-size-2 gloo test of that plumbing on CPU."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    from paper_2606_09061_b200 import workloads as wl
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.dist_env() == (rank, rank, world)
    spec = wl.config_tiny(seed=rank)                      # each replica draws its own batch
    ms_local = 10.0 + 5.0 * rank                          # rank 1 is the slow replica
    dist.barrier()
    ms = bench.max_over_ranks(ms_local)
    rate = bench.whole_job_rate(spec.T, 4, world, ms)
    q.put((rank, ms, rate, [bt.tolist() for bt in spec.block_tables]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_replicas_world2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=150) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, ms0, rate0, bt0), (_, ms1, rate1, bt1) = res
    assert ms0 == ms1 == 15.0                              # max over ranks on both
    assert rate0 == rate1 == 2 * 50 * 4 / 15e-3            # whole-job tokens/s: both replicas' tokens
    assert bt0 != bt1                                      # independent replicas, own seeds


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_rate(2048, 10, 1, 10.0) == 2048 * 10 / 10e-3
