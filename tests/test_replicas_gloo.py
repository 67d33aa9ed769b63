"""world_size-2 gloo test of the only cross-rank step the path has: the timing reduction of the
"replicas only" multi-GPU mode (max of the elapsed time, sum of the work)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1406_6158_b200.replicas import aggregate, replica_seed
    from workloads import make_ic
    pos, _ = make_ic("plummer", 256, replica_seed(5, rank))
    t_ms, units, rate = aggregate(10.0 * (rank + 1), 1000.0 * (rank + 1))
    out.put((rank, t_ms, units, rate, float(pos[:, 0].sum())))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_two_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for _, t_ms, units, rate, _ in res:
        assert t_ms == 20.0 and units == 3000.0            # slowest rank, work of both
        assert rate == pytest.approx(3000.0 / 0.020)
    assert res[0][4] != res[1][4]                           # independent replicas: different seeds


def test_aggregate_single_process():
    from paper_1406_6158_b200.replicas import aggregate
    assert aggregate(4.0, 8.0) == (4.0, 8.0, 2000.0)
