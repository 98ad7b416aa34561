"""world_size-2 gloo test of the N > 1 timing plumbing (barrier + max over ranks)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1309_1894_b200.dist import make_dist_max, whole_job_value


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    f = make_dist_max(torch, world, "cpu")
    q.put((rank, f(1.0 + rank), f(0.0)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(120)
        assert p.exitcode == 0
    assert got == [(0, 2.0, 0.0), (1, 2.0, 0.0)]


def test_identity_and_value():
    assert make_dist_max(torch, 1, "cpu")(3.5) == 3.5
    assert whole_job_value(10.0, 4, 2.0) == 20.0
