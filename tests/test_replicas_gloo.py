"""The N > 1 path is "replicas only": world_size-2 gloo test of its host logic on CPU."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2605_06392_b200.replicas import aggregate_throughput, max_over_ranks, replica_thetas, world_size
    th = np.array([0.1, -0.2, 0.3, 0.0])
    pts = replica_thetas(th, rank, 3)
    ms = max_over_ranks([100.0 + 50.0 * rank, 7.0 - rank])
    val = aggregate_throughput(3, ms[0])
    out.put((rank, [p.tolist() for p in pts], ms, val, world_size()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, pts0, ms0, v0, w0), (r1, pts1, ms1, v1, w1) = res
    assert w0 == w1 == 2
    assert ms0 == ms1 == [150.0, 7.0]                       # max over ranks, same on both
    assert v0 == v1 == 2 * 3 / 0.150                         # whole-job throughput
    th = [0.1, -0.2, 0.3, 0.0]
    allpts = [None] * 6
    allpts[0::2], allpts[1::2] = pts0, pts1                  # dealt round-robin: global point q = rank + 2 i
    assert allpts[0] == th
    assert np.allclose(allpts[1], [0.105, -0.2, 0.3, 0.0]) and np.allclose(allpts[2], [0.095, -0.2, 0.3, 0.0])
    assert np.allclose(allpts[3], [0.1, -0.195, 0.3, 0.0]) and np.allclose(allpts[5], [0.1, -0.2, 0.305, 0.0])


def test_single_process_identity():
    from paper_2605_06392_b200.replicas import max_over_ranks, replica_thetas, world_size
    assert world_size() == 1
    assert max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    pts = replica_thetas(np.zeros(4), 0, 9)
    assert len(pts) == 9 and np.count_nonzero(pts[0]) == 0 and pts[8][3] == -5e-3
