"""World_size-2 gloo test (CPU) of the host side of the multi-rank time-domain partitioning
(paper_2605_06392_b200/partitioned.py): the order of the three phases, ONE all-gather of the slabs
in rank order, ONE all-reduce of the partial sums, the same result on every rank.  The compute phases are the C-ABI
calls inla_part_* (GPU only); here a stand-in with the same three methods records what the orchestration hands it.
The real thing runs in tests/test_gpu_parity.py::test_partitioning_across_ranks_*."""
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


class _StandIn:
    """Has the three phase methods of BtaModel; no method arithmetic -- slabs and partial sums are index patterns."""
    SLAB, NPART = 7, 5

    def __init__(self):
        self.calls = []

    def inla_part_phase1(self, theta, rank, nranks):
        self.calls.append(("phase1", rank, nranks))
        return torch.arange(self.SLAB, dtype=torch.float64) + 100.0 * rank + float(np.sum(theta))

    def inla_part_phase2(self, rank, nranks, gathered):
        self.calls.append(("phase2", rank, nranks))
        self.gathered = gathered.clone()
        return torch.full((self.NPART,), float(rank + 1), dtype=torch.float64) * torch.arange(1, self.NPART + 1)

    def inla_part_finish(self, partials):
        self.calls.append(("finish",))
        return float(partials.sum()), partials.numpy().copy()


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2605_06392_b200.partitioned import TorchCollectives, value_and_grad
    coll = TorchCollectives()
    m = _StandIn()
    theta = np.array([0.25, 0.25])
    f, g = value_and_grad(m, theta, coll)
    out.put((rank, m.calls, m.gathered.tolist(), f, g.tolist(), coll.world))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_gloo_orchestration():
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
    for rank, calls, gathered, f, g, world in res:
        assert world == 2
        assert calls == [("phase1", rank, 2), ("phase2", rank, 2), ("finish",)]
        # the slabs of rank 0 and rank 1, in rank order, on every rank
        want = [i + 0.5 for i in range(7)] + [i + 100.5 for i in range(7)]
        assert gathered == want
        # partial sums added over ranks: (1 + 2) * [1..5]
        assert g == [3.0, 6.0, 9.0, 12.0, 15.0] and f == 45.0
    assert res[0][3:5] == res[1][3:5]


def test_exchange_volume_formula():
    """(4P-2) b^2 + (2P-1)(a+1) b + a^2 + d + 1 distinct doubles per gradient; our slabs (two matrices,
    three b x b blocks each per rank) stay within a small constant of it."""
    from paper_2605_06392_b200.partitioned import exchange_doubles
    P, b, a, d = 4, 400, 4, 4
    assert exchange_doubles(P, b, a, d) == 14 * 160000 + 7 * 5 * 400 + 16 + 4 + 1
    ours = P * (2 * (3 * b * b + a * (a + 1)) + 2 * (a + 1) * b)
    assert ours < 2 * exchange_doubles(P, b, a, d)
