"""Multi-rank form of the time-domain partitioning (§III-C a-b; include/bta.h: inla_part_*).

One process per GPU; rank r owns partition r.  The library does the three compute phases; this module moves the two
device buffers between them with torch.distributed -- ONE all-gather of the boundary slabs and ONE all-reduce of the
partial sums per gradient, the paper's communication pattern, over NCCL/NVLink on GPUs instead of the
paper's CPU-staged MPI.  No arithmetic of the method happens here.
"""
from __future__ import annotations


class TorchCollectives:
    """all_gather / all_reduce on a torch.distributed process group (NCCL on GPUs; gloo stages through the host)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank = dist.get_rank(group)
        self.world = dist.get_world_size(group)
        self.backend = dist.get_backend(group)

    def all_gather(self, slab):
        import torch
        if self.backend == "gloo" and slab.is_cuda:          # gloo moves host memory: stage the slab
            host = slab.cpu()
            out = torch.empty(self.world * host.numel(), dtype=host.dtype)
            self.dist.all_gather_into_tensor(out, host, group=self.group)
            return out.to(slab.device)
        out = torch.empty(self.world * slab.numel(), dtype=slab.dtype, device=slab.device)
        self.dist.all_gather_into_tensor(out, slab, group=self.group)
        return out

    def all_reduce_(self, partials):
        if self.backend == "gloo" and partials.is_cuda:
            host = partials.cpu()
            self.dist.all_reduce(host, group=self.group)
            partials.copy_(host)
            return partials
        self.dist.all_reduce(partials, group=self.group)
        return partials


def exchange_doubles(P, b, a, d):
    """Distinct doubles the paper's collectives move per gradient: (4P-2) b^2 + (2P-1)(a+1) b + a^2 + d + 1."""
    return (4 * P - 2) * b * b + (2 * P - 1) * (a + 1) * b + a * a + d + 1


def value_and_grad(model, theta, coll):
    """f, grad f with one partition per rank.  `model`: a BtaModel (or anything with the three inla_part_* methods)
    prepared with bta_set_partitions(world); `coll`: TorchCollectives or an object with the same two methods."""
    slab = model.inla_part_phase1(theta, coll.rank, coll.world)          # Phase 1: no communication
    gathered = coll.all_gather(slab)                                     # the one exchange of boundary data
    partials = model.inla_part_phase2(coll.rank, coll.world, gathered)   # Phase 2 (redundant) + Phase 1'
    partials = coll.all_reduce_(partials)                                # the one reduction
    return model.inla_part_finish(partials)
