"""Worker of tests/test_gpu_parity.py::test_partitioning_across_ranks_two_processes: one rank of a 2-rank gradient with
one time partition per rank (paper_2605_06392_b200/partitioned.py).  Launched by torch.distributed.run; both ranks use
cuda:0 and the gloo backend (this box has one GPU; on a multi-GPU node the backend is nccl and LOCAL_RANK picks the GPU)."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np
import torch
import torch.distributed as dist


def main():
    ngpu = torch.cuda.device_count()
    local = int(os.environ.get("LOCAL_RANK", "0"))
    device = local if ngpu > local else 0
    backend = "nccl" if ngpu >= int(os.environ["WORLD_SIZE"]) else "gloo"
    dist.init_process_group(backend)
    torch.cuda.set_device(device)
    from oracle import bta_oracle as O
    from paper_2605_06392_b200 import BtaModel
    from paper_2605_06392_b200.partitioned import TorchCollectives, value_and_grad
    from workloads import make_config
    model, obs, th = make_config(1, nt=12, m_per_var=4000)
    ref = O.value_and_grad(model, obs, th)
    M = BtaModel.from_workload(model, obs, device=device)
    M.bta_set_partitions(dist.get_world_size())
    coll = TorchCollectives()
    f, g = value_and_grad(M, th, coll)
    f2, g2 = value_and_grad(M, th, coll)
    M.close()
    gate = np.maximum(np.abs(ref["grad"]), 1e-3 * np.max(np.abs(ref["grad"])))
    ok = (abs(f - ref["f"]) <= 1e-9 * abs(ref["f"]) and bool(np.all(np.abs(g - ref["grad"]) <= 1e-6 * gate))
          and f2 == f and bool(np.array_equal(g, g2)))
    # one write call per rank, newline on both sides (the ranks share a pipe)
    sys.stdout.write("\n" + json.dumps({"rank": dist.get_rank(), "f": f, "grad": g.tolist(), "ok": bool(ok),
                                        "backend": backend}) + "\n")
    sys.stdout.flush()
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
