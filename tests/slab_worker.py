"""One rank of the cross-process slab test (tests/test_slabs_gpu.py): builds its slab of a seeded
workload, maps the neighbour's workspace with CUDA IPC, advances, writes its fields.

    python tests/slab_worker.py RANK WORLD PORT CONFIG NX,NY,NZ STEPS OUT.npz
"""
import os
import sys


def main():
    rank, world, port, cfg = int(sys.argv[1]), int(sys.argv[2]), int(sys.argv[3]), int(sys.argv[4])
    shape = tuple(int(v) for v in sys.argv[5].split(","))
    steps, out = int(sys.argv[6]), sys.argv[7]
    import numpy as np
    import torch.distributed as dist
    from paper_2103_12819_b200 import workloads as wl
    from paper_2103_12819_b200.slabs import PERIODIC, DistSlab, cut_workload, plan_slabs
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.make_config(cfg, shape=shape)
    plan = plan_slabs(w.nz, world, w.bc[2] == PERIODIC)[rank]
    slab = DistSlab(cut_workload(w, plan), plan, "cuda:0")
    slab.step(steps)
    f = {k: v.numpy() for k, v in slab.sim.read_fields().items()}
    f["iters_total"] = np.int64(slab.sim.stats()["iters_total"])
    np.savez(out, **f)
    slab.close()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
