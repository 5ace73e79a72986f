"""Worker of tests/test_gpu_distributed.py: one rank of a DistributedLattice whose ranks SHARE cuda:0 (the only GPU
the tests have). Host ordering (su_synchronize + gloo barrier) replaces the stream-ordered NCCL all-reduce, which
NCCL refuses between two ranks on one device; everything else - CUDA IPC export / open of the neighbours' link
buffers, the fused peer-store halo push in the update kernels, su_slab_halo_push after the import, the ordering
after reunitarise - is the multi-GPU code path."""
import os
import sys

import numpy as np


def main():
    rank, world, port, tmp = int(sys.argv[1]), int(sys.argv[2]), sys.argv[3], sys.argv[4]
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import torch
    import torch.distributed as dist
    from paper_1112_4533_b200.slab import DistributedLattice

    # "shared" (default): every rank on cuda:0, gloo, host ordering. "multi": rank r on cuda:r, NCCL, the stream-ordered
    # all-reduce between sub-steps and peer stores that really cross NVLink (needs >= world GPUs)
    multi = len(sys.argv) > 5 and sys.argv[5] == "multi"
    dev = rank if multi else 0
    torch.cuda.set_device(dev)
    if multi:
        dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world,
                                device_id=torch.device("cuda", dev))
    else:
        dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    cfg = np.load(os.path.join(tmp, "cfg.npy"), allow_pickle=True).item()
    start = np.load(os.path.join(tmp, "start.npy"))
    D = DistributedLattice(cfg["Nc"], cfg["dims"], cfg["precision"], cfg["recon12"], cfg["kernel"], device=dev,
                           order="nccl" if multi else "host")
    lt = cfg["dims"][3] // world
    D.import_links(start[rank * lt:(rank + 1) * lt])
    D.sweep_counter, D.seed = cfg["sweep0"], cfg["seed"]
    D.lat.set_rng(cfg["seed"], cfg["sweep0"])
    D.sweep(cfg["beta"], 1, 4)
    np.save(os.path.join(tmp, f"after1_{rank}.npy"), D.export_links())
    plaq = D.plaquette()
    # sweep -> reunitarise -> sweep with nothing in between (reunitarise rewrites the halos)
    D.reunitarize()
    D.sweep(cfg["beta"], 1, 2)
    D.reunitarize()
    D.sweep(cfg["beta"], 0, 1)
    np.save(os.path.join(tmp, f"after2_{rank}.npy"), D.export_links())
    if rank == 0:
        np.save(os.path.join(tmp, "plaq.npy"), np.array([plaq]))
    D.close()
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
