"""Worker of tests/test_gpu_sharded.py::test_two_processes_over_cuda_ipc, launched by
torch.distributed.run with 2 ranks on one GPU: each rank is one member of a distributed-Hamiltonian
group (gamma slice of L, 6 own walkers), 3 steps + local energy; rank 0 gathers and saves."""
from __future__ import annotations

import os
import sys

import numpy as np


def main(out_path):
    import torch
    import torch.distributed as dist

    from paper_2406_16238_b200 import inputs, sharded

    dist.init_process_group("gloo")
    rank, G = dist.get_rank(), dist.get_world_size()
    torch.cuda.set_device(0)
    nw, steps = 6, 3
    cfg, h1, L, trial, walkers = inputs.make_problem_host("c1", nw=G * nw)
    slices = sharded.gamma_slices(cfg.n_chol, G)
    a, b = slices[rank]
    Ld = torch.from_numpy(np.ascontiguousarray(L[a:b])).cuda()
    grp = sharded.DistGroup(h1, Ld, trial, slices, M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta,
                            max_walkers=nw, walker_kind=cfg.walker_kind, taylor_order=cfg.taylor_order)
    W = torch.from_numpy(np.ascontiguousarray(walkers[rank * nw:(rank + 1) * nw])).cuda()
    wt = torch.ones(nw, dtype=torch.float64, device="cuda")
    E = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")
    for s in range(steps):
        x = inputs.make_aux_fields(cfg, 0, s, G * nw)[rank * nw:(rank + 1) * nw]
        grp.step(W, wt, torch.from_numpy(np.ascontiguousarray(x)).cuda(), cfg.dt)
    grp.local_energy(W, E)
    grp.sync()
    parts = [None] * G
    dist.all_gather_object(parts, (W.cpu().numpy(), wt.cpu().numpy(), E.cpu().numpy()))
    if rank == 0:
        np.savez(out_path, W=np.concatenate([p[0] for p in parts]), wt=np.concatenate([p[1] for p in parts]),
                 E=np.concatenate([p[2] for p in parts]), steps=steps)
    grp.close()
    dist.destroy_process_group()


if __name__ == "__main__":
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    main(sys.argv[1])
