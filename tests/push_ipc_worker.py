"""Worker of tests/test_gpu_halo.py::test_push_mode_between_two_processes: one rank of a 2-rank decomposition in push
mode, the neighbour's halo buffers opened through CUDA IPC.  Both ranks use cuda:0 (this box has one GPU; no kernel
waits on another: a host barrier separates the stages); the process group is gloo and carries only the IPC handles, the
barriers and the wavespeed maximum.  Prints OK when this rank's block equals the single-context run bit for bit."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2006_15698_b200 import DG                         # noqa: E402
from paper_2006_15698_b200 import decomposed as D            # noqa: E402
from paper_2006_15698_b200 import inputs as I                # noqa: E402


def main():
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n, p, ext, G = (6, 5, 4), 3, (1.0, 0.9, 0.8), 1.4
    procs = (2, 1, 1) if world == 2 else (world, 1, 1)
    q = I.density_wave(*n, p, ext, vel=(0.5, -0.3, 0.2), noise=5e-2, seed=9, waves=(1, 2, 1))
    variant = D.choose_variant(D.Decomposition(n, procs), p, D.variant_shapes(p))
    me = D.DistributedDG(n, p, G, ext, procs, rank, device="cuda:0", variant=variant, push=True)
    (x0, x1), (y0, y1), (z0, z1) = me.box
    me.set_state(np.ascontiguousarray(q[z0:z1, y0:y1, x0:x1]))
    lam = me.max_wavespeed()
    dt = I.cfl_dt(lam, p, ext, n, 0.1)
    r_loc = me.residual()
    me.rk_step(dt, 2)
    q_loc = me.get_state()
    single = DG(*n, p, G, ext, variant=variant).set_state(q)
    assert abs(single.max_wavespeed() - lam) <= 4e-16 * lam
    assert np.array_equal(r_loc, single.residual()[z0:z1, y0:y1, x0:x1]), "residual differs"
    assert np.array_equal(q_loc, single.rk_step(dt, 2).get_state()[z0:z1, y0:y1, x0:x1]), "state differs"
    dist.barrier()
    me.close()
    single.close()
    dist.destroy_process_group()
    print(f"OK rank {rank}", flush=True)


if __name__ == "__main__":
    main()
