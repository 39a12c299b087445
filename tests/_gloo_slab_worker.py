"""Worker of tests/test_slabs.py::test_slab_split_over_two_gloo_ranks: one box over WORLD_SIZE gloo processes (no GPU), the oracle as
the compute engine, the halo refresh and the final gather over torch.distributed."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np
import torch.distributed as dist

import oracle as orc
import sph_inputs as si
from orc_setup import raw_copy, sort_grid
from paper_2606_23891_b200 import slabs

GAMMA = float(np.float32(5.0 / 3.0))


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    orc.set_threads(2)
    ps, cells, tasks, _, _ = sort_grid(si.jittered_lattice(12, 5, jitter=0.6, sigma_v=0.3, h_spread=0.2, mass_spread=0.4, u_spread=0.3), 4)
    owner = slabs.partition(cells, world)
    prob = slabs.LocalProblem(cells, tasks, owner, rank)
    lp = prob.take(ps)
    orc.density_cycle(lp, prob.cells, prob.tasks)
    plan = slabs.HaloPlan(cells, tasks, owner, prob, rank)
    sent = slabs.exchange_fields(lp, prob, ("rho", "rho_dh", "wcount", "wcount_dh"), plan, dist)
    orc.ghost(lp, GAMMA)
    orc.force_cycle(lp, prob.cells, prob.tasks)
    got = slabs.gather_owned(lp, prob, np.zeros_like(ps), dist)
    owned = [None] * world
    dist.all_gather_object(owned, int(prob.owned.sum()))
    if rank == 0:
        ref = raw_copy(ps)
        orc.density_cycle(ref, cells, tasks)
        orc.ghost(ref, GAMMA)
        orc.force_cycle(ref, cells, tasks)
        same = bool(np.array_equal(got.view(np.uint8).reshape(-1, 128)[:, :108], ref.view(np.uint8).reshape(-1, 128)[:, :108]))
        print(json.dumps({"world": world, "identical": same, "n": int(ps.shape[0]), "owned": owned, "halo_particles": int((~prob.owned).sum()),
                          "sent_bytes": sent, "n_send": plan.n_send, "n_recv": plan.n_recv}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
