"""Worker of tests/test_multirank_gloo.py: one of WORLD_SIZE processes on the gloo backend (no GPU).

Exercises the host side of `bench.py --gpus N`: rendezvous, one independent box per rank (weak scaling, no
data-path collective), max-over-ranks time, whole-job particle count.
"""
import hashlib
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np
import torch.distributed as dist

import bench
import paper_2606_23891_b200 as sph


def main():
    rank, world, local = bench.dist_setup(int(os.environ["WORLD_SIZE"]))
    assert dist.get_backend() == "gloo"
    ps, cells, tasks = bench.build_config1(sph, seed=1 + rank)
    digest = hashlib.sha256(ps.view(np.uint8).tobytes()).hexdigest()
    digests = [None] * world
    dist.all_gather_object(digests, digest)
    bench.dist_barrier(world)
    ms = bench.dist_max(1.0 + rank, world)           # the slowest rank defines the step
    total = bench.dist_sum(float(ps.shape[0]), world)
    if rank == 0:
        print(json.dumps({"world": world, "digests": digests, "ms": ms, "total": total, "n": int(ps.shape[0]),
                          "tasks": int(tasks.shape[0])}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
