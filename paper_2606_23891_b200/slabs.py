"""One box spread over several GPUs: slabs of cells with one layer of halo cells.

The path shards naturally: tasks only read inputs and reduce into per-particle outputs.  The cell table is cut into
`world` contiguous ranges of about equal particle counts ("slabs"); rank r OWNS the particles of its cells, keeps every
task that has at least one owned side, and so also holds the cells on the other side of those tasks ("halo").  It runs
the ordinary pack -> loop -> unpack cycle over its local tasks; the results of owned particles are complete and are, bit
for bit, those of the undivided box (every task that touches an owned cell is kept, in the same order, so the ordered
reduction of the unpack sees the same records in the same order); the results of halo particles are partial and are
never read.  Between the loops one exchange step refreshes the halo particles' fields from their owners (rho, rho_dh
before the ghost and the force loop).  Boundary pair tasks are computed on both owners, one-sided: no cross-rank reduction.

Everything here is host-side indexing (numpy) plus one `torch.distributed.all_gather` per exchange; none of the method's
arithmetic.  The kernels are the library's, unchanged; with the `gloo` backend the same code runs on CPU processes (the
tests drive it with the oracle as the compute engine, and on one GPU by running the ranks' local problems one after the other).
"""
import numpy as np


def partition(cells, world: int) -> np.ndarray:
    """owner[c] in [0, world): contiguous ranges of cells of about equal particle counts (empty ranges are allowed)"""
    first = cells["first"].astype(np.int64)
    end = first + cells["count"].astype(np.int64)
    n = int(end[-1]) if cells.shape[0] else 0
    owner = np.zeros(cells.shape[0], dtype=np.int32)
    lo = 0
    for r in range(1, world):
        hi = max(lo, int(np.searchsorted(end, r * n // world, side="left")))
        owner[hi:] = r
        lo = hi
    return owner


class LocalProblem:
    """What rank `rank` holds of the box: its particles (owned cells first-to-last in global cell order, halo cells among
    them at their place), a cell table and a task list re-indexed to those, and where everything sits in the global arrays."""

    def __init__(self, cells, tasks, owner, rank: int):
        ci = tasks["ci"].astype(np.int64)
        cj = tasks["cj"].astype(np.int64)
        mine = owner[ci] == rank
        mine |= (cj >= 0) & (owner[np.maximum(cj, 0)] == rank)
        self.task_index = np.flatnonzero(mine)                        # global task indices kept, ascending (= task order)
        kept = tasks[self.task_index]
        used = np.unique(np.concatenate([kept["ci"].astype(np.int64), kept["cj"][kept["cj"] >= 0].astype(np.int64)])) if kept.shape[0] else np.zeros(0, np.int64)
        self.cell_index = used                                        # global cell indices held, ascending
        local_of = np.full(cells.shape[0], -1, dtype=np.int64)
        local_of[used] = np.arange(used.shape[0])
        count = cells["count"][used].astype(np.int64)
        first_g = cells["first"][used].astype(np.int64)
        first_l = np.concatenate([[0], np.cumsum(count)[:-1]]) if used.shape[0] else np.zeros(0, np.int64)
        self.n = int(count.sum())
        # local particle k <- global particle particle_index[k]
        self.particle_index = (np.concatenate([np.arange(f, f + c) for f, c in zip(first_g, count)]) if self.n else np.zeros(0, np.int64)).astype(np.int64)
        self.owned = np.repeat(owner[used] == rank, count)            # per local particle
        self.cells = cells[used].copy()
        self.cells["first"] = first_l.astype(self.cells["first"].dtype)
        self.tasks = kept.copy()
        self.tasks["ci"] = local_of[kept["ci"].astype(np.int64)].astype(kept["ci"].dtype)
        has_j = kept["cj"] >= 0
        lj = np.where(has_j, local_of[np.maximum(kept["cj"].astype(np.int64), 0)], -1)
        self.tasks["cj"] = lj.astype(kept["cj"].dtype)
        self.n_self = int((~has_j).sum())

    def take(self, global_parts):
        """the rank's particles out of the global (cell-ordered) array"""
        return np.ascontiguousarray(global_parts[self.particle_index])


def exchange_fields(local_parts, prob: LocalProblem, fields, n_global: int, dist=None, device="cpu"):
    """Halo refresh: every rank contributes the listed fields of its OWNED particles, every rank overwrites those fields of its
    halo particles with their owners' values.  One all-gather (of (global index, values) blocks padded to the largest rank's
    count; tensors live on `device`: "cpu" for gloo, the rank's CUDA device for NCCL over NVLink); with dist = None (a single process standing in for all ranks) `local_parts` / `prob` are lists over the ranks."""
    single = dist is None
    parts_list = local_parts if single else [local_parts]
    probs = prob if single else [prob]
    blocks = []
    for ps, pr in zip(parts_list, probs):
        idx = pr.particle_index[pr.owned]
        blocks.append((idx, {f: np.ascontiguousarray(ps[f][pr.owned]) for f in fields}))
    if not single:
        import torch
        world = dist.get_world_size()
        idx, vals = blocks[0]
        counts = [None] * world
        dist.all_gather_object(counts, int(idx.shape[0]))
        cap = max(counts)
        send_idx = torch.zeros(cap, dtype=torch.int64, device=device)
        send_idx[:idx.shape[0]] = torch.from_numpy(idx).to(device)
        recv_idx = [torch.zeros(cap, dtype=torch.int64, device=device) for _ in range(world)]
        dist.all_gather(recv_idx, send_idx)
        gathered_vals = {}
        for f in fields:
            v = np.ascontiguousarray(vals[f]).reshape(idx.shape[0], -1)
            send = torch.zeros((cap, v.shape[1]), dtype=torch.from_numpy(v).dtype, device=device)
            send[:v.shape[0]] = torch.from_numpy(v).to(device)
            recv = [torch.zeros_like(send) for _ in range(world)]
            dist.all_gather(recv, send)
            gathered_vals[f] = recv
        blocks = [(recv_idx[r][:counts[r]].cpu().numpy(), {f: gathered_vals[f][r][:counts[r]].cpu().numpy() for f in fields}) for r in range(world)]
    # global scratch of the owners' values, then each rank reads its halo out of it
    for f in fields:
        sample = parts_list[0][f]
        glob = np.zeros((n_global,) + sample.shape[1:], dtype=sample.dtype)
        for idx, vals in blocks:
            glob[idx] = vals[f].reshape((idx.shape[0],) + sample.shape[1:])
        for ps, pr in zip(parts_list, probs):
            halo = ~pr.owned
            ps[f][halo] = glob[pr.particle_index[halo]]


def gather_owned(local_parts, prob: LocalProblem, global_out, dist=None):
    """owned particles back into a global array (on every rank with dist; lists over the ranks without)"""
    if dist is None:
        for ps, pr in zip(local_parts, prob):
            global_out[pr.particle_index[pr.owned]] = ps[pr.owned]
        return global_out
    world = dist.get_world_size()
    payload = [None] * world
    dist.all_gather_object(payload, (prob.particle_index[prob.owned], local_parts[prob.owned].tobytes()))
    for idx, raw in payload:
        global_out[idx] = np.frombuffer(raw, dtype=global_out.dtype)
    return global_out
