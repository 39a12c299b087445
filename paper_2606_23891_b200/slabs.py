"""One box spread over several GPUs: slabs of cells with one layer of halo cells.

The path shards naturally: tasks only read inputs and reduce into per-particle outputs.  The cell table is cut into
`world` contiguous ranges of about equal particle counts ("slabs"); rank r OWNS the particles of its cells, keeps every
task that has at least one owned side, and so also holds the cells on the other side of those tasks ("halo").  It runs
the ordinary pack -> loop -> unpack cycle over its local tasks; the results of owned particles are complete and are, bit
for bit, those of the undivided box (every task that touches an owned cell is kept, in the same order, so the ordered
reduction of the unpack sees the same records in the same order); the results of halo particles are partial and are
never read.  Between the loops one exchange step refreshes the halo particles' fields from their owners (rho, rho_dh
before the ghost and the force loop).  Boundary pair tasks are computed on both owners, one-sided: no cross-rank reduction.

Everything here is host-side indexing (numpy) plus one batched isend / irecv per neighbour pair and exchange (`HaloPlan`,
`exchange_fields`: O(halo) bytes, no all-gather, no array of global size); none of the method's arithmetic.  The kernels are the library's, unchanged; with the `gloo` backend the same code runs on CPU processes (the
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


class HaloPlan:
    """Who sends what to whom in a halo refresh, worked out once per decomposition and without communication (every rank holds the
    global cell table, task list and owner map -- host metadata, as in the paper where the task graph is global):
    send[p] = local indices of MY OWNED particles that rank p holds as halo, recv[p] = local indices of my HALO particles that
    rank p owns; both in ascending global particle order, so the two sides of a transfer agree element by element.
    A cell is halo on rank a exactly when a pair task joins it to a cell that a owns while another rank owns it."""

    def __init__(self, cells, tasks, owner, prob: LocalProblem, rank: int):
        ci, cj = tasks["ci"].astype(np.int64), tasks["cj"].astype(np.int64)
        has_j = cj >= 0
        oi, oj = owner[ci], owner[np.maximum(cj, 0)]
        cross = has_j & (oi != oj)
        holder = np.concatenate([oi[cross], oj[cross]]).astype(np.int64)       # the rank that holds ...
        cell = np.concatenate([cj[cross], ci[cross]])                          # ... this cell as halo
        pairs = np.unique(np.stack([holder, cell], axis=1), axis=0) if holder.shape[0] else np.zeros((0, 2), np.int64)
        local_first = np.full(cells.shape[0], -1, dtype=np.int64)
        local_first[prob.cell_index] = prob.cells["first"].astype(np.int64)
        count = cells["count"].astype(np.int64)

        def particles(cs):
            return (np.concatenate([np.arange(local_first[c], local_first[c] + count[c]) for c in cs]) if len(cs) else np.zeros(0, np.int64)).astype(np.int64)
        self.send, self.recv = {}, {}
        for p in range(int(owner.max()) + 1 if owner.shape[0] else 0):
            if p == rank:
                continue
            out_cells = pairs[(pairs[:, 0] == p) & (owner[pairs[:, 1]] == rank), 1]       # mine, halo on p (np.unique left them ascending)
            in_cells = pairs[(pairs[:, 0] == rank) & (owner[pairs[:, 1]] == p), 1]        # p's, halo on me
            if out_cells.shape[0]:
                self.send[p] = particles(out_cells)
            if in_cells.shape[0]:
                self.recv[p] = particles(in_cells)
        self.n_send = int(sum(v.shape[0] for v in self.send.values()))
        self.n_recv = int(sum(v.shape[0] for v in self.recv.values()))


def exchange_fields(local_parts, prob, fields, plan, dist=None):
    """Halo refresh, O(halo): every rank sends the listed fields of exactly those owned particles a peer holds as halo, and
    overwrites those fields of its own halo particles with what their owners send -- one batched isend / irecv per neighbour pair
    (`dist.batch_isend_irecv`: NCCL over NVLink on GPUs, gloo on CPU processes), no all-gather, no array of global size.
    `local_parts`: the rank's particles, either a numpy record array on the host (gloo) or a dict {field: torch tensor [n_local(, k)]}
    on the rank's device (NCCL: gather, transfer and scatter all stay on the device); fields must share one dtype.
    With dist = None (one process standing in for all ranks) local_parts / prob / plan are lists over the ranks.
    Returns the payload bytes this rank (or, without dist, all ranks together) sent."""
    if dist is None:
        moved = 0
        for r, (ps, pl) in enumerate(zip(local_parts, plan)):
            for p, r_idx in pl.recv.items():
                s_idx = plan[p].send[r]
                for f in fields:
                    ps[f][r_idx] = local_parts[p][f][s_idx]
                    moved += int(ps[f][r_idx].nbytes)
        return moved
    import torch
    is_np = isinstance(local_parts, np.ndarray)
    cols = {f: (torch.from_numpy(np.ascontiguousarray(local_parts[f])) if is_np else local_parts[f]).reshape(prob.n, -1) for f in fields}
    first = cols[fields[0]]
    assert all(c.dtype == first.dtype and c.device == first.device for c in cols.values()), "exchanged fields must share dtype and device"
    widths = [cols[f].shape[1] for f in fields]
    ops, keep, landed = [], [], []
    for p in sorted(set(plan.send) | set(plan.recv)):
        if p in plan.send:
            s_idx = torch.from_numpy(plan.send[p]).to(first.device)
            keep.append(torch.cat([cols[f].index_select(0, s_idx) for f in fields], dim=1).contiguous())
            ops.append(dist.P2POp(dist.isend, keep[-1], p))
        if p in plan.recv:
            buf = torch.empty((plan.recv[p].shape[0], sum(widths)), dtype=first.dtype, device=first.device)
            ops.append(dist.P2POp(dist.irecv, buf, p))
            landed.append((torch.from_numpy(plan.recv[p]).to(first.device), buf))
    if ops:
        for work in dist.batch_isend_irecv(ops):
            work.wait()
    for r_idx, buf in landed:
        c0 = 0
        for f, w in zip(fields, widths):
            cols[f].index_copy_(0, r_idx, buf[:, c0:c0 + w])
            c0 += w
    if is_np:
        for f in fields:
            local_parts[f] = cols[f].numpy().reshape(local_parts[f].shape)
    return int(sum(t.numel() * t.element_size() for t in keep))


def gather_owned(local_parts, prob: LocalProblem, global_out, dist=None):
    """owned particles back into a global array (on every rank with dist; lists over the ranks without).  A verification helper
    for the tests -- O(N) by its purpose -- not a step of the path."""
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
