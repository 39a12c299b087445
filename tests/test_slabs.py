"""One box over several ranks: slabs of cells + one layer of halo cells (paper_2606_23891_b200/slabs.py).

The decomposition is host-side indexing; what must hold is that the owned particles of every rank end up, BIT FOR BIT, with the
results of the undivided box (every task that touches an owned cell is kept, in the same order, so the ordered reduction of the
unpack sees the same records in the same order), for any number of ranks.  Here the compute engine is the oracle (CPU); the same
check runs through the CUDA path in tests/test_gpu_parity.py::test_slab_split_equals_single_box, and through two gloo
processes below."""
import json
import os
import sys

import numpy as np
import pytest

import oracle as orc
import sph_inputs as si
from orc_setup import raw_copy, sort_grid
from paper_2606_23891_b200 import slabs
from test_multirank_gloo import ROOT, _json_lines, _torchrun

GAMMA = float(np.float32(5.0 / 3.0))
HALO_FIELDS = ("rho", "rho_dh", "wcount", "wcount_dh")


def test_partition_is_contiguous_and_balanced():
    ps, cells, tasks, _, _ = sort_grid(si.jittered_lattice(12, 5, jitter=0.6, h_spread=0.2), 4)
    for world in (1, 2, 3, 5):
        owner = slabs.partition(cells, world)
        assert owner.min() == 0 and owner.max() == world - 1 and np.all(np.diff(owner) >= 0)
        per = np.bincount(owner, weights=cells["count"], minlength=world)
        assert per.sum() == ps.shape[0] and per.max() - per.min() <= 2 * cells["count"].max()


def whole_box(ps, cells, tasks):
    ref = raw_copy(ps)
    orc.density_cycle(ref, cells, tasks)
    orc.ghost(ref, GAMMA)
    orc.force_cycle(ref, cells, tasks)
    return ref


@pytest.mark.parametrize("world", [2, 3])
def test_slab_split_equals_single_box_oracle(world):
    orc.set_threads(8)
    ps, cells, tasks, _, _ = sort_grid(si.jittered_lattice(12, 5, jitter=0.6, sigma_v=0.3, h_spread=0.2, mass_spread=0.4, u_spread=0.3), 4)
    ref = whole_box(ps, cells, tasks)
    owner = slabs.partition(cells, world)
    probs = [slabs.LocalProblem(cells, tasks, owner, r) for r in range(world)]
    # every task is kept by at least one rank, boundary tasks by two; every particle is owned exactly once
    kept = np.zeros(tasks.shape[0], dtype=int)
    owned = np.zeros(ps.shape[0], dtype=int)
    for p in probs:
        kept[p.task_index] += 1
        owned[p.particle_index[p.owned]] += 1
        assert np.all(p.tasks["cj"][:p.n_self] < 0) and np.all(p.tasks["cj"][p.n_self:] >= 0)      # self tasks first (C22)
    assert kept.min() == 1 and kept.max() == 2 and np.all(owned == 1)
    assert sum(p.n for p in probs) > ps.shape[0]                         # halo particles are replicated
    local = [p.take(ps) for p in probs]
    for lp, p in zip(local, probs):
        orc.density_cycle(lp, p.cells, p.tasks)
    plans = [slabs.HaloPlan(cells, tasks, owner, p, r) for r, p in enumerate(probs)]
    for r, (p, pl) in enumerate(zip(probs, plans)):
        # the plan covers exactly the rank's halo particles, each once, and what r receives from q is what q sends to r
        got_idx = np.sort(np.concatenate(list(pl.recv.values()))) if pl.recv else np.zeros(0, np.int64)
        assert np.array_equal(got_idx, np.flatnonzero(~p.owned))
        for q, idx in pl.recv.items():
            assert np.array_equal(p.particle_index[idx], probs[q].particle_index[plans[q].send[r]])
        assert all(np.all(p.owned[idx]) for idx in pl.send.values())
    moved = slabs.exchange_fields(local, probs, HALO_FIELDS, plans)
    halo = sum(int((~p.owned).sum()) for p in probs)
    # O(halo) bytes: nothing but the halo particles' fields moves (in this small periodic box -- two or three slabs of a 4^3 grid --
    # nearly every cell is somebody's halo; on a large box the halo is one layer of cells per slab face)
    assert moved == halo * 4 * len(HALO_FIELDS)
    for lp, p in zip(local, probs):
        orc.ghost(lp, GAMMA)
        orc.force_cycle(lp, p.cells, p.tasks)
    got = slabs.gather_owned(local, probs, np.zeros_like(ps))
    assert np.array_equal(got.view(np.uint8).reshape(-1, 128)[:, :108], ref.view(np.uint8).reshape(-1, 128)[:, :108])
    assert np.array_equal(got["id"], ref["id"])


def test_slab_split_over_two_gloo_ranks():
    r = _torchrun([os.path.join(ROOT, "tests", "_gloo_slab_worker.py")])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1, r.stdout
    d = lines[0]
    assert d["world"] == 2 and d["identical"] is True and d["halo_particles"] > 0 and d["owned"] == [d["n"] - d["owned"][1], d["owned"][1]]
    # O(halo): rank 0 received its halo particles and sent 16 bytes (4 f32 fields) for each particle rank 1 holds as halo
    assert d["n_recv"] == d["halo_particles"] and d["sent_bytes"] == 16 * d["n_send"] and 0 < d["n_send"] <= d["owned"][0]


def test_halo_plan_moves_one_layer_of_cells_per_slab_face():
    """on a 16^3 periodic grid cut into 4 slabs every rank's halo is one layer of 16^2 cells on each of its two faces, so a refresh
    sends the fields of 2 x 256 cells' particles per rank -- an eighth of the box in total per rank pair, not the whole box"""
    import paper_2606_23891_b200 as sph
    x = np.random.default_rng(11).random((40000, 3))
    perm, cells = sph.sph_cells_build_grid(x, 16)
    tasks, _, _ = sph.sph_tasks_build(cells, np.full(cells.shape[0], 0.02, dtype=np.float32))
    cells, tasks = cells.view(orc.CELL_DTYPE), tasks.view(orc.TASK_DTYPE)
    world = 4
    owner = slabs.partition(cells, world)
    for r in range(world):
        prob = slabs.LocalProblem(cells, tasks, owner, r)
        plan = slabs.HaloPlan(cells, tasks, owner, prob, r)
        assert sorted(plan.recv) == sorted({(r - 1) % world, (r + 1) % world}) == sorted(plan.send)
        halo_cells = int((owner[prob.cell_index] != r).sum())
        assert 2 * 256 <= halo_cells <= 2 * 256 + 2 * 16 * 16            # slab cuts follow particle counts, not cell layers: at most one ragged layer more
        assert plan.n_recv == int((~prob.owned).sum()) and plan.n_recv < 0.2 * x.shape[0] and plan.n_send < 0.2 * x.shape[0]
