"""Test-side helpers that drive the oracle (tests only)."""
import numpy as np

import oracle as orc
from sph_inputs.format import PART_DTYPE


def sort_grid(parts, cpd, box=1.0):
    """-> (parts in cell order, cells, tasks, n_self, n_pair) via the oracle's builders."""
    perm, cells = orc.cells_build_grid(parts["x"], cpd, box)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    tasks, ns, npair = orc.tasks_build(cells, orc.cell_hmax(ps, cells), box)
    return ps, cells, tasks, ns, npair


def sort_octree(parts, max_per_leaf, box=1.0):
    perm, cells = orc.cells_build_octree(parts["x"], parts["h"], max_per_leaf, box)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    tasks, ns, npair = orc.tasks_build(cells, orc.cell_hmax(ps, cells), box)
    return ps, cells, tasks, ns, npair


def lattice(n_side, h_over_dx, u=1.0):
    """Unperturbed simple-cubic lattice, equal masses 1/N, v = 0."""
    n = n_side ** 3
    parts = np.zeros(n, dtype=PART_DTYPE)
    p = np.arange(n)
    ijk = np.stack([p // (n_side * n_side), (p // n_side) % n_side, p % n_side], axis=1)
    parts["x"] = (ijk + 0.5) / n_side
    parts["mass"] = 1.0 / n
    parts["h"] = h_over_dx / n_side
    parts["u"] = u
    parts["id"] = p
    parts["time_bin"] = 1
    return parts


def scaled_err(val, ref, scale):
    """|val - ref| / max(|ref|, scale)  (reading C32: sign-changing outputs need a natural scale)."""
    return np.abs(val - ref) / np.maximum(np.abs(ref), scale)


def raw_copy(parts):
    """Byte-exact copy of a record array (numpy's .copy() does not promise to keep pad bytes)."""
    out = np.zeros(parts.shape[0], dtype=parts.dtype)
    out.view(np.uint8)[:] = parts.view(np.uint8)
    return out
