"""Workload builders shared by bench.py and the full-size tests: seeded synthetic particles (sph_inputs/) put into cell order with
the library's own builders, with cells and tasks.  Setup only (untimed); `sph` is the binding module."""
import time

import numpy as np

from .pipeline import GAMMA, iterate_h_on_gpu


def build_config2(sph, torch, seed, n):
    """-> particles in cell order with h (48 neighbours), rho, rho_dh, u (P = 1 | 0.1), P, c_s set; cells; tasks"""
    import sph_inputs as si
    scale = max(1, int(round((2 ** 21 / n) ** (1.0 / 3.0))))
    n_yz, n_left, n_right, cpd = 128 // scale, 102 // scale, 26 // scale, 32 // scale
    parts = si.config2_positions(seed, n_yz=n_yz, n_left=n_left, n_right=n_right)
    perm, cells = sph.sph_cells_build_grid(parts["x"], cpd)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    width = float(cells["width"][0])
    ps["h"] = np.minimum(ps["h"], np.float32(0.4999 * width))
    hmax = np.full(cells.shape[0], np.float32(0.4999 * width), dtype=np.float32)
    tasks, n_self, n_pair = sph.sph_tasks_build(cells, hmax)
    h, worst, iters = iterate_h_on_gpu(sph, torch, ps, cells, tasks)
    ps["h"] = h
    # density pass -> rho, rho_dh; u from the target pressure; ghost -> P, c_s
    layout = sph.sph_layout_aos()
    store = sph.sph_store_create(layout, ps.shape[0])
    sph.sph_store_set_cells(store, cells)
    sph.sph_store_import_aos(store, ps)
    batch = sph.sph_batch_create(store, tasks)
    s_in, s_out = sph.sph_attrset_canonical(0), sph.sph_attrset_canonical(1)
    b_in = torch.empty(sph.sph_batch_buffer_bytes(batch, s_in), dtype=torch.uint8, device="cuda")
    b_out = torch.empty(sph.sph_batch_buffer_bytes(batch, s_out), dtype=torch.uint8, device="cuda")
    sph.sph_store_zero(store, s_out)
    sph.sph_pack(store, batch, s_in, b_in)
    sph.sph_density(batch, b_in, b_out)
    sph.sph_unpack(store, batch, s_out, b_out, sph.SPH_UNPACK_REDUCE)
    torch.cuda.synchronize()
    sph.sph_store_export_aos(store, ps)
    p_target = np.where(ps["x"][:, 0] < 0.5, 1.0, 0.1)
    ps["u"] = (p_target / ((GAMMA - 1.0) * ps["rho"].astype(np.float64))).astype(np.float32)
    sph.sph_store_import_aos(store, ps)
    sph.sph_ghost(store, sph.sph_params(np.float32(GAMMA), 0.8, 3.0))
    torch.cuda.synchronize()
    sph.sph_store_export_aos(store, ps)
    sph.sph_batch_destroy(batch)
    sph.sph_store_destroy(store)
    del b_in, b_out
    # ordered pairs inside the cut-off of the force loop, r < max(2h_i, 2h_j): with the 48-neighbour h every particle has
    # (4/3) pi (2h)^3 n = 48 / (mean kernel weight) others inside its own 2h; counted from wcount's definition instead:
    # N_i = (4/3) pi (2 h_i)^3 n_i where n_i = rho_i / m is the number density the particle sees
    ngb = (32.0 / 3.0) * np.pi * ps["h"].astype(np.float64) ** 3 * (ps["rho"].astype(np.float64) / ps["mass"])
    info = {"cells_per_dim": cpd, "h_iterations": iters, "worst_neighbour_error": worst, "h_min": float(h.min()), "h_max": float(h.max()),
            "per_cell_min": int(cells["count"].min()), "per_cell_max": int(cells["count"].max()),
            "neighbour_pairs": float(ngb.sum()), "neighbours_per_particle": float(ngb.mean())}
    return ps, cells, tasks, info


def build_clumpy(sph, which, seed, n):
    """clustered particles -> octree (<= 400 per leaf) -> cell order, cells, tasks"""
    import sph_inputs as si
    t0 = time.perf_counter()
    parts = si.config3(seed, n) if which == 3 else si.config4(seed, n)
    t1 = time.perf_counter()
    perm, cells = sph.sph_cells_build_octree(parts["x"], parts["h"], 400)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    del parts
    hmax = np.maximum.reduceat(ps["h"], cells["first"].astype(np.int64)).astype(np.float32)
    tasks, n_self, n_pair = sph.sph_tasks_build(cells, hmax)
    cnt = cells["count"]
    info = {"cells": int(cells.shape[0]), "per_cell_min": int(cnt.min()), "per_cell_max": int(cnt.max()), "per_cell_mean": round(float(cnt.mean()), 1),
            "per_cell_median": float(np.median(cnt)), "self_tasks": int(n_self), "pair_tasks": int(n_pair),
            "generate_s": round(t1 - t0, 1), "cells_and_tasks_s": round(time.perf_counter() - t1, 1)}
    return ps, cells, tasks, info
