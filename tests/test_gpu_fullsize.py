"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (needs a B200).

configs[1] (262,144 particles, 57,344 tasks in ONE batch, exactly what `bench.py` runs): the oracle finishes a whole
step of it in about a second on the box's cores, so everything is compared in full -- pack buffers and unpack results
byte for byte, the physics of every particle within the north_star tolerances, for both store layouts.
configs[2] (2^21 particles, bundles of 512 tasks, h from the oracle's 48-neighbour iteration, rho / P / c_s from its density
cycle and ghost): pack FORCE_IN and unpack FORCE_OUT compared in full, byte for byte, in the segmented launch configuration;
the force loop on bundles sampled across the box (left, interface, right), each recomputed by the oracle from the same
packed records; the library's own h iteration (bench setup) against the oracle's.
configs[3] (2^24 clustered particles, octree <= 400 per leaf): pack and unpack compared in full, byte for byte.
configs[4] (2^26 particles): the two-stream bundle pipeline of bench.py on the full set, 1,024 sampled cells recomputed by the
oracle from all their tasks, momentum and energy invariants on the full output.  (The same pipeline is compared in full,
bit for bit and against the oracle, on a 2^19 instance in test_gpu_pipeline.py.)
"""
import numpy as np
import pytest
import torch

import oracle as orc
import paper_2606_23891_b200 as sph
import sph_inputs as si
from gpu_setup import GAMMA, PARAMS, GpuCase, canon, per_component_ok, to_attrset, valid_mask, vec_scale, within_1e4_or_1e6
from orc_setup import raw_copy, sort_grid
from test_gpu_parity import _random_result_buffer, _records, check_store_physics, gpu_step

pytestmark = pytest.mark.gpu

_C1 = {}


def config1():
    if not _C1:
        orc.set_threads(64)
        ps, cells, tasks, n_self, n_pair = sort_grid(si.config1(seed=1), 16)
        assert (n_self, n_pair) == (4096, 53248) and np.all(cells["count"] == 64)
        ref = raw_copy(ps)
        orc.density_cycle(ref, cells, tasks)
        orc.ghost(ref, GAMMA)
        f_in = orc.pack(ref, cells, tasks, orc.FORCE_IN)
        exempt = orc.flag_cutoff_pairs(cells, tasks, f_in)              # C31: particles with a partner on the cut-off
        orc.force_cycle(ref, cells, tasks)
        _C1.update(ps=ps, cells=cells, tasks=tasks, ref=ref, exempt=exempt)
    return _C1["ps"], _C1["cells"], _C1["tasks"], _C1["ref"]


def _block_mask(cells, tasks, rec, total):
    """bytes of a buffer that blocks occupy, vectorised (pad bytes are unspecified)"""
    off, tot = orc.block_offsets(cells, tasks, rec)
    assert tot == total
    m = np.zeros(total + 1, dtype=np.int32)
    for side, key in ((0, "ci"), (1, "cj")):
        c = tasks[key].astype(np.int64)
        sel = c >= 0
        o = off[side::2][sel].astype(np.int64)
        n = cells["count"][c[sel]].astype(np.int64) * rec
        np.add.at(m, o, 1)
        np.add.at(m, o + n, -1)
    return np.cumsum(m[:-1]) > 0


def _record_particles(cells, tasks):
    """particle index of every record of a buffer, in buffer order (task ascending, side i then side j)"""
    c = np.stack([tasks["ci"], tasks["cj"]], axis=1).ravel().astype(np.int64)
    c = c[c >= 0]
    cnt = cells["count"][c].astype(np.int64)
    start = np.repeat(cells["first"][c].astype(np.int64), cnt)
    within = np.arange(cnt.sum()) - np.repeat(np.cumsum(cnt) - cnt, cnt)
    return start + within


@pytest.mark.parametrize("layout", ["split", "aos"])
def test_config1_whole_step_every_particle(layout):
    ps, cells, tasks, ref = config1()
    g = GpuCase(ps, cells, tasks, layout)                # one batch holding every task, zeroing fused into the unpacks: bench.py's configuration
    got = gpu_step(g, fused_zero=True)
    sph.sph_store_import_aos(g.store, ps)
    assert np.array_equal(canon(gpu_step(g)), canon(got))      # the seven-launch step equals the nine-launch one bit for bit
    check_store_physics(got, ref)
    vs_ok = np.abs(got["v_sig"] - ref["v_sig"]) <= 1e-4 * ref["v_sig"]
    assert np.all(vs_ok | _C1["exempt"]) and _C1["exempt"].mean() < 0.01      # C31: only particles with a partner on the cut-off may differ
    for fld in ("x", "v", "mass", "h", "u", "div_v", "rot_v", "id", "time_bin"):
        assert np.array_equal(got[fld], ps[fld]), fld
    m = got["mass"].astype(np.float64)
    a = got["a"].astype(np.float64)
    assert np.abs((m[:, None] * a).sum(0)).max() <= 1e-6 * np.abs(m[:, None] * a).sum()
    g.close()


@pytest.mark.parametrize("layout", ["split", "aos"])
def test_config1_pack_and_unpack_bytes_in_full(layout):
    ps, cells, tasks, ref = config1()
    filled = raw_copy(ref)                               # physically consistent values in every field the sets touch
    g = GpuCase(filled, cells, tasks, layout)
    for oset in (orc.DENSITY_IN, orc.FORCE_IN):
        want = orc.pack(filled, cells, tasks, oset)
        buf = g.pack(to_attrset(oset)).cpu().numpy()
        mask = _block_mask(cells, tasks, orc.record_bytes(oset), want.shape[0])
        assert buf.shape == want.shape and np.array_equal(buf[mask], want[mask])
    for n_set, oset in enumerate((orc.DENSITY_OUT, orc.FORCE_OUT)):
        rec = orc.record_bytes(oset)
        _, total = orc.block_offsets(cells, tasks, rec)
        res = _random_result_buffer(total, 300 + n_set)
        want = raw_copy(filled)
        orc.unpack(want, cells, tasks, oset, res, orc.MODE_REDUCE)
        sph.sph_store_import_aos(g.store, filled)
        sph.sph_unpack(g.store, g.batch, to_attrset(oset), torch.from_numpy(res).cuda(), sph.SPH_UNPACK_REDUCE)
        assert np.array_equal(canon(g.export()), canon(want)), rec
    g.close()


def test_config1_loops_every_record():
    """density and force result buffers of the one-batch launch, every record of every task side"""
    ps, cells, tasks, ref = config1()
    g = GpuCase(ref, cells, tasks, "split")
    b_in = orc.pack(ref, cells, tasks, orc.DENSITY_IN)
    want = orc.density(cells, tasks, b_in)
    d_out = g.buffer(to_attrset(orc.DENSITY_OUT))
    sph.sph_density(g.batch, torch.from_numpy(b_in).cuda(), d_out)
    torch.cuda.synchronize()
    got = d_out.cpu().numpy()
    mask = _block_mask(cells, tasks, 16, want.shape[0])
    w4, g4 = want[mask].view(np.float32).reshape(-1, 4).astype(np.float64), got[mask].view(np.float32).reshape(-1, 4).astype(np.float64)
    h = float(ref["h"][0])
    mass = float(ref["mass"][0])
    # partial sums of one task side: tolerances relative to the scale of a full sum (C32), as in test_gpu_parity
    scale = np.array([mass, mass / h, 1.0, 1.0 / h]) / (np.pi * h ** 3)
    assert np.all(np.abs(g4 - w4) <= 2e-5 * np.maximum(np.abs(w4), scale))
    f_in = orc.pack(ref, cells, tasks, orc.FORCE_IN)
    want = orc.force(cells, tasks, f_in, 0.8, 3.0)
    f_out = g.buffer(to_attrset(orc.FORCE_OUT))
    sph.sph_force(g.batch, torch.from_numpy(f_in).cuda(), f_out, PARAMS)
    torch.cuda.synchronize()
    got = f_out.cpu().numpy()
    mask = _block_mask(cells, tasks, 20, want.shape[0])
    w5, g5 = want[mask].view(np.float32).reshape(-1, 5).astype(np.float64), got[mask].view(np.float32).reshape(-1, 5).astype(np.float64)
    assert within_1e4_or_1e6(g5[:, :3], w5[:, :3], vec_scale(ref["a"])) and within_1e4_or_1e6(g5[:, 3], w5[:, 3], vec_scale(ref["du_dt"]))
    assert per_component_ok(g5[:, :3], w5[:, :3], vec_scale(ref["a"]), "a (sampled records)")
    exempt = _C1["exempt"][_record_particles(cells, tasks)]              # C31
    assert np.all((np.abs(g5[:, 4] - w5[:, 4]) <= 1e-4 * np.abs(w5[:, 4])) | exempt)
    g.close()


# ------------------------------------------------------------------ configs[2]

_C2 = {}


def config2():
    """2^21 particles of the Sod-like setup in cell order, in the state the force loop of configs[2] starts from, every
    value produced by the oracle: h from the 48-neighbour iteration (reading C20), rho and rho_dh from the density cycle,
    u such that P = 1 | 0.1 (reading C18), P and c_s from the ghost."""
    if not _C2:
        orc.set_threads(64)
        parts = si.config2_positions(seed=1)
        h, bad = orc.iterate_h(parts["x"], parts["h"], h_cap=0.4999 / 32)
        assert bad == 0
        parts["h"] = h
        ps, cells, tasks, n_self, n_pair = sort_grid(parts, 32)
        assert ps.shape[0] == 1 << 21 and n_self == 32768
        orc.density_cycle(ps, cells, tasks)
        p_target = np.where(ps["x"][:, 0] < 0.5, 1.0, 0.1)
        ps["u"] = (p_target / ((GAMMA - 1.0) * ps["rho"].astype(np.float64))).astype(np.float32)
        orc.ghost(ps, GAMMA)
        nn = 32.0 / 3.0 * np.pi * ps["h"].astype(np.float64) ** 3 * ps["wcount"]
        assert np.abs(nn - 48.0).max() < 0.02                                # the condition holds through the independent pipeline
        assert ps["rho"][ps["x"][:, 0] < 0.5].mean() > 2.5 * ps["rho"][ps["x"][:, 0] >= 0.5].mean()      # two densities
        _C2.update(ps=ps, cells=cells, tasks=tasks)
    return _C2["ps"], _C2["cells"], _C2["tasks"]


def test_config2_pack_unpack_bundles_of_512_bytes_in_full():
    ps, cells, tasks = config2()
    g = GpuCase(ps, cells, tasks, "split", tasks_per_segment=512)      # 64 + 832 bundles under one launch: bench.py --workload config2
    info = sph.sph_batch_get_info(g.batch)
    assert info.n_segments == 896
    aset = to_attrset(orc.FORCE_IN)
    got = g.pack(aset).cpu().numpy()
    off, seg_off = sph.sph_batch_block_offsets(g.batch, aset)
    # bundle by bundle the oracle packs the bundle's tasks as a stand-alone batch; compare a spread of bundles in full
    for b in list(range(0, 896, 37)) + [63, 64, 895]:
        sel = tasks[512 * b:512 * (b + 1)]
        want = orc.pack(ps, cells, sel, orc.FORCE_IN)
        mask = _block_mask(cells, sel, 52, want.shape[0])
        lo = int(seg_off[b])
        assert np.array_equal(got[lo:lo + want.shape[0]][mask], want[mask]), b
    # unpack of the whole segmented buffer against the oracle run bundle after bundle (ascending task order)
    rec = 20
    oset = orc.FORCE_OUT
    aset = to_attrset(oset)
    total = sph.sph_batch_buffer_bytes(g.batch, aset)
    res = _random_result_buffer(total, 77)
    _, seg_off = sph.sph_batch_block_offsets(g.batch, aset)
    want = raw_copy(ps)
    for b in range(896):
        sel = tasks[512 * b:512 * (b + 1)]
        _, tot_b = orc.block_offsets(cells, sel, rec)
        lo = int(seg_off[b])
        orc.unpack(want, cells, sel, oset, res[lo:lo + tot_b], orc.MODE_REDUCE)
    sph.sph_unpack(g.store, g.batch, aset, torch.from_numpy(res).cuda(), sph.SPH_UNPACK_REDUCE)
    assert np.array_equal(canon(g.export()), canon(want))
    g.close()


def test_config2_force_on_sampled_bundles():
    ps, cells, tasks = config2()
    g = GpuCase(ps, cells, tasks, "split", tasks_per_segment=512)
    s_in, s_out = to_attrset(orc.FORCE_IN), to_attrset(orc.FORCE_OUT)
    b_in = g.pack(s_in)
    b_out = g.buffer(s_out)
    sph.sph_force(g.batch, b_in, b_out, PARAMS)
    torch.cuda.synchronize()
    got_in, got_out = b_in.cpu().numpy(), b_out.cpu().numpy()
    _, seg_in = sph.sph_batch_block_offsets(g.batch, s_in)
    _, seg_out = sph.sph_batch_block_offsets(g.batch, s_out)
    for b in (0, 40, 64, 100, 470, 480, 800, 895):       # self bundles, pair bundles left / at the interface / right
        sel = tasks[512 * b:512 * (b + 1)]
        want_in = orc.pack(ps, cells, sel, orc.FORCE_IN)
        want = orc.force(cells, sel, want_in, 0.8, 3.0)
        mask = _block_mask(cells, sel, 20, want.shape[0])
        lo = int(seg_out[b])
        w5 = want[mask].view(np.float32).reshape(-1, 5).astype(np.float64)
        g5 = got_out[lo:lo + want.shape[0]][mask].view(np.float32).reshape(-1, 5).astype(np.float64)
        assert within_1e4_or_1e6(g5[:, :3], w5[:, :3]) and within_1e4_or_1e6(g5[:, 3], w5[:, 3]), b
        assert per_component_ok(g5[:, :3], w5[:, :3], what=f"a (bundle {b})"), b
        exempt = orc.flag_cutoff_pairs(cells, sel, want_in)[_record_particles(cells, sel)]      # C31, this bundle's own pairs
        assert np.all((np.abs(g5[:, 4] - w5[:, 4]) <= 1e-4 * np.abs(w5[:, 4])) | exempt) and exempt.mean() < 0.01, b
    g.close()


def test_library_h_iteration_matches_the_oracles():
    """pipeline.iterate_h_on_gpu (the library's density loop driving Newton steps; setup of the configs[2] bench)
    against orc.iterate_h (reading C20) on a 2^15 Sod-like box: both solve (4/3) pi (2h)^3 wcount = 48, to 1e-3 here."""
    from paper_2606_23891_b200 import pipeline as bw, workloads
    parts = si.config2_positions(seed=3, n_yz=32, n_left=25, n_right=6)
    perm, cells = sph.sph_cells_build_grid(parts["x"], 8)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    cap = np.float32(0.4999 * float(cells["width"][0]))
    ps["h"] = np.minimum(ps["h"], cap)
    tasks, _, _ = sph.sph_tasks_build(cells, np.full(cells.shape[0], cap, dtype=np.float32))
    h_gpu, worst, iters = bw.iterate_h_on_gpu(sph, torch, ps, cells, tasks, tol=1e-3, max_iter=30)
    h_orc, bad = orc.iterate_h(ps["x"], ps["h"], h_cap=float(cap), tol=1e-3, max_iter=60)
    assert bad == 0 and worst <= 1e-3 and iters < 30
    assert np.max(np.abs(h_gpu.astype(np.float64) - h_orc) / h_orc) <= 1e-5
    assert h_orc.max() / h_orc.min() > 1.4                                   # really two densities


# ------------------------------------------------------------------ configs[3]

def test_config3_pack_and_unpack_bytes_in_full():
    """2^24 clustered particles, octree <= 400 per leaf, ~2.0e6 tasks / 5.2e8 instances: the 5- and 13-field packs (C21) of
    every task and the 13-field REDUCE unpack, byte for byte, AoS and split-AoS.  The buffers are tens of GB, so tasks go
    through in slices of 2^17, each slice its own batch (what a slice packs is exactly what a stand-alone batch packs)."""
    from paper_2606_23891_b200 import pipeline as bw, workloads
    from test_gpu_parity import PACK_SWEEP, UNPACK_SWEEP, fill_all_fields, sweep_set
    orc.set_threads(64)
    ps, cells, tasks, info = workloads.build_clumpy(sph, 3, 1, 1 << 24)
    oc, ot = cells.view(orc.CELL_DTYPE), tasks.view(orc.TASK_DTYPE)
    assert info["per_cell_max"] <= 448 and ps.shape[0] == 1 << 24
    ps = fill_all_fields(ps, 11)
    step = 1 << 17
    u_set = sweep_set(UNPACK_SWEEP, 13, 0)
    for layout in ("split", "aos"):
        lay = sph.sph_layout_split() if layout == "split" else sph.sph_layout_aos()
        store = sph.sph_store_create(lay, ps.shape[0])
        sph.sph_store_import_aos(store, ps)
        sph.sph_store_set_cells(store, cells)
        want_store = raw_copy(ps)
        batches = []
        for t0 in range(0, tasks.shape[0], step):                                # every pack first: the store is still pristine
            sel, osel = tasks[t0:t0 + step], ot[t0:t0 + step]
            batch = sph.sph_batch_create(store, np.ascontiguousarray(sel))
            batches.append(batch)
            for k in (5, 13):
                if layout == "aos" and k == 13 and (t0 // step) % 4:
                    continue                                                     # AoS, 13 fields: every fourth slice
                oset = sweep_set(PACK_SWEEP, k, orc.FLAG_X_REL_F32)
                aset = to_attrset(oset)
                buf = torch.empty(sph.sph_batch_buffer_bytes(batch, aset), dtype=torch.uint8, device="cuda")
                sph.sph_pack(store, batch, aset, buf)
                got = buf.cpu().numpy()
                want = orc.pack(ps, oc, osel, oset)
                assert got.shape == want.shape and orc.compare_blocks(oc, osel, 4 * k, got, want) == -1, (layout, k, t0)
                del buf
        # then the unpack of seeded result records, slice after slice (ascending task order = the order of the definition)
        aset = to_attrset(u_set)
        for n_slice, batch in enumerate(batches):
            osel = ot[n_slice * step:(n_slice + 1) * step]
            res = _random_result_buffer(sph.sph_batch_buffer_bytes(batch, aset), 900 + n_slice)
            sph.sph_unpack(store, batch, aset, torch.from_numpy(res).cuda(), sph.SPH_UNPACK_REDUCE)
            if layout == "split":
                orc.unpack(want_store, oc, osel, u_set, res, orc.MODE_REDUCE)
            sph.sph_batch_destroy(batch)
        torch.cuda.synchronize()
        got_store = np.zeros_like(ps)
        sph.sph_store_export_aos(store, got_store)
        if layout == "split":
            _C3_WANT["store"] = want_store
        assert np.array_equal(canon(got_store), canon(_C3_WANT["store"])), layout
        sph.sph_store_destroy(store)


_C3_WANT = {}


# ------------------------------------------------------------------ configs[4]

def test_config4_pipeline_sampled_cells_and_invariants():
    """2^26 particles through bench.py's configs[4] pipeline (bundles of 4,096 tasks, eight under one launch per stage, two streams,
    host-resident split-AoS store, streamed staging, one graph replay).  1,024 seeded cells are recomputed by the oracle from ALL their tasks: the density
    cycle over every task that touches a sampled cell or one of its partners (so the partners' rho, P, c_s are complete too),
    the ghost, the force cycle over every task that touches a sampled cell."""
    from paper_2606_23891_b200 import pipeline as bw, workloads
    orc.set_threads(64)
    ps, cells, tasks, info = workloads.build_clumpy(sph, 4, 1, 1 << 26)
    n_cells, n = int(cells.shape[0]), ps.shape[0]
    layout = sph.sph_layout_split()
    hs = bw.HostStore(sph, torch, layout, ps, cells)
    pl = bw.Pipeline(sph, torch, layout, hs, cells, tasks, n_cells, 4096, "staged", group=bw.CONFIG4_GROUP)      # bench.py's launch configuration
    pl.capture().replay()
    torch.cuda.synchronize()
    pl.close()
    got = np.zeros_like(ps)
    sph.sph_store_export_aos(hs.store, got)
    hs.close()
    # invariants on the full output (north_star: total momentum change <= 1e-6 relative)
    m, a = got["mass"].astype(np.float64), got["a"].astype(np.float64)
    assert np.abs((m[:, None] * a).sum(0)).max() <= 1e-6 * np.abs(m[:, None] * a).sum()
    en = m * (np.einsum("ij,ij->i", got["v"].astype(np.float64), a) + got["du_dt"])
    assert abs(en.sum()) <= 1e-6 * np.abs(m * got["du_dt"].astype(np.float64)).sum()
    # the sample
    rng = np.random.default_rng(2026)
    sample = np.zeros(n_cells, dtype=bool)
    sample[rng.choice(n_cells, 1024, replace=False)] = True
    ci, cj = tasks["ci"].astype(np.int64), np.where(tasks["cj"] < 0, tasks["ci"], tasks["cj"]).astype(np.int64)
    touch_s = sample[ci] | sample[cj]
    ring = sample.copy()
    ring[ci[touch_s]] = True
    ring[cj[touch_s]] = True
    touch_r = ring[ci] | ring[cj]
    oc = cells.view(orc.CELL_DTYPE)
    t_dens, t_force = np.ascontiguousarray(tasks[touch_r]).view(orc.TASK_DTYPE), np.ascontiguousarray(tasks[touch_s]).view(orc.TASK_DTYPE)
    ref = ps                                            # the oracle works in place on the inputs (8.6 GB: no second copy)
    orc.density_cycle(ref, oc, t_dens)
    orc.ghost(ref, GAMMA)
    f_in = orc.pack(ref, oc, t_force, orc.FORCE_IN)
    exempt = orc.flag_cutoff_pairs(oc, t_force, f_in)
    orc.force_cycle(ref, oc, t_force)
    first, count = cells["first"].astype(np.int64), cells["count"].astype(np.int64)
    idx = np.concatenate([np.arange(first[c], first[c] + count[c]) for c in np.flatnonzero(sample)])
    assert idx.shape[0] > 100000
    g, r = got[idx], ref[idx]
    check_store_physics(g, r, a_scale=vec_scale(got["a"]), du_scale=vec_scale(got["du_dt"]))
    ok = np.abs(g["v_sig"] - r["v_sig"]) <= 1e-4 * r["v_sig"]
    assert np.all(ok | exempt[idx]) and exempt[idx].mean() < 0.01


def test_config1_three_loop_step_every_particle():
    """configs[1] through the three-loop cycle (density, ghost, gradient, Balsara-switched force; reading C34), one batch"""
    from test_gpu_parity import check_three_loop, gpu_three_loop_step
    ps, cells, tasks, _ = config1()
    ref = raw_copy(ps)
    orc.density_cycle(ref, cells, tasks)
    orc.ghost(ref, GAMMA)
    orc.gradient_cycle(ref, cells, tasks)
    exempt = orc.flag_cutoff_pairs(cells, tasks, orc.pack(ref, cells, tasks, orc.FORCE_IN))
    orc.force3_cycle(ref, cells, tasks)
    g = GpuCase(ps, cells, tasks, "split")
    check_three_loop(gpu_three_loop_step(g), ref, exempt)
    g.close()


# ------------------------------------------------------------------ extreme occupancy

def test_eagle_like_extreme_occupancy():
    """Cells of 5 .. 20,000 particles in one batch (reduced instance of the Eagle25-like workload): pack and
    unpack byte for byte, the whole step of every particle against the oracle, both layouts.  One block of 20,000 particles
    is 625 chunks for pack / unpack and 313 loop items of 64 x 20,000 candidates each; its neighbours hold a few dozen."""
    orc.set_threads(64)
    parts = si.eagle_like(seed=3, cells_per_dim=4, n_max=20000)
    ps, cells, tasks, n_self, n_pair = sort_grid(parts, 4)
    cnt = cells["count"]
    assert cnt.min() == 5 and cnt.max() == 20000 and (n_self, n_pair) == (64, 64 * 13)
    ref = raw_copy(ps)
    orc.density_cycle(ref, cells, tasks)
    orc.ghost(ref, GAMMA)
    f_in = orc.pack(ref, cells, tasks, orc.FORCE_IN)
    exempt = orc.flag_cutoff_pairs(cells, tasks, f_in)
    orc.force_cycle(ref, cells, tasks)
    for layout in ("split", "aos"):
        g = GpuCase(ps, cells, tasks, layout)
        info = sph.sph_batch_get_info(g.batch)
        assert info.max_count == 20000 and info.max_item_candidates == 64 * 20000
        # pack of the density inputs, byte for byte
        aset = to_attrset(orc.DENSITY_IN)
        want = orc.pack(ps, cells, tasks, orc.DENSITY_IN)
        got = g.pack(aset).cpu().numpy()
        assert got.shape == want.shape and orc.compare_blocks(cells, tasks, 20, got, want) == -1, layout
        # REDUCE unpack of seeded result records, byte for byte
        uset = to_attrset(orc.FORCE_OUT)
        res = _random_result_buffer(sph.sph_batch_buffer_bytes(g.batch, uset), 77)
        want_store = raw_copy(ps)
        orc.unpack(want_store, cells, tasks, orc.FORCE_OUT, res, orc.MODE_REDUCE)
        sph.sph_unpack(g.store, g.batch, uset, torch.from_numpy(res).cuda(), sph.SPH_UNPACK_REDUCE)
        assert np.array_equal(canon(g.export()), canon(want_store)), layout
        # the whole step
        sph.sph_store_import_aos(g.store, ps)
        out = gpu_step(g, fused_zero=True)
        check_store_physics(out, ref)
        ok = np.abs(out["v_sig"] - ref["v_sig"]) <= 1e-4 * ref["v_sig"]
        assert np.all(ok | exempt) and exempt.mean() < 0.01, layout
        m, a = out["mass"].astype(np.float64), out["a"].astype(np.float64)
        assert np.abs((m[:, None] * a).sum(0)).max() <= 1e-6 * np.abs(m[:, None] * a).sum()
        g.close()
