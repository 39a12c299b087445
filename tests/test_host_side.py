"""Host logic of the library (no GPU): exported symbols, layouts, attribute sets, cell / task builders.

The builders are cross-checked against the oracle's independent ones: same permutation, same cells, same
task list and frames.
"""
import ctypes
import re
import os

import numpy as np
import pytest

import oracle as orc
import paper_2606_23891_b200 as sph
import sph_inputs as si

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "sph_b200.h")).read()
    declared = set(re.findall(r"^int32_t\s+(sph_\w+)\s*\(", header, flags=re.M))
    assert declared == set(sph.EXPORTS)
    lib = ctypes.CDLL(sph.lib_path())
    for name in declared:
        assert hasattr(lib, name), name


def test_slot_attribute_sets():
    """cell-slot records (row f4): the loop's input set with x as raw f64 and time_bin as a last word -- 9 and 17 words"""
    for loop, (nbytes, canon) in enumerate(((36, sph.SPH_SET_DENSITY_IN), (68, sph.SPH_SET_FORCE_IN))):
        s, c = sph.sph_slot_attrset(loop), sph.sph_attrset_canonical(canon)
        assert sph.sph_attrset_record_bytes(s) == nbytes and s.flags == 0 and s.n == c.n + 1
        assert [int(e.field) for e in list(s.ent)[:c.n]] == [int(e.field) for e in list(c.ent)[:c.n]]
        assert int(s.ent[c.n].field) == sph.FIELD["time_bin"]
    with pytest.raises(sph.SphError):
        sph.sph_slot_attrset(2)


def test_split_pack_loop_partitions():
    """row f4 / PAPER.md:150-152: the passes of every split are a partition of the record's words"""
    f_in = sph.sph_attrset_canonical(sph.SPH_SET_FORCE_IN)          # x(3) h m rho rho_dh v(3) u P cs: 13 words
    split, aos = sph.sph_layout_split(), sph.sph_layout_aos()
    for lay in (split, aos):
        for mode in range(4):
            masks = sph.sph_pack_pass_masks(lay, f_in, mode)
            assert sum(masks) == (1 << 13) - 1 and all(a & b == 0 for i, a in enumerate(masks) for b in masks[i + 1:])
    # split-AoS: x h m in S0, rho rho_dh in S1, v u P cs in S2; AoS: one struct
    assert sph.sph_pack_pass_masks(split, f_in, sph.SPLIT_BY_STRUCT) == [0b0000000011111, 0b0000001100000, 0b1111110000000]
    assert sph.sph_pack_pass_masks(aos, f_in, sph.SPLIT_BY_STRUCT) == [(1 << 13) - 1]
    assert len(sph.sph_pack_pass_masks(split, f_in, sph.SPLIT_BY_ELEMENT)) == 9
    assert sph.sph_pack_pass_masks(aos, f_in, sph.SPLIT_BY_TYPE) == [0b111, ((1 << 13) - 1) ^ 0b111]            # f64 coordinates, f32 rest
    assert len(sph.sph_pack_pass_masks(split, f_in, sph.SPLIT_BY_STRUCT_AND_TYPE)) == 4
    with pytest.raises(sph.SphError):
        sph.sph_pack_pass_masks(split, f_in, 4)


def test_library_is_built_for_sm_100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", sph.lib_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, out


def test_layouts():
    aos, split = sph.sph_layout_aos(), sph.sph_layout_split()
    assert aos.n_sub == 1 and aos.stride[0] == 128
    # canonical offsets = the numpy dtype both sides use as exchange format
    for f, name in enumerate(si.FIELDS):
        assert aos.loc[f].off == si.PART_DTYPE.fields[name][1] and aos.loc[f].sub == 0
    assert split.n_sub == 6 and list(split.stride)[:6] == [32, 16, 24, 20, 16, 16]      # 124 bytes of payload
    groups = {0: ["x", "h", "mass"], 1: ["rho", "rho_dh", "wcount", "wcount_dh"], 2: ["v", "u", "P", "c_s"],
              3: ["a", "du_dt", "v_sig"], 4: ["id", "time_bin"], 5: ["div_v", "rot_v"]}
    for s, names in groups.items():
        for name in names:
            assert split.loc[sph.FIELD[name]].sub == s
    sph.sph_layout_validate(aos)
    sph.sph_layout_validate(split)
    bad = sph.sph_layout_split()
    bad.loc[sph.FIELD["h"]].off = 20          # overlaps x[2]
    with pytest.raises(sph.SphError) as e:
        sph.sph_layout_validate(bad)
    assert e.value.code == 2
    bad = sph.sph_layout_aos()
    bad.loc[sph.FIELD["id"]].off = 124        # runs past the stride
    with pytest.raises(sph.SphError):
        sph.sph_layout_validate(bad)
    bad = sph.sph_layout_aos()
    bad.n_sub = 9
    with pytest.raises(sph.SphError):
        sph.sph_layout_validate(bad)


def test_paper_layout_variants():
    """random-order AoS, kernel-driven sAoS variants and their splits by type, via sph_layout_from_groups"""
    from paper_2606_23891_b200 import layouts
    sizes = {"x": 24, "v": 12, "a": 12, "rot_v": 12, "id": 8, "time_bin": 1}
    for name, loops in [(n, 2) for n in layouts.NAMES] + [(n, 3) for n in layouts.NAMES3]:
        lay = layouts.layout(sph, name, seed=3, loops=loops)
        sph.sph_layout_validate(lay)
        spans = {}
        for fname, f in sph.FIELD.items():
            loc = lay.loc[f]
            nb = sizes.get(fname, 4)
            assert loc.sub < lay.n_sub and loc.off + nb <= lay.stride[loc.sub], (name, fname)
            spans.setdefault(loc.sub, []).append((loc.off, loc.off + nb))
        for sub, sp in spans.items():                      # no two members overlap
            sp.sort()
            assert all(a[1] <= b[0] for a, b in zip(sp[:-1], sp[1:])), (name, sub)
    # the density inputs of pack-force live in the 64-byte force struct; pack-density keeps them in a 32-byte one
    pf, pd = layouts.layout(sph, "pack-force"), layouts.layout(sph, "pack-density")
    assert pf.stride[pf.loc[sph.FIELD["x"]].sub] == 64 and pd.stride[pd.loc[sph.FIELD["x"]].sub] == 32
    assert {pf.loc[sph.FIELD[k]].sub for k in ("x", "h", "mass", "rho", "rho_dh", "v", "u", "P", "c_s")} == {0}
    # three-loop flavours: pack-gradient keeps the six gradient inputs in one 48-byte struct, pack-force all twelve
    # force inputs in one, pack-shared puts what all three packs share, what gradient and force share and the force-only rest apart
    F = sph.FIELD
    G_IN = ("x", "v", "mass", "h", "u", "rho")
    F_ONLY = ("rho_dh", "P", "c_s", "div_v", "rot_v", "time_bin")
    pg, pf3, psh = (layouts.layout(sph, k, loops=3) for k in ("pack-gradient", "pack-force", "pack-shared"))
    assert {pg.loc[F[k]].sub for k in G_IN} == {0} and pg.stride[0] == 56 and {pg.loc[F[k]].sub for k in F_ONLY} == {1}
    assert {pf3.loc[F[k]].sub for k in G_IN + F_ONLY} == {0}
    assert [len({psh.loc[F[k]].sub for k in grp}) for grp in (("x", "h", "mass"), ("v", "u", "rho"), F_ONLY)] == [1, 1, 1]
    assert len({psh.loc[F[k]].sub for k in ("x", "v", "rho_dh")}) == 3
    pgt = layouts.layout(sph, "pack-gradient-type", loops=3)
    assert pgt.stride[pgt.loc[F["x"]].sub] == 24 and pgt.stride[pgt.loc[F["time_bin"]].sub] <= 4
    ro = layouts.layout(sph, "random-order", seed=3)
    assert ro.n_sub == 1 and ro.stride[0] == 128
    assert [ro.loc[f].off for f in range(18)] != [sph.sph_layout_aos().loc[f].off for f in range(18)]
    with pytest.raises(sph.SphError):                      # a field twice
        sph.sph_layout_from_groups([["x", "x"] + layouts.AOS_ORDER[2:]])
    with pytest.raises(sph.SphError):                      # a field missing
        sph.sph_layout_from_groups([layouts.AOS_ORDER[:-1]])
    with pytest.raises(sph.SphError):                      # more substructs than SPH_MAX_SUB
        sph.sph_layout_from_groups([[f] for f in layouts.AOS_ORDER[:9]] + [layouts.AOS_ORDER[9:]])


def test_attribute_sets():
    for which, rec, oset in [(sph.SPH_SET_DENSITY_IN, 20, orc.DENSITY_IN), (sph.SPH_SET_DENSITY_OUT, 16, orc.DENSITY_OUT),
                             (sph.SPH_SET_FORCE_IN, 52, orc.FORCE_IN), (sph.SPH_SET_FORCE_OUT, 20, orc.FORCE_OUT)]:
        a = sph.sph_attrset_canonical(which)
        assert sph.sph_attrset_record_bytes(a) == rec == orc.record_bytes(oset)
        assert [(a.ent[k].field, a.ent[k].comp0, a.ent[k].ncomp) for k in range(a.n)] == [tuple(e) for e in oset[0]]
        assert a.flags == oset[1]
    assert sph.sph_attrset_record_bytes(sph.make_attrset([("x", 0, 3), ("id", 0, 1), ("time_bin", 0, 1)])) == 36
    for entries in ([("v", 0, 2), ("v", 1, 1)], [("mass", 0, 2)], [(18, 0, 1)], []):
        with pytest.raises(sph.SphError) as e:
            sph.sph_attrset_record_bytes(sph.make_attrset(entries))
        assert e.value.code == 2


def test_store_sub_bytes_and_errors():
    split = sph.sph_layout_split()
    assert sph.sph_store_sub_bytes(split, 1000, 3) >= 1000 * 20 + 64
    assert sph.sph_store_sub_bytes(split, 1000, 3) % 256 == 0
    with pytest.raises(sph.SphError) as e:
        sph.sph_store_sub_bytes(split, 1000, 6)
    assert e.value.code == 3 and "substruct" in str(e.value)


@pytest.mark.parametrize("cpd,n_side,seed", [(4, 12, 1), (3, 10, 2), (5, 11, 3)])
def test_grid_builder_matches_oracle(cpd, n_side, seed):
    parts = si.jittered_lattice(n_side, seed, jitter=0.9)
    perm_o, cells_o = orc.cells_build_grid(parts["x"], cpd)
    perm, cells = sph.sph_cells_build_grid(parts["x"], cpd)
    assert np.array_equal(perm, perm_o)
    assert cells.tobytes() == cells_o.tobytes()
    ps = parts[perm.astype(np.int64)]
    hmax = orc.cell_hmax(ps, cells_o)
    tasks_o, ns_o, np_o = orc.tasks_build(cells_o, hmax)
    tasks, ns, npair = sph.sph_tasks_build(cells, hmax)
    assert (ns, npair) == (ns_o, np_o)
    assert tasks.tobytes() == tasks_o.tobytes()


def test_task_rule_with_large_h_matches_oracle():
    parts = si.jittered_lattice(12, 4, jitter=0.3, eta=1.1 / 1.0, h_spread=0.3)      # 2h up to ~2.5 dx > width 2 dx
    perm, cells = sph.sph_cells_build_grid(parts["x"], 6)
    ps = parts[perm.astype(np.int64)]
    hmax = orc.cell_hmax(ps, cells)
    tasks_o, ns_o, np_o = orc.tasks_build(cells.view(orc.CELL_DTYPE), hmax)
    tasks, ns, npair = sph.sph_tasks_build(cells, hmax)
    assert npair == np_o > 216 * 13
    assert tasks.tobytes() == tasks_o.tobytes()


def test_tasks_reject_box_too_small_for_cutoff():
    parts = si.jittered_lattice(6, 5, eta=1.2348)
    parts["h"] = 0.2                           # 2h = 0.4: with 3 cells per dim a second image is within reach
    perm, cells = sph.sph_cells_build_grid(parts["x"], 3)
    hmax = orc.cell_hmax(parts[perm.astype(np.int64)], cells)
    with pytest.raises(sph.SphError) as e:
        sph.sph_tasks_build(cells, hmax)
    assert e.value.code == 3
    with pytest.raises(ValueError):
        orc.tasks_build(cells.view(orc.CELL_DTYPE), hmax)


@pytest.mark.parametrize("seed,leaf", [(3, 100), (6, 37)])
def test_octree_builder_matches_oracle(seed, leaf):
    parts = si.clumpy_mixture(20000, seed=seed, n_clumps=4, frac_clumps=0.7, sigma=0.03, h_cap=1.0 / 32)
    perm_o, cells_o = orc.cells_build_octree(parts["x"], parts["h"], leaf)
    perm, cells = sph.sph_cells_build_octree(parts["x"], parts["h"], leaf)
    assert np.array_equal(perm, perm_o)
    assert cells.tobytes() == cells_o.tobytes()
    ps = parts[perm.astype(np.int64)]
    hmax = orc.cell_hmax(ps, cells_o)
    tasks_o, ns_o, np_o = orc.tasks_build(cells_o, hmax)
    tasks, ns, npair = sph.sph_tasks_build(cells, hmax)
    assert (ns, npair) == (ns_o, np_o)
    assert tasks.tobytes() == tasks_o.tobytes()


def test_grid_builder_rejects_out_of_box():
    x = np.array([[0.1, 0.2, 1.0]])
    with pytest.raises(sph.SphError) as e:
        sph.sph_cells_build_grid(x, 4)
    assert e.value.code == 3


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(sph.SphError) as e:
        sph.sph_store_create(sph.sph_layout_aos(), 128)
    assert e.value.code == 5


def _host_store(n, layout=None):
    """a store over caller-owned (numpy) memory: no CUDA call is made, so the host-side checks run without a device"""
    layout = layout or sph.sph_layout_aos()
    bufs = []
    for s in range(layout.n_sub):
        raw = np.zeros(sph.sph_store_sub_bytes(layout, n, s) + 256, dtype=np.uint8)
        off = (-raw.ctypes.data) % 256
        bufs.append(raw[off:off + sph.sph_store_sub_bytes(layout, n, s)])
    return sph.sph_store_create(layout, n, sph.SPH_MEM_HOST_PINNED, ext=bufs), bufs


def test_cell_table_checks_do_not_wrap():
    store, keep = _host_store(100)
    cells = np.zeros(3, dtype=sph.CELL_DTYPE)
    cells["first"], cells["count"], cells["width"] = [0, 40, 70], [40, 30, 30], 1.0
    sph.sph_store_set_cells(store, cells)
    for first, count in [(2 ** 64 - 10, 30), (90, 30), (101, 0)]:          # a huge `first` must not wrap around the range check
        bad = cells.copy()
        bad["first"][2], bad["count"][2] = first, count
        with pytest.raises(sph.SphError) as e:
            sph.sph_store_set_cells(store, bad)
        assert e.value.code == 3
    bad = cells.copy()
    bad["first"][1] = 39                                                    # overlaps cell 0
    with pytest.raises(sph.SphError) as e:
        sph.sph_store_set_cells(store, bad)
    assert e.value.code == 3
    sph.sph_store_destroy(store)


def test_null_arguments_are_errors_not_crashes():
    import ctypes as C
    lib = C.CDLL(sph.lib_path())
    store, keep = _host_store(64)
    aset = sph.sph_attrset_canonical(sph.SPH_SET_DENSITY_IN)
    out = C.c_uint64(0)
    fake = C.c_void_p(keep[0].ctypes.data)                                   # any non-NULL buffer pointer
    assert lib.sph_batch_buffer_bytes(None, C.byref(aset), C.byref(out)) == 1
    assert lib.sph_pack(store, None, C.byref(aset), fake, C.c_uint64(1024), None) == 1
    assert lib.sph_pack(None, None, None, None, C.c_uint64(0), None) == 1
    assert lib.sph_unpack(store, None, None, fake, C.c_uint64(1024), C.c_int32(0), None) == 1
    assert lib.sph_density(None, fake, C.c_uint64(0), fake, C.c_uint64(0), None) == 1
    assert lib.sph_force(None, fake, C.c_uint64(0), fake, C.c_uint64(0), None, None) == 1
    assert lib.sph_store_zero(store, None, None) == 1
    assert lib.sph_store_set_cells(store, None, C.c_uint32(3)) == 1
    assert lib.sph_batch_create(store, None, C.c_uint64(1), C.c_uint32(0), C.byref(C.c_void_p())) == 1
    assert "NULL" in sph.sph_last_error() or "no tasks" in sph.sph_last_error()
    # the row (f4) entry points check their arguments the same way
    assert lib.sph_batch_slot_bytes(None, C.c_int32(0), C.byref(out)) == 1
    assert lib.sph_pack_slots(store, None, C.c_int32(0), fake, C.c_uint64(1024), None) == 1
    assert lib.sph_density_slots(None, fake, C.c_uint64(0), fake, C.c_uint64(0), None) == 1
    assert lib.sph_force_slots(None, fake, C.c_uint64(0), fake, C.c_uint64(0), None, None) == 1
    assert lib.sph_pack_pass(store, None, C.byref(aset), C.c_uint64(1), fake, C.c_uint64(1024), None) == 1
    assert lib.sph_pack_pass_masks(None, C.byref(aset), C.c_int32(0), None, None) == 1
    masks, n_masks = (C.c_uint64 * 48)(), C.c_uint32(0)
    assert lib.sph_pack_pass_masks(C.byref(sph.sph_layout_aos()), None, C.c_int32(0), masks, C.byref(n_masks)) == 1      # NULL set
    assert lib.sph_slot_attrset(C.c_int32(0), None) == 1
    sph.sph_store_destroy(store)


def test_batch_rejects_a_cell_too_large_for_the_item_tables():
    """a loop item holds its source count in 25 bits: a cell of 2^25 particles is an error, not a silently cut count"""
    import ctypes as C
    n = 1 << 25
    raw = np.zeros(512, dtype=np.uint8)                       # never touched: the check comes before any table is built
    base = (raw.ctypes.data + 255) // 256 * 256
    store = sph.sph_store_create(sph.sph_layout_aos(), n, sph.SPH_MEM_HOST_PINNED, ext=[base])
    cells = np.zeros(1, dtype=sph.CELL_DTYPE)
    cells["first"], cells["count"], cells["width"] = 0, n, 1.0
    sph.sph_store_set_cells(store, cells)
    task = np.zeros(1, dtype=sph.TASK_DTYPE)
    task["ci"], task["cj"] = 0, -1
    with pytest.raises(sph.SphError) as e:
        sph.sph_batch_create(store, task)
    assert e.value.code == 3 and "2^25" in str(e.value)
    sph.sph_store_destroy(store)


def test_tasks_reject_a_cell_that_sees_its_own_image():
    # one cell per dimension: the self task is not periodic, so neighbours through the wrap would be lost silently
    x = np.random.default_rng(1).random((50, 3))
    perm, cells = sph.sph_cells_build_grid(x, 1)
    with pytest.raises(sph.SphError) as e:
        sph.sph_tasks_build(cells, np.array([0.05], dtype=np.float32))
    assert e.value.code == 3 and "own periodic image" in str(e.value)
    # two cells per dimension, 2 hmax = 0.6 > box - width = 0.5: the same
    perm, cells = sph.sph_cells_build_grid(x, 2)
    with pytest.raises(sph.SphError) as e:
        sph.sph_tasks_build(cells, np.full(8, 0.3, dtype=np.float32))
    assert e.value.code == 3


def test_eagle_like_occupancies_have_the_papers_statistics():
    """row (f3), reading C37: PAPER.md:164 gives per-cell min 5, max 125,113, mean 184, median 109 for Eagle25"""
    c = si.eagle_like_counts(seed=1, n_cells=32 ** 3)
    assert c.min() == 5 and c.max() == 125113
    assert 100 <= np.median(c) <= 118 and 170 <= c.mean() <= 200
    small = si.eagle_like(seed=3, cells_per_dim=4, n_max=20000)
    perm, cells = sph.sph_cells_build_grid(small["x"], 4)
    assert cells["count"].min() == 5 and cells["count"].max() == 20000 and int(cells["count"].sum()) == small.shape[0]
    # a cell's particles keep h <= half the cell width, so the 27-cell stencil holds whatever the occupancy
    assert float(small["h"].max()) < 0.5 * 0.25
    assert np.array_equal(np.sort(small["id"]), np.arange(small.shape[0]))


def test_synthetic_trace_covers_every_task_once_per_loop_and_step():
    """row (f3), reading C38: every bundle of a step is packed and unpacked once per loop, density before force, self before pair"""
    n_tasks, n_self = 5000, 700
    trace = si.synthetic_trace(n_tasks, n_self, seed=7, steps=3)
    for st in range(3):
        for loop in ("density", "force"):
            for action in ("pack", "unpack"):
                rows = [(t0, m) for s_, l_, a_, t0, m in trace if (s_, l_, a_) == (st, loop, action)]
                covered = np.zeros(n_tasks, dtype=int)
                for t0, m in rows:
                    covered[t0:t0 + m] += 1
                    assert 1 <= m <= 1024 and (t0 + m <= n_self or t0 >= n_self)        # homogeneous bundles (C22)
                assert np.all(covered == 1)
    order = [(s_, l_) for s_, l_, _, _, _ in trace]
    assert order == sorted(order, key=lambda x: (x[0], x[1] != "density"))
    assert trace == si.synthetic_trace(n_tasks, n_self, seed=7, steps=3) and trace != si.synthetic_trace(n_tasks, n_self, seed=8, steps=3)


def test_cell_slabs_cover_the_cell_table_in_order():
    from paper_2606_23891_b200 import pipeline as bw
    cells = np.zeros(1000, dtype=sph.CELL_DTYPE)
    rng = np.random.default_rng(3)
    cells["count"] = rng.integers(1, 200, 1000)
    cells["first"] = np.concatenate([[0], np.cumsum(cells["count"])[:-1]])
    for slabs in (bw.cell_slabs(cells, 16), bw.cell_slabs(cells, fractions=(3, 1, 2, 2, 4, 4))):
        assert slabs[0][0] == 0 and sum(s[1] for s in slabs) == 1000 and sum(s[3] for s in slabs) == int(cells["count"].sum())
        for (c0, nc, p0, npart), nxt in zip(slabs, slabs[1:] + [None]):
            assert p0 == int(cells["first"][c0]) and npart == int(cells["count"][c0:c0 + nc].sum())
            assert nxt is None or nxt[0] == c0 + nc
    big = bw.cell_slabs(cells, fractions=(3, 1, 2, 2, 4, 4))
    assert big[0][3] > 2 * big[1][3] and big[-1][3] > big[2][3]
