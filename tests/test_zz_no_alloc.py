"""sph_pack_static -- the pack for callers that may not allocate device memory -- against the ordinary sph_pack.

Why the entry point exists: a task-based SPH host (the paper's setting) reserves its device memory once at
start-up and then packs from many worker threads, each on its own stream.  Inside such a worker cudaMalloc / cudaFree is off
limits: it may wait for the whole device (stalling the other workers' streams) and, with the store filling the GPU, it may
fail outright.  sph_batch_create allocates, so those callers get sph_pack_static: same kernel, tables for one call in a
fixed 2.1 MiB array inside the library, at most SPH_PACK_STATIC_MAX_TASKS tasks / SPH_PACK_STATIC_MAX_CHUNKS 32-particle
slices per call.

This file is named to be collected last (pytest -x stops at the first failure, and a failure here should not hide the
parity tests); it builds its own inputs, so it passes alone in a fresh process as well as after the other files.
The bar is the pack bar of tests/test_gpu_parity.py: block bytes identical (pad bytes are unspecified and left out).
"""
import numpy as np
import pytest
import torch

import paper_2606_23891_b200 as sph
import sph_inputs as si
from gpu_setup import GpuCase, valid_mask
from orc_setup import sort_grid, sort_octree


def _seeded_fields(ps, seed):
    rng = np.random.default_rng(seed)
    for name in ("v", "a", "rot_v"):
        ps[name] = rng.standard_normal((ps.shape[0], 3)).astype(np.float32)
    for name in ("u", "rho", "rho_dh", "P", "c_s", "wcount", "div_v"):
        ps[name] = (rng.random(ps.shape[0]) + 0.5).astype(np.float32)
    ps["time_bin"] = rng.integers(-100, 100, ps.shape[0]).astype(np.int8)
    return ps


def _block_bytes(buf, g, tasks, aset):
    """the bytes of a buffer that belong to blocks, with the layout the ordinary path reports for these tasks"""
    batch = sph.sph_batch_create(g.store, tasks)
    off, _ = sph.sph_batch_block_offsets(batch, aset)
    total = sph.sph_batch_buffer_bytes(batch, aset)
    sph.sph_batch_destroy(batch)
    m = valid_mask(off, g.cells, tasks, sph.sph_attrset_record_bytes(aset), total)
    return buf.cpu().numpy()[:total][m], total


def _ordinary_pack(g, tasks, aset):
    batch = sph.sph_batch_create(g.store, tasks)
    buf = torch.full((sph.sph_batch_buffer_bytes(batch, aset),), 0xCD, dtype=torch.uint8, device="cuda")
    sph.sph_pack(g.store, batch, aset, buf)
    torch.cuda.synchronize()
    sph.sph_batch_destroy(batch)
    return buf


@pytest.mark.gpu
@pytest.mark.parametrize("layout", ["aos", "split"])
def test_pack_static_equals_pack_on_two_calls_in_a_row(layout):
    """Two calls back to back on one stream share the scratch array: the second (other tasks, other record, fewer blocks)
    must not see anything of the first, and the first call repeated afterwards gives the first result again."""
    ps, cells, tasks, _, _ = sort_octree(si.clumpy_mixture(20000, seed=5, n_clumps=3, frac_clumps=0.6, sigma=0.05, h_cap=1.0 / 24), 150)
    g = GpuCase(_seeded_fields(ps, 23), cells, tasks, layout)      # cells of 7..1303 particles: many slices, ragged tails
    g.cells = np.ascontiguousarray(cells).view(sph.CELL_DTYPE)
    all_tasks = g.tasks
    some_tasks = np.ascontiguousarray(all_tasks[5::3][::-1])        # another bundle: a subset, in another order
    calls = [(all_tasks, sph.sph_attrset_canonical(sph.SPH_SET_FORCE_IN)),
             (some_tasks, sph.sph_attrset_canonical(sph.SPH_SET_DENSITY_IN)),
             (all_tasks, sph.sph_attrset_canonical(sph.SPH_SET_FORCE_IN)),
             (some_tasks, sph.make_attrset([("v", 1, 2), ("x", 0, 3), ("id", 0, 1), ("time_bin", 0, 1), ("c_s", 0, 1)], 0))]
    # all the new entry point's calls first, back to back, nothing in between ...
    got = []
    for tk, aset in calls:
        need = sph.sph_pack_static(g.store, tk, aset)               # size query
        buf = torch.full((need,), 0xCD, dtype=torch.uint8, device="cuda")
        assert sph.sph_pack_static(g.store, tk, aset, buf) == need
        got.append(buf)
    torch.cuda.synchronize()
    # ... then the ordinary path for the same bundles
    for (tk, aset), buf in zip(calls, got):
        ref = _ordinary_pack(g, tk, aset)
        assert ref.numel() == buf.numel()
        a, total = _block_bytes(buf, g, tk, aset)
        b, _ = _block_bytes(ref, g, tk, aset)
        assert total == buf.numel() and a.size > 0 and np.array_equal(a, b), (layout, tk.shape[0], sph.sph_attrset_record_bytes(aset))
    g.close()


@pytest.mark.gpu
def test_pack_static_rejects_what_does_not_fit():
    """beyond the fixed sizes the call fails before it uploads or launches anything, and says which limit it was"""
    ps, cells, tasks, _, _ = sort_grid(si.config0(seed=1), 4)
    g = GpuCase(ps, cells, tasks, "split")
    aset = sph.sph_attrset_canonical(sph.SPH_SET_DENSITY_IN)
    too_many = np.ascontiguousarray(np.tile(g.tasks, sph.SPH_PACK_STATIC_MAX_TASKS // g.tasks.shape[0] + 1))
    with pytest.raises(sph.SphError) as e:
        sph.sph_pack_static(g.store, too_many, aset)
    assert e.value.code == 3 and "SPH_PACK_STATIC_MAX_TASKS" in str(e.value)
    buf = torch.zeros(sph.sph_pack_static(g.store, g.tasks, aset) - 128, dtype=torch.uint8, device="cuda")
    with pytest.raises(sph.SphError) as e:
        sph.sph_pack_static(g.store, g.tasks, aset, buf)           # buffer one block line short
    assert e.value.code == 3
    g.close()
    # a store whose touched cells hold more 32-particle slices than the scratch has entries for: cells of one particle
    # each cost a whole slice, so MAX_CHUNKS + 1 of them in self tasks is the smallest such input
    n = sph.SPH_PACK_STATIC_MAX_CHUNKS + 1
    lay = sph.sph_layout_split()
    store = sph.sph_store_create(lay, n)
    c = np.zeros(n, dtype=sph.CELL_DTYPE)
    c["first"], c["count"], c["width"] = np.arange(n), 1, 1.0
    sph.sph_store_set_cells(store, c)
    buf = torch.zeros(128 * sph.SPH_PACK_STATIC_MAX_TASKS, dtype=torch.uint8, device="cuda")
    for start in (0, n - sph.SPH_PACK_STATIC_MAX_TASKS):           # any MAX_TASKS self tasks fit ...
        t = np.zeros(sph.SPH_PACK_STATIC_MAX_TASKS, dtype=sph.TASK_DTYPE)
        t["ci"], t["cj"] = np.arange(start, start + t.shape[0]), -1
        assert sph.sph_pack_static(store, t, aset, buf) == buf.numel()
    torch.cuda.synchronize()
    sph.sph_store_destroy(store)
    # ... and a cell table whose few cells are large does not: 3 cells of 2^20 particles = 98,304 slices
    store = sph.sph_store_create(lay, 3 << 20)
    c = np.zeros(3, dtype=sph.CELL_DTYPE)
    c["first"], c["count"], c["width"] = np.arange(3) << 20, 1 << 20, 1.0
    sph.sph_store_set_cells(store, c)
    t = np.zeros(3, dtype=sph.TASK_DTYPE)
    t["ci"], t["cj"] = np.arange(3), -1
    need = sph.sph_pack_static(store, t, aset)                      # the size query still answers
    assert need == 3 * (20 << 20)
    with pytest.raises(sph.SphError) as e:
        sph.sph_pack_static(store, t, aset, torch.zeros(need, dtype=torch.uint8, device="cuda"))
    assert e.value.code == 3 and "SPH_PACK_STATIC_MAX_CHUNKS" in str(e.value)
    sph.sph_store_destroy(store)


def test_pack_static_size_query_and_null_arguments_without_a_device():
    """host logic only (no GPU): a store over caller memory, the size query and the argument checks touch no CUDA call"""
    import ctypes as C
    lay = sph.sph_layout_aos()
    n = 100
    backing = np.zeros(sph.sph_store_sub_bytes(lay, n, 0) + 256, dtype=np.uint8)
    base = (backing.ctypes.data + 255) // 256 * 256
    store = sph.sph_store_create(lay, n, sph.SPH_MEM_HOST_PINNED, [base])
    c = np.zeros(2, dtype=sph.CELL_DTYPE)
    c["first"], c["count"], c["width"] = [0, 37], [37, 63], 0.5
    sph.sph_store_set_cells(store, c)
    t = np.zeros(3, dtype=sph.TASK_DTYPE)
    t["ci"], t["cj"] = [0, 1, 0], [-1, -1, 1]
    aset = sph.sph_attrset_canonical(sph.SPH_SET_FORCE_IN)          # 52-byte records
    blocks = [37, 63, 37, 63]                                        # self 0, self 1, pair (0, 1): blocks start on 128-byte lines
    assert sph.sph_pack_static(store, t, aset) == sum((k * 52 + 127) // 128 * 128 for k in blocks)
    lib = C.CDLL(sph.lib_path())
    lib.sph_pack_static.restype = C.c_int32
    need = C.c_uint64(0)
    args = lambda st, tk, se, out: (st, tk, C.c_uint32(3), se, None, C.c_uint64(0), out, None)
    tp = C.c_void_p(t.ctypes.data)
    assert lib.sph_pack_static(*args(None, tp, C.byref(aset), C.byref(need))) == 1
    assert lib.sph_pack_static(*args(store, None, C.byref(aset), C.byref(need))) == 1
    assert lib.sph_pack_static(*args(store, tp, None, C.byref(need))) == 1
    assert lib.sph_pack_static(*args(store, tp, C.byref(aset), None)) == 1          # no buffer and nowhere to put the size
    t["cj"][2] = 2
    with pytest.raises(sph.SphError) as e:
        sph.sph_pack_static(store, t, aset)                         # a task that names a cell the store does not have
    assert e.value.code == 3
    sph.sph_store_destroy(store)
