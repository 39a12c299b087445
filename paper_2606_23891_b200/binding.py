"""ctypes binding of libsph_b200.so -- one Python function per C entry point, same name.

Only argument marshalling happens here: numpy arrays / torch tensors become pointers, status codes become
exceptions.  There is no Python or CPU implementation of any step: if the shared library cannot be loaded
the import fails.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

__all__ = [
    "SphError", "lib_path", "sph_layout", "sph_attr", "sph_attrset", "sph_params", "sph_batch_info", "CELL_DTYPE", "TASK_DTYPE",
    "FIELD", "SPH_ATTR_X_REL_F32", "SPH_MEM_DEVICE", "SPH_MEM_HOST_PINNED", "SPH_UNPACK_REDUCE", "SPH_UNPACK_ASSIGN", "SPH_UNPACK_REDUCE_ZERO",
    "SPH_SET_DENSITY_IN", "SPH_SET_DENSITY_OUT", "SPH_SET_FORCE_IN", "SPH_SET_FORCE_OUT", "EXPORTS",
    "sph_last_error", "sph_layout_aos", "sph_layout_split", "sph_layout_validate", "sph_layout_from_groups", "sph_attrset_canonical", "make_attrset",
    "sph_attrset_record_bytes", "sph_store_sub_bytes", "sph_store_create", "sph_store_destroy", "sph_store_import_aos",
    "sph_store_export_aos", "sph_store_set_cells", "sph_store_sub_ptr", "sph_store_upload_sub", "sph_store_download_sub",
    "sph_store_upload_range", "sph_store_download_range",
    "sph_cells_build_grid", "sph_cells_build_octree", "sph_tasks_build", "sph_batch_create", "sph_batch_destroy", "sph_batch_get_info", "sph_batch_buffer_bytes",
    "sph_batch_block_offsets", "sph_store_zero", "sph_pack", "sph_pack_cells", "sph_density", "sph_force", "sph_gradient", "sph_force3", "sph_unpack",
    "sph_unpack_cells", "sph_ghost", "SPH_SET_GRADIENT_IN", "SPH_SET_GRADIENT_OUT", "SPH_SET_FORCE3_IN",
    "sph_slot_attrset", "sph_batch_slot_bytes", "sph_pack_slots", "sph_density_slots", "sph_force_slots", "sph_pack_pass_masks", "sph_pack_pass",
    "sph_pack_static", "SPH_PACK_STATIC_MAX_TASKS", "SPH_PACK_STATIC_MAX_CHUNKS",
    "SPLIT_BY_STRUCT", "SPLIT_BY_ELEMENT", "SPLIT_BY_TYPE", "SPLIT_BY_STRUCT_AND_TYPE",
]

SPH_NFIELDS, SPH_MAX_SUB, SPH_MAX_ATTR = 18, 8, 32
FIELD = {name: i for i, name in enumerate(
    ["x", "v", "a", "mass", "h", "u", "du_dt", "rho", "rho_dh", "wcount", "wcount_dh", "div_v", "rot_v", "P", "c_s", "v_sig",
     "id", "time_bin"])}
SPH_ATTR_X_REL_F32 = 1
SPH_MEM_DEVICE, SPH_MEM_HOST_PINNED = 0, 1
SPH_UNPACK_REDUCE, SPH_UNPACK_ASSIGN, SPH_UNPACK_REDUCE_ZERO = 0, 1, 2
SPH_SET_DENSITY_IN, SPH_SET_DENSITY_OUT, SPH_SET_FORCE_IN, SPH_SET_FORCE_OUT = 0, 1, 2, 3
SPH_SET_GRADIENT_IN, SPH_SET_GRADIENT_OUT, SPH_SET_FORCE3_IN = 4, 5, 6

#: every symbol include/sph_b200.h declares
EXPORTS = [
    "sph_last_error", "sph_layout_aos", "sph_layout_split", "sph_layout_validate", "sph_layout_from_groups", "sph_attrset_canonical",
    "sph_attrset_record_bytes", "sph_store_sub_bytes", "sph_store_create", "sph_store_destroy", "sph_store_import_aos",
    "sph_store_export_aos", "sph_store_set_cells", "sph_store_sub_ptr", "sph_store_upload_sub", "sph_store_download_sub",
    "sph_store_upload_range", "sph_store_download_range", "sph_pack_cells", "sph_unpack_cells",
    "sph_cells_build_grid", "sph_cells_build_octree", "sph_tasks_build", "sph_free", "sph_batch_create", "sph_batch_destroy", "sph_batch_get_info", "sph_batch_buffer_bytes",
    "sph_batch_block_offsets", "sph_store_zero", "sph_pack", "sph_density", "sph_force", "sph_gradient", "sph_force3", "sph_unpack", "sph_ghost",
    "sph_slot_attrset", "sph_batch_slot_bytes", "sph_pack_slots", "sph_density_slots", "sph_force_slots", "sph_pack_pass_masks", "sph_pack_pass",
    "sph_pack_static",
]


class _Loc(C.Structure):
    _fields_ = [("sub", C.c_uint8), ("pad", C.c_uint8), ("off", C.c_uint16)]


class sph_layout(C.Structure):
    _fields_ = [("n_sub", C.c_uint32), ("stride", C.c_uint32 * SPH_MAX_SUB), ("loc", _Loc * SPH_NFIELDS)]


class sph_attr(C.Structure):
    _fields_ = [("field", C.c_uint8), ("comp0", C.c_uint8), ("ncomp", C.c_uint8), ("pad", C.c_uint8)]


class sph_attrset(C.Structure):
    _fields_ = [("n", C.c_uint32), ("flags", C.c_uint32), ("ent", sph_attr * SPH_MAX_ATTR)]


class sph_params(C.Structure):
    _fields_ = [("gamma", C.c_float), ("alpha", C.c_float), ("beta", C.c_float)]


class sph_batch_info(C.Structure):
    _fields_ = [("n_tasks", C.c_uint64), ("n_self", C.c_uint64), ("n_pair", C.c_uint64), ("n_sides", C.c_uint64),
                ("n_instances", C.c_uint64), ("n_candidates", C.c_uint64), ("n_cells_touched", C.c_uint64),
                ("n_segments", C.c_uint32), ("max_count", C.c_uint32), ("n_items", C.c_uint64), ("max_item_candidates", C.c_uint64)]


CELL_DTYPE = np.dtype({"names": ["first", "count", "pad", "origin", "width"],
                       "formats": ["<u8", "<u4", "<u4", ("<f8", (3,)), "<f8"], "offsets": [0, 8, 12, 16, 40], "itemsize": 48})
TASK_DTYPE = np.dtype({"names": ["ci", "cj", "frame_i", "frame_j"],
                       "formats": ["<i4", "<i4", ("<f8", (3,)), ("<f8", (3,))], "offsets": [0, 4, 8, 32], "itemsize": 56})


class SphError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libsph_b200 error {code}: {msg}")
        self.code = code


def lib_path() -> str:
    return _build.LIB


def _load():
    path = os.environ.get("SPH_B200_LIB") or _build.build()   # (re)builds with nvcc when sources are newer; raises if that is impossible
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2606_23891_b200.build`")
    lib = C.CDLL(path)
    for name in EXPORTS:
        getattr(lib, name).restype = C.c_int32      # AttributeError here = a declared symbol is not exported
    return lib


_lib = _load()


def _check(rc):
    if rc != 0:
        buf = C.create_string_buffer(512)
        _lib.sph_last_error(buf, C.c_size_t(512))
        raise SphError(rc, buf.value.decode(errors="replace"))


def _ptr(x):
    """host numpy array / torch tensor / int / None -> void*"""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        return C.c_void_p(x.ctypes.data)
    if hasattr(x, "data_ptr"):
        return C.c_void_p(x.data_ptr())
    return C.c_void_p(int(x))


def _ref(struct):
    """ctypes structure or None -> pointer argument"""
    return None if struct is None else C.byref(struct)


def _nbytes(x):
    if isinstance(x, np.ndarray):
        return x.nbytes
    return x.numel() * x.element_size()


def _stream(stream):
    if stream is None:
        return None
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def sph_last_error() -> str:
    buf = C.create_string_buffer(512)
    _lib.sph_last_error(buf, C.c_size_t(512))
    return buf.value.decode(errors="replace")


def sph_layout_aos() -> sph_layout:
    out = sph_layout()
    _check(_lib.sph_layout_aos(C.byref(out)))
    return out


def sph_layout_split() -> sph_layout:
    out = sph_layout()
    _check(_lib.sph_layout_split(C.byref(out)))
    return out


def sph_layout_validate(layout: sph_layout) -> None:
    _check(_lib.sph_layout_validate(C.byref(layout)))


def sph_layout_from_groups(groups, min_stride=None) -> sph_layout:
    """groups: list of lists of field ids or names, every field exactly once; min_stride: optional stride floor per group"""
    flat = np.array([FIELD[f] if isinstance(f, str) else int(f) for g in groups for f in g], dtype=np.uint8)
    sizes = np.array([len(g) for g in groups], dtype=np.uint32)
    ms = None if min_stride is None else np.ascontiguousarray(min_stride, dtype=np.uint32)
    out = sph_layout()
    _check(_lib.sph_layout_from_groups(_ptr(flat), C.c_uint32(flat.shape[0]), _ptr(sizes), C.c_uint32(sizes.shape[0]),
                                       _ptr(ms) if ms is not None else None, C.byref(out)))
    return out


def sph_attrset_canonical(which: int) -> sph_attrset:
    out = sph_attrset()
    _check(_lib.sph_attrset_canonical(C.c_int32(which), C.byref(out)))
    return out


def make_attrset(entries, flags: int = 0) -> sph_attrset:
    """entries: list of (field, comp0, ncomp) with field an id or a name."""
    out = sph_attrset()
    out.n, out.flags = len(entries), flags
    if len(entries) > SPH_MAX_ATTR:
        raise SphError(2, "too many entries")
    for k, (f, c0, nc) in enumerate(entries):
        out.ent[k] = sph_attr(FIELD[f] if isinstance(f, str) else f, c0, nc, 0)
    return out


def sph_attrset_record_bytes(aset: sph_attrset) -> int:
    out = C.c_uint32(0)
    _check(_lib.sph_attrset_record_bytes(C.byref(aset), C.byref(out)))
    return out.value


def sph_store_sub_bytes(layout: sph_layout, n: int, sub: int) -> int:
    out = C.c_uint64(0)
    _check(_lib.sph_store_sub_bytes(C.byref(layout), C.c_uint64(n), C.c_uint32(sub), C.byref(out)))
    return out.value


def sph_store_create(layout: sph_layout, n: int, mem_kind: int = SPH_MEM_DEVICE, ext=None):
    """ext: optional list of n_sub caller-owned buffers (torch tensors); returns the store handle."""
    handle = C.c_void_p()
    arr = None
    if ext is not None:
        arr = (C.c_void_p * layout.n_sub)(*[_ptr(t) for t in ext])
    _check(_lib.sph_store_create(C.byref(layout), C.c_uint64(n), C.c_int32(mem_kind), arr, C.byref(handle)))
    return handle


def sph_store_destroy(store) -> None:
    _check(_lib.sph_store_destroy(store))


def sph_store_import_aos(store, parts: np.ndarray) -> None:
    assert parts.dtype.itemsize == 128 and parts.flags.c_contiguous
    _check(_lib.sph_store_import_aos(store, _ptr(parts), C.c_uint64(parts.shape[0])))


def sph_store_export_aos(store, parts_out: np.ndarray) -> np.ndarray:
    assert parts_out.dtype.itemsize == 128 and parts_out.flags.c_contiguous
    _check(_lib.sph_store_export_aos(store, _ptr(parts_out), C.c_uint64(parts_out.shape[0])))
    return parts_out


def sph_store_set_cells(store, cells: np.ndarray) -> None:
    assert cells.dtype.itemsize == 48 and cells.flags.c_contiguous
    _check(_lib.sph_store_set_cells(store, _ptr(cells), C.c_uint32(cells.shape[0])))


def sph_store_sub_ptr(store, sub: int) -> int:
    out = C.c_void_p()
    _check(_lib.sph_store_sub_ptr(store, C.c_uint32(sub), C.byref(out)))
    return out.value


def sph_store_upload_sub(store, sub: int, host_src, stream=None) -> None:
    _check(_lib.sph_store_upload_sub(store, C.c_uint32(sub), _ptr(host_src), C.c_uint64(_nbytes(host_src)), _stream(stream)))


def sph_store_download_sub(store, sub: int, host_dst, stream=None) -> None:
    _check(_lib.sph_store_download_sub(store, C.c_uint32(sub), _ptr(host_dst), C.c_uint64(_nbytes(host_dst)), _stream(stream)))


def sph_store_upload_range(store, sub: int, host_base, first: int, count: int, stream=None) -> None:
    """host_base: the whole host substruct array; particles [first, first + count) are copied"""
    _check(_lib.sph_store_upload_range(store, C.c_uint32(sub), _ptr(host_base), C.c_uint64(first), C.c_uint64(count), _stream(stream)))


def sph_store_download_range(store, sub: int, host_base, first: int, count: int, stream=None) -> None:
    _check(_lib.sph_store_download_range(store, C.c_uint32(sub), _ptr(host_base), C.c_uint64(first), C.c_uint64(count), _stream(stream)))


def sph_cells_build_grid(x: np.ndarray, cells_per_dim: int, box: float = 1.0):
    """-> (perm u64[n], cells[cells_per_dim^3])"""
    x = np.ascontiguousarray(x, dtype=np.float64)
    perm = np.empty(x.shape[0], dtype=np.uint64)
    cells = np.zeros(cells_per_dim ** 3, dtype=CELL_DTYPE)
    _check(_lib.sph_cells_build_grid(_ptr(x), C.c_uint64(x.shape[0]), C.c_uint32(cells_per_dim), C.c_double(box), _ptr(perm), _ptr(cells)))
    return perm, cells


def sph_cells_build_octree(x: np.ndarray, h: np.ndarray, max_per_leaf: int, box: float = 1.0):
    x = np.ascontiguousarray(x, dtype=np.float64)
    h = np.ascontiguousarray(h, dtype=np.float32)
    perm = np.empty(x.shape[0], dtype=np.uint64)
    p, n = C.c_void_p(), C.c_uint32(0)
    _check(_lib.sph_cells_build_octree(_ptr(x), _ptr(h), C.c_uint64(x.shape[0]), C.c_uint32(max_per_leaf), C.c_double(box),
                                       _ptr(perm), C.byref(p), C.byref(n)))
    cells = np.frombuffer(C.string_at(p.value, n.value * 48), dtype=CELL_DTYPE).copy() if n.value else np.zeros(0, CELL_DTYPE)
    _lib.sph_free(p)
    return perm, cells


def sph_tasks_build(cells: np.ndarray, hmax: np.ndarray, box: float = 1.0):
    """-> (tasks, n_self, n_pair)"""
    hmax = np.ascontiguousarray(hmax, dtype=np.float32)
    p, ns, npair = C.c_void_p(), C.c_uint64(0), C.c_uint64(0)
    _check(_lib.sph_tasks_build(_ptr(cells), _ptr(hmax), C.c_uint32(cells.shape[0]), C.c_double(box), C.byref(p), C.byref(ns), C.byref(npair)))
    nt = ns.value + npair.value
    tasks = np.frombuffer(C.string_at(p.value, nt * 56), dtype=TASK_DTYPE).copy()
    _lib.sph_free(p)
    return tasks, ns.value, npair.value


def sph_batch_create(store, tasks: np.ndarray, tasks_per_segment: int = 0):
    assert tasks.dtype.itemsize == 56 and tasks.flags.c_contiguous
    handle = C.c_void_p()
    _check(_lib.sph_batch_create(store, _ptr(tasks), C.c_uint64(tasks.shape[0]), C.c_uint32(tasks_per_segment), C.byref(handle)))
    return handle


def sph_batch_destroy(batch) -> None:
    _check(_lib.sph_batch_destroy(batch))


def sph_batch_get_info(batch) -> sph_batch_info:
    out = sph_batch_info()
    _check(_lib.sph_batch_get_info(batch, C.byref(out)))
    return out


def sph_batch_buffer_bytes(batch, aset: sph_attrset) -> int:
    out = C.c_uint64(0)
    _check(_lib.sph_batch_buffer_bytes(batch, _ref(aset), C.byref(out)))
    return out.value


def sph_batch_block_offsets(batch, aset: sph_attrset):
    """-> (off u64[2*n_tasks], seg_off u64[n_segments])"""
    info = sph_batch_get_info(batch)
    off = np.empty(2 * info.n_tasks, dtype=np.uint64)
    seg = np.empty(info.n_segments, dtype=np.uint64)
    _check(_lib.sph_batch_block_offsets(batch, _ref(aset), _ptr(off), _ptr(seg)))
    return off, seg


def sph_store_zero(store, aset: sph_attrset, stream=None) -> None:
    _check(_lib.sph_store_zero(store, _ref(aset), _stream(stream)))


def sph_pack(store, batch, aset: sph_attrset, d_buf, stream=None) -> None:
    _check(_lib.sph_pack(store, batch, _ref(aset), _ptr(d_buf), C.c_uint64(_nbytes(d_buf)), _stream(stream)))


SPH_PACK_STATIC_MAX_TASKS, SPH_PACK_STATIC_MAX_CHUNKS = 16384, 65536


def sph_pack_static(store, tasks: np.ndarray, aset: sph_attrset, d_buf=None, stream=None) -> int:
    """sph_pack for callers that must not allocate device memory (see include/sph_b200.h): takes the tasks instead of a
    batch and works out of a fixed scratch array inside the library.  Returns the buffer size the tasks need; with
    d_buf=None it only reports that size."""
    assert tasks.dtype.itemsize == 56 and tasks.flags.c_contiguous
    need = C.c_uint64(0)
    _check(_lib.sph_pack_static(store, _ptr(tasks), C.c_uint32(tasks.shape[0]), _ref(aset), _ptr(d_buf),
                                C.c_uint64(0 if d_buf is None else _nbytes(d_buf)), C.byref(need), _stream(stream)))
    return int(need.value)


def sph_pack_cells(store, batch, aset: sph_attrset, d_buf, cell_first: int, cell_count: int, stream=None) -> None:
    _check(_lib.sph_pack_cells(store, batch, _ref(aset), _ptr(d_buf), C.c_uint64(_nbytes(d_buf)), C.c_uint32(cell_first), C.c_uint32(cell_count),
                               _stream(stream)))


def sph_density(batch, d_in, d_out, stream=None) -> None:
    _check(_lib.sph_density(batch, _ptr(d_in), C.c_uint64(_nbytes(d_in)), _ptr(d_out), C.c_uint64(_nbytes(d_out)), _stream(stream)))


def sph_force(batch, d_in, d_out, params: sph_params, stream=None) -> None:
    _check(_lib.sph_force(batch, _ptr(d_in), C.c_uint64(_nbytes(d_in)), _ptr(d_out), C.c_uint64(_nbytes(d_out)),
                          C.byref(params), _stream(stream)))


SPLIT_BY_STRUCT, SPLIT_BY_ELEMENT, SPLIT_BY_TYPE, SPLIT_BY_STRUCT_AND_TYPE = 0, 1, 2, 3


def sph_pack_pass_masks(layout: sph_layout, aset: sph_attrset, split: int):
    """word masks of the passes of a split pack loop"""
    masks = (C.c_uint64 * 48)()
    n = C.c_uint32(0)
    _check(_lib.sph_pack_pass_masks(C.byref(layout), _ref(aset), C.c_int32(split), masks, C.byref(n)))
    return [int(masks[k]) for k in range(n.value)]


def sph_pack_pass(store, batch, aset: sph_attrset, word_mask: int, d_buf, stream=None) -> None:
    _check(_lib.sph_pack_pass(store, batch, _ref(aset), C.c_uint64(word_mask), _ptr(d_buf), C.c_uint64(_nbytes(d_buf)), _stream(stream)))


def sph_slot_attrset(loop: int) -> sph_attrset:
    out = sph_attrset()
    _check(_lib.sph_slot_attrset(C.c_int32(loop), C.byref(out)))
    return out


def sph_batch_slot_bytes(batch, loop: int) -> int:
    out = C.c_uint64(0)
    _check(_lib.sph_batch_slot_bytes(batch, C.c_int32(loop), C.byref(out)))
    return int(out.value)


def sph_pack_slots(store, batch, loop: int, d_slots, stream=None) -> None:
    _check(_lib.sph_pack_slots(store, batch, C.c_int32(loop), _ptr(d_slots), C.c_uint64(_nbytes(d_slots)), _stream(stream)))


def sph_density_slots(batch, d_slots, d_out, stream=None) -> None:
    _check(_lib.sph_density_slots(batch, _ptr(d_slots), C.c_uint64(_nbytes(d_slots)), _ptr(d_out), C.c_uint64(_nbytes(d_out)), _stream(stream)))


def sph_force_slots(batch, d_slots, d_out, params: sph_params, stream=None) -> None:
    _check(_lib.sph_force_slots(batch, _ptr(d_slots), C.c_uint64(_nbytes(d_slots)), _ptr(d_out), C.c_uint64(_nbytes(d_out)),
                                C.byref(params), _stream(stream)))


def sph_gradient(batch, d_in, d_out, stream=None) -> None:
    _check(_lib.sph_gradient(batch, _ptr(d_in), C.c_uint64(_nbytes(d_in)), _ptr(d_out), C.c_uint64(_nbytes(d_out)), _stream(stream)))


def sph_force3(batch, d_in, d_out, params: sph_params, stream=None) -> None:
    _check(_lib.sph_force3(batch, _ptr(d_in), C.c_uint64(_nbytes(d_in)), _ptr(d_out), C.c_uint64(_nbytes(d_out)),
                           C.byref(params), _stream(stream)))


def sph_unpack(store, batch, aset: sph_attrset, d_buf, mode: int = SPH_UNPACK_REDUCE, stream=None) -> None:
    _check(_lib.sph_unpack(store, batch, _ref(aset), _ptr(d_buf), C.c_uint64(_nbytes(d_buf)), C.c_int32(mode), _stream(stream)))


def sph_unpack_cells(store, batch, aset: sph_attrset, d_buf, cell_first: int, cell_count: int, mode: int = SPH_UNPACK_REDUCE, stream=None) -> None:
    _check(_lib.sph_unpack_cells(store, batch, _ref(aset), _ptr(d_buf), C.c_uint64(_nbytes(d_buf)), C.c_int32(mode), C.c_uint32(cell_first),
                                 C.c_uint32(cell_count), _stream(stream)))


def sph_ghost(store, params: sph_params, stream=None) -> None:
    _check(_lib.sph_ghost(store, C.byref(params), _stream(stream)))
