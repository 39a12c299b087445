"""ORACLE -- test infrastructure, not the product.

ctypes binding of oracle/sph_oracle.cpp (plain CPU C++ restatement of the hot
path of arxiv/paper_2606_23891, see that file's header for the citations).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference leg may import this package.  It imports nothing from
paper_2606_23891_b200 and shares no code with it.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sph_oracle.cpp")
_LIB = os.path.join(_HERE, "libsph_oracle.so")

# field ids (same order as sph_inputs.FIELDS; restated, not imported from the product)
X, V, A, MASS, H, U, DU_DT, RHO, RHO_DH, WCOUNT, WCOUNT_DH, DIV_V, ROT_V, P, CS, V_SIG, ID, TIME_BIN = range(18)
FLAG_X_REL_F32 = 1
MODE_REDUCE, MODE_ASSIGN = 0, 1

CELL_DTYPE = np.dtype({"names": ["first", "count", "pad", "origin", "width"],
                       "formats": ["<u8", "<u4", "<u4", ("<f8", (3,)), "<f8"],
                       "offsets": [0, 8, 12, 16, 40], "itemsize": 48})
TASK_DTYPE = np.dtype({"names": ["ci", "cj", "frame_i", "frame_j"],
                       "formats": ["<i4", "<i4", ("<f8", (3,)), ("<f8", (3,))],
                       "offsets": [0, 4, 8, 32], "itemsize": 56})
ATTR_DTYPE = np.dtype([("field", "<i4"), ("comp0", "<i4"), ("ncomp", "<i4")])

# the four canonical attribute sets: (entries, flags)
DENSITY_IN = ([(X, 0, 3), (H, 0, 1), (MASS, 0, 1)], FLAG_X_REL_F32)
DENSITY_OUT = ([(RHO, 0, 1), (RHO_DH, 0, 1), (WCOUNT, 0, 1), (WCOUNT_DH, 0, 1)], 0)
FORCE_IN = ([(X, 0, 3), (H, 0, 1), (MASS, 0, 1), (RHO, 0, 1), (RHO_DH, 0, 1), (V, 0, 3), (U, 0, 1), (P, 0, 1), (CS, 0, 1)],
            FLAG_X_REL_F32)
FORCE_OUT = ([(A, 0, 3), (DU_DT, 0, 1), (V_SIG, 0, 1)], 0)
# the three-loop cycle (reading C34): Table 1's p-g column; div_v, rot_v out; the force inputs plus div_v, rot_v, time_bin
GRADIENT_IN = ([(X, 0, 3), (V, 0, 3), (MASS, 0, 1), (H, 0, 1), (U, 0, 1), (RHO, 0, 1)], FLAG_X_REL_F32)
GRADIENT_OUT = ([(DIV_V, 0, 1), (ROT_V, 0, 3)], 0)
FORCE3_IN = (FORCE_IN[0] + [(DIV_V, 0, 1), (ROT_V, 0, 3), (TIME_BIN, 0, 1)], FLAG_X_REL_F32)


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no CUDA).  -ffp-contract=off: no fused multiply-adds."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c++17",
                               _SRC, "-o", _LIB])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        for name in ("orc_w", "orc_dw"):
            getattr(_lib, name).restype = C.c_double
            getattr(_lib, name).argtypes = [C.c_double]
        for name in ("orc_W", "orc_dW_dh", "orc_dW_dr"):
            getattr(_lib, name).restype = C.c_double
            getattr(_lib, name).argtypes = [C.c_double, C.c_double]
        _lib.orc_block_offsets.restype = C.c_uint64
        _lib.orc_cells_build_octree.restype = C.c_int64
        _lib.orc_tasks_build.restype = C.c_int64
        _lib.orc_iterate_h.restype = C.c_int64
        _lib.orc_compare_blocks.restype = C.c_int64
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _attrs(attrset):
    entries, flags = attrset
    arr = np.array([tuple(e) for e in entries], dtype=ATTR_DTYPE)
    return arr, len(entries), int(flags)


def set_threads(n: int) -> int:
    return lib().orc_set_threads(C.c_int(n))


def w(q): return lib().orc_w(q)
def dw(q): return lib().orc_dw(q)
def W(r, h): return lib().orc_W(r, h)
def dW_dh(r, h): return lib().orc_dW_dh(r, h)
def dW_dr(r, h): return lib().orc_dW_dr(r, h)


def record_bytes(attrset) -> int:
    arr, n, flags = _attrs(attrset)
    return lib().orc_record_bytes(_p(arr), C.c_int(n), C.c_uint32(flags))


def cells_build_grid(x: np.ndarray, cpd: int, box: float = 1.0):
    """-> (perm u64[n], cells[cpd^3])"""
    x = np.ascontiguousarray(x, dtype=np.float64)
    n = x.shape[0]
    perm = np.empty(n, dtype=np.uint64)
    cells = np.zeros(cpd ** 3, dtype=CELL_DTYPE)
    rc = lib().orc_cells_build_grid(_p(x), C.c_uint64(n), C.c_uint32(cpd), C.c_double(box), _p(perm), _p(cells))
    if rc != 0:
        raise ValueError(f"orc_cells_build_grid: {rc}")
    return perm, cells


def cells_build_octree(x: np.ndarray, h: np.ndarray, max_per_leaf: int, box: float = 1.0):
    x = np.ascontiguousarray(x, dtype=np.float64)
    h = np.ascontiguousarray(h, dtype=np.float32)
    n = x.shape[0]
    perm = np.empty(n, dtype=np.uint64)
    nl = lib().orc_cells_build_octree(_p(x), _p(h), C.c_uint64(n), C.c_uint32(max_per_leaf), C.c_double(box), _p(perm), None,
                                      C.c_uint64(0))
    if nl < 0:
        raise ValueError(f"orc_cells_build_octree: {nl}")
    cells = np.zeros(nl, dtype=CELL_DTYPE)
    nl2 = lib().orc_cells_build_octree(_p(x), _p(h), C.c_uint64(n), C.c_uint32(max_per_leaf), C.c_double(box), _p(perm),
                                       _p(cells), C.c_uint64(nl))
    assert nl2 == nl
    return perm, cells


def cell_hmax(parts_sorted: np.ndarray, cells: np.ndarray) -> np.ndarray:
    """max h of each cell's particles (input to the task rule)."""
    h = parts_sorted["h"]
    out = np.zeros(cells.shape[0], dtype=np.float32)
    for c in range(cells.shape[0]):
        f, k = int(cells["first"][c]), int(cells["count"][c])
        if k:
            out[c] = h[f:f + k].max()
    return out


def tasks_build(cells: np.ndarray, hmax: np.ndarray, box: float = 1.0):
    """-> (tasks, n_self, n_pair)"""
    hmax = np.ascontiguousarray(hmax, dtype=np.float32)
    ns, npair = C.c_uint64(0), C.c_uint64(0)
    nt = lib().orc_tasks_build(_p(cells), _p(hmax), C.c_uint32(cells.shape[0]), C.c_double(box), None, C.c_uint64(0),
                               C.byref(ns), C.byref(npair))
    if nt < 0:
        raise ValueError(f"orc_tasks_build: {nt}")
    tasks = np.zeros(nt, dtype=TASK_DTYPE)
    nt2 = lib().orc_tasks_build(_p(cells), _p(hmax), C.c_uint32(cells.shape[0]), C.c_double(box), _p(tasks), C.c_uint64(nt),
                                C.byref(ns), C.byref(npair))
    assert nt2 == nt
    return tasks, ns.value, npair.value


def block_offsets(cells, tasks, rec_bytes: int):
    """-> (off u64[2*n_tasks], total_bytes)"""
    off = np.empty(2 * tasks.shape[0], dtype=np.uint64)
    total = lib().orc_block_offsets(_p(cells), _p(tasks), C.c_int64(tasks.shape[0]), C.c_int(rec_bytes), _p(off))
    return off, int(total)


def pack(parts, cells, tasks, attrset, fill: int = 0xCD) -> np.ndarray:
    """Pack tasks into a fresh buffer (pad bytes = fill)."""
    arr, n, flags = _attrs(attrset)
    _, total = block_offsets(cells, tasks, record_bytes(attrset))
    buf = np.full(total, fill, dtype=np.uint8)
    rc = lib().orc_pack(_p(parts), _p(cells), _p(tasks), C.c_int64(tasks.shape[0]), _p(arr), C.c_int(n), C.c_uint32(flags),
                        _p(buf), C.c_uint64(total))
    if rc != 0:
        raise ValueError(f"orc_pack: {rc}")
    return buf


def unpack(parts, cells, tasks, attrset, buf, mode=MODE_REDUCE) -> None:
    arr, n, flags = _attrs(attrset)
    buf = np.ascontiguousarray(buf, dtype=np.uint8)
    rc = lib().orc_unpack(_p(parts), _p(cells), _p(tasks), C.c_int64(tasks.shape[0]), _p(arr), C.c_int(n), C.c_uint32(flags),
                          _p(buf), C.c_uint64(buf.shape[0]), C.c_int(mode))
    if rc != 0:
        raise ValueError(f"orc_unpack: {rc}")


def zero(parts, attrset) -> None:
    arr, n, _ = _attrs(attrset)
    rc = lib().orc_zero(_p(parts), C.c_uint64(parts.shape[0]), _p(arr), C.c_int(n))
    if rc != 0:
        raise ValueError(f"orc_zero: {rc}")


def density(cells, tasks, buf_in, fill: int = 0xCD) -> np.ndarray:
    _, total = block_offsets(cells, tasks, 16)
    out = np.full(total, fill, dtype=np.uint8)
    lib().orc_density(_p(cells), _p(tasks), C.c_int64(tasks.shape[0]), _p(buf_in), _p(out))
    return out


def force(cells, tasks, buf_in, alpha: float = 0.8, beta: float = 3.0, fill: int = 0xCD) -> np.ndarray:
    _, total = block_offsets(cells, tasks, 20)
    out = np.full(total, fill, dtype=np.uint8)
    lib().orc_force(_p(cells), _p(tasks), C.c_int64(tasks.shape[0]), _p(buf_in), _p(out), C.c_double(alpha), C.c_double(beta))
    return out


def compare_blocks(cells, tasks, rec_bytes: int, buf_a, buf_b) -> int:
    """test support: -1 if the two buffers agree on every record byte (pad bytes skipped), else the first differing offset"""
    assert buf_a.dtype == np.uint8 and buf_b.dtype == np.uint8 and buf_a.flags.c_contiguous and buf_b.flags.c_contiguous
    return int(lib().orc_compare_blocks(_p(cells), _p(tasks), C.c_int64(tasks.shape[0]), C.c_int(rec_bytes), _p(buf_a), _p(buf_b)))


def flag_cutoff_pairs(cells, tasks, buf_in, rel: float = 1e-5) -> np.ndarray:
    """reading C31: bool[n], True where a particle has a partner within rel of the cut-off in some task (buf_in: FORCE_IN)."""
    n = int((cells["first"].astype(np.int64) + cells["count"]).max())
    flags = np.zeros(n, dtype=np.uint8)
    lib().orc_flag_cutoff_pairs(_p(cells), _p(tasks), C.c_int64(tasks.shape[0]), _p(buf_in), C.c_double(rel), _p(flags))
    return flags.astype(bool)


def gradient(cells, tasks, buf_in, fill: int = 0xCD) -> np.ndarray:
    _, total = block_offsets(cells, tasks, 16)
    out = np.full(total, fill, dtype=np.uint8)
    lib().orc_gradient(_p(cells), _p(tasks), C.c_int64(tasks.shape[0]), _p(buf_in), _p(out))
    return out


def force3(cells, tasks, buf_in, alpha: float = 0.8, beta: float = 3.0, fill: int = 0xCD) -> np.ndarray:
    _, total = block_offsets(cells, tasks, 20)
    out = np.full(total, fill, dtype=np.uint8)
    lib().orc_force3(_p(cells), _p(tasks), C.c_int64(tasks.shape[0]), _p(buf_in), _p(out), C.c_double(alpha), C.c_double(beta))
    return out


def brute_gradient(parts, box: float = 1.0) -> np.ndarray:
    out = np.empty((parts.shape[0], 4), dtype=np.float64)
    lib().orc_brute_gradient(_p(parts), C.c_uint64(parts.shape[0]), C.c_double(box), _p(out))
    return out


def ghost(parts, gamma: float = 5.0 / 3.0) -> None:
    lib().orc_ghost(_p(parts), C.c_uint64(parts.shape[0]), C.c_double(gamma))


def brute_density(parts, box: float = 1.0) -> np.ndarray:
    out = np.empty((parts.shape[0], 4), dtype=np.float64)
    lib().orc_brute_density(_p(parts), C.c_uint64(parts.shape[0]), C.c_double(box), _p(out))
    return out


def brute_force(parts, box: float = 1.0, alpha: float = 0.8, beta: float = 3.0) -> np.ndarray:
    out = np.empty((parts.shape[0], 5), dtype=np.float64)
    lib().orc_brute_force(_p(parts), C.c_uint64(parts.shape[0]), C.c_double(box), C.c_double(alpha), C.c_double(beta), _p(out))
    return out


def iterate_h(x, h0, h_cap: float, n_target: float = 48.0, tol: float = 0.01, max_iter: int = 30, box: float = 1.0):
    """-> (h f32[n], number of particles not converged)"""
    x = np.ascontiguousarray(x, dtype=np.float64)
    h0 = np.ascontiguousarray(h0, dtype=np.float32)
    out = np.empty_like(h0)
    bad = lib().orc_iterate_h(_p(x), C.c_uint64(x.shape[0]), C.c_double(box), _p(h0), C.c_double(h_cap), C.c_double(n_target),
                              C.c_double(tol), C.c_int(max_iter), _p(out))
    if bad < 0:
        raise ValueError(f"orc_iterate_h: {bad}")
    return out, int(bad)


# ---- whole-loop drivers used by tests and the CPU baseline (plain sequencing of the steps) ----

def density_cycle(parts, cells, tasks, batch: int = 0):
    """zero -> for each batch: pack, density, unpack.  parts must already be in cell order."""
    zero(parts, DENSITY_OUT)
    nb = tasks.shape[0] if batch <= 0 else batch
    for s in range(0, tasks.shape[0], nb):
        t = tasks[s:s + nb]
        unpack(parts, cells, t, DENSITY_OUT, density(cells, t, pack(parts, cells, t, DENSITY_IN)))


def force_cycle(parts, cells, tasks, batch: int = 0, alpha: float = 0.8, beta: float = 3.0):
    zero(parts, FORCE_OUT)
    nb = tasks.shape[0] if batch <= 0 else batch
    for s in range(0, tasks.shape[0], nb):
        t = tasks[s:s + nb]
        unpack(parts, cells, t, FORCE_OUT, force(cells, t, pack(parts, cells, t, FORCE_IN), alpha, beta))


def gradient_cycle(parts, cells, tasks, batch: int = 0):
    zero(parts, GRADIENT_OUT)
    nb = tasks.shape[0] if batch <= 0 else batch
    for s in range(0, tasks.shape[0], nb):
        t = tasks[s:s + nb]
        unpack(parts, cells, t, GRADIENT_OUT, gradient(cells, t, pack(parts, cells, t, GRADIENT_IN)))


def force3_cycle(parts, cells, tasks, batch: int = 0, alpha: float = 0.8, beta: float = 3.0):
    zero(parts, FORCE_OUT)
    nb = tasks.shape[0] if batch <= 0 else batch
    for s in range(0, tasks.shape[0], nb):
        t = tasks[s:s + nb]
        unpack(parts, cells, t, FORCE_OUT, force3(cells, t, pack(parts, cells, t, FORCE3_IN), alpha, beta))
