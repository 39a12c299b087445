"""The canonical particle record: a 128-byte AoS struct.

Member list, order and "128-byte" are fixed by BASELINE.json:configs[0]
(x[3] f64, v[3], a[3], mass, h, u, du_dt, rho, rho_dh, wcount, wcount_dh,
div_v, rot_v[3], P, c_s, v_sig f32, id i64, time_bin i8, padding); the types
are the paper's Table 1 (x double, everything else float,
time_bin int8_t).  Offsets are natural C alignment (reading C16).
"""
import numpy as np

# name, numpy format, byte offset, number of scalar components
_MEMBERS = [
    ("x", "<f8", 0, 3),
    ("v", "<f4", 24, 3),
    ("a", "<f4", 36, 3),
    ("mass", "<f4", 48, 1),
    ("h", "<f4", 52, 1),
    ("u", "<f4", 56, 1),
    ("du_dt", "<f4", 60, 1),
    ("rho", "<f4", 64, 1),
    ("rho_dh", "<f4", 68, 1),
    ("wcount", "<f4", 72, 1),
    ("wcount_dh", "<f4", 76, 1),
    ("div_v", "<f4", 80, 1),
    ("rot_v", "<f4", 84, 3),
    ("P", "<f4", 96, 1),
    ("c_s", "<f4", 100, 1),
    ("v_sig", "<f4", 104, 1),
    ("id", "<i8", 112, 1),
    ("time_bin", "i1", 120, 1),
]

PART_DTYPE = np.dtype({
    "names": [m[0] for m in _MEMBERS],
    "formats": [(m[1], (3,)) if m[3] == 3 else m[1] for m in _MEMBERS],
    "offsets": [m[2] for m in _MEMBERS],
    "itemsize": 128,
})

#: field ids, in the order both C interfaces use
FIELDS = [m[0] for m in _MEMBERS]
FIELD_NCOMP = [m[3] for m in _MEMBERS]


def field_id(name: str) -> int:
    return FIELDS.index(name)


def empty_parts(n: int) -> np.ndarray:
    """n zero-filled canonical records (pad bytes zero as well)."""
    return np.zeros(n, dtype=PART_DTYPE)
