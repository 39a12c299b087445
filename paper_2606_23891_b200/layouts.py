"""The paper's particle memory layouts (section 3.1) as field groupings for `sph_layout_from_groups`.

Data only: which member lives in which substruct.  The paper's sAoS variants are defined for three interaction loops
(density, gradient, force); this build has two (density, force), and the density inputs {x, h, mass} are a subset of the
force inputs {x, h, mass, rho, rho_dh, v, u, P, c_s}, so:
  pack-density  every variable the DENSITY pack needs in one struct, the rest of the force inputs in another (the paper's
                pack-gradient idea: the first loop's pack has priority); with two nested input sets this is also
                pack-shared (the shared variables {x, h, mass} in a struct of their own)
  pack-force    every variable the FORCE pack needs in one struct (64 bytes): the density pack has to gather its three
                members out of it
  *-type        the same, every substruct further split by data type (f64 | f32 | i64 | i8)
  random-order  the 128-byte AoS record with its members shuffled (seeded)
`split` (sph_layout_split, BASELINE.json:configs[1]) groups by kernel read / write pattern instead.
"""
import numpy as np

AOS_ORDER = ["x", "v", "a", "mass", "h", "u", "du_dt", "rho", "rho_dh", "wcount", "wcount_dh", "div_v", "rot_v", "P", "c_s", "v_sig",
             "id", "time_bin"]
_REST = [["wcount", "wcount_dh"], ["a", "du_dt", "v_sig"], ["div_v", "rot_v"]]

GROUPS = {
    "pack-density": [["x", "h", "mass"], ["rho", "rho_dh", "v", "u", "P", "c_s"]] + _REST + [["id", "time_bin"]],
    "pack-force": [["x", "h", "mass", "rho", "rho_dh", "v", "u", "P", "c_s"]] + _REST + [["id", "time_bin"]],
    "pack-density-type": [["x"], ["h", "mass"], ["rho", "rho_dh", "v", "u", "P", "c_s"]] + _REST + [["id"], ["time_bin"]],
    "pack-force-type": [["x"], ["h", "mass", "rho", "rho_dh", "v", "u", "P", "c_s"]] + _REST + [["id"], ["time_bin"]],
}
NAMES = ["aos", "random-order", "split"] + list(GROUPS)

# The three-loop cycle (density, gradient, force; reading C34) -- the paper's own three sAoS subflavours:
#   GRADIENT_IN = {x, v, mass, h, u, rho} is a subset of FORCE3_IN = GRADIENT_IN + {rho_dh, P, c_s, div_v, rot_v, time_bin};
#   DENSITY_IN = {x, h, mass} is a subset of both.
#   pack-gradient  "all variables required for [the gradient pack] are placed into its associated struct, disadvantaging the
#                  force packing loop's access thereof": the force pack gathers from two structs
#   pack-force     every variable the force pack needs in one struct (92 bytes): the gradient and density packs gather out of it
#   pack-shared    "all variables shared between those two operations in a separate 'shared' struct", applied to all three
#                  packs: {x, h, mass} (all three), {v, u, rho} (gradient and force), the force-only rest
#   *-type         every substruct further split by data type
_REST3 = [["wcount", "wcount_dh"], ["a", "du_dt", "v_sig"]]
_F_ONLY = ["rho_dh", "P", "c_s", "div_v", "rot_v"]
GROUPS3 = {
    "pack-gradient": [["x", "v", "mass", "h", "u", "rho"], _F_ONLY + ["time_bin"]] + _REST3 + [["id"]],
    "pack-force": [["x", "h", "mass", "rho", "rho_dh", "v", "u", "P", "c_s", "div_v", "rot_v", "time_bin"]] + _REST3 + [["id"]],
    "pack-shared": [["x", "h", "mass"], ["v", "u", "rho"], _F_ONLY + ["time_bin"]] + _REST3 + [["id"]],
    "pack-gradient-type": [["x"], ["v", "mass", "h", "u", "rho"], _F_ONLY, ["time_bin"]] + _REST3 + [["id"]],
    "pack-force-type": [["x"], ["h", "mass", "rho", "rho_dh", "v", "u", "P", "c_s", "div_v", "rot_v"], ["time_bin"]] + _REST3 + [["id"]],
    "pack-shared-type": [["x"], ["h", "mass"], ["v", "u", "rho"], _F_ONLY, ["time_bin"]] + _REST3 + [["id"]],
}
NAMES3 = ["aos", "random-order", "split"] + list(GROUPS3)


def layout(sph, name: str, seed: int = 1, loops: int = 2):
    """the named layout as an sph_layout (sph = the binding module); loops = 3 selects the three-loop groupings"""
    if name == "aos":
        return sph.sph_layout_aos()
    if name == "split":
        return sph.sph_layout_split()
    if name == "random-order":
        order = [AOS_ORDER[i] for i in np.random.default_rng(seed).permutation(len(AOS_ORDER))]
        return sph.sph_layout_from_groups([order], min_stride=[128])
    return sph.sph_layout_from_groups((GROUPS3 if loops == 3 else GROUPS)[name])
