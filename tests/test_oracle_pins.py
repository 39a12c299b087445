"""Pins of the oracle against what the mathematics fixes (no GPU, no product code).

The paper prints no formula, constant or worked example (PAPER.md:39-41 cite
Price 2012), so the pins are closed forms, invariants, brute force on tiny
inputs and the independent lattice sums recorded in tests/golden/ (SURVEY.md
section 8(c)).  Each test names the plausible mistake it would catch.
"""
import math
import os

import numpy as np
import pytest

import oracle as orc
import sph_inputs as si
from orc_setup import lattice, raw_copy, scaled_err, sort_grid, sort_octree

GOLD = os.path.join(os.path.dirname(__file__), "golden", "lattice_sums.txt")
GAMMA = 5.0 / 3.0


def _gold_rows():
    rows = []
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            rows.append([float(t) for t in line.split()])
    return rows


# ------------------------------------------------------------------ kernel function (C2)

def test_kernel_point_values():
    # w(0.5) = 1 - 1.5/4 + 0.75/8, w'(0.5) = -1.5 + 2.25/4: wrong coefficient or branch
    assert orc.w(0.5) == pytest.approx(0.71875, abs=1e-15)
    assert orc.dw(0.5) == pytest.approx(-0.9375, abs=1e-15)
    assert orc.w(0.0) == 1.0 and orc.w(2.0) == 0.0 and orc.w(2.5) == 0.0
    # continuity of both branches at q = 1 (w = 0.25, w' = -0.75)
    assert orc.w(1.0) == pytest.approx(0.25, abs=1e-15) and orc.w(1.0 - 1e-12) == pytest.approx(0.25, abs=1e-11)
    assert orc.dw(1.0) == pytest.approx(-0.75, abs=1e-15) and orc.dw(1.0 - 1e-12) == pytest.approx(-0.75, abs=1e-11)
    h = 0.37
    assert orc.W(0.0, h) * h ** 3 == pytest.approx(1.0 / math.pi, rel=1e-15)


def test_kernel_normalisation_and_dh_integral():
    # 4 pi int_0^2h W r^2 dr = 1 and 4 pi int dW/dh r^2 dr = 0 (d/dh of the normalisation): wrong sigma,
    # wrong power of h, dropped 3w term
    h = 0.13
    m = 200001
    r = np.linspace(0.0, 2.0 * h, m)
    simpson = np.ones(m)
    simpson[1:-1:2], simpson[2:-1:2] = 4.0, 2.0
    simpson *= (r[1] - r[0]) / 3.0
    Wv = np.array([orc.W(x, h) for x in r])
    dv = np.array([orc.dW_dh(x, h) for x in r])
    assert 4 * math.pi * np.sum(simpson * Wv * r * r) == pytest.approx(1.0, abs=1e-10)
    assert 4 * math.pi * np.sum(simpson * dv * r * r) * h == pytest.approx(0.0, abs=1e-10)


def test_kernel_derivatives_by_finite_differences():
    # dW/dr and dW/dh against central differences of W itself: sign or chain-rule mistakes
    for r, h in [(0.03, 0.1), (0.12, 0.1), (0.17, 0.09), (0.001, 0.2)]:
        e = 1e-6
        assert orc.dW_dr(r, h) == pytest.approx((orc.W(r + e, h) - orc.W(r - e, h)) / (2 * e), rel=1e-6)
        assert orc.dW_dh(r, h) == pytest.approx((orc.W(r, h + e) - orc.W(r, h - e)) / (2 * e), rel=1e-6)


# ------------------------------------------------------------------ density

@pytest.mark.parametrize("row", _gold_rows())
def test_lattice_density_closed_form(row):
    # whole pipeline (cells, tasks, frames, pack, density, unpack) on a 12^3 lattice in 3^3 cells
    h_dx, npts, rho_ref, rho_dh_ref = row
    n_side = 12
    parts = lattice(n_side, h_dx)
    ps, cells, tasks, ns, npair = sort_grid(parts, 3)
    assert (ns, npair) == (27, 27 * 13)
    orc.density_cycle(ps, cells, tasks)
    dx, m = 1.0 / n_side, 1.0 / n_side ** 3
    # f32 store: ~27 f32 additions per particle -> a few 1e-7
    assert np.max(np.abs(ps["rho"] / (m / dx ** 3) - rho_ref)) < 2e-6
    assert np.max(np.abs(ps["wcount"] * dx ** 3 - rho_ref)) < 2e-6
    assert np.max(np.abs(ps["rho_dh"] * dx ** 4 / m - rho_dh_ref)) < 2e-6
    assert np.max(np.abs(ps["wcount_dh"] * dx ** 4 - rho_dh_ref)) < 2e-6
    # number of lattice points inside the support = hits per particle, counted by brute force
    d = ps["x"][0] - ps["x"]
    d -= np.round(d)
    # (points exactly on the cut-off, h = 1.0 dx, carry zero weight and are not counted)
    assert np.sum(np.einsum("ij,ij->i", d, d) < (2 * h_dx * dx) ** 2 * (1 - 1e-9)) == npts


def test_two_particles_closed_form():
    # rho_1 h^3 / m = (w(0) + w(0.5)) / pi = (1 + 0.71875) / pi: self term dropped, wrong q
    parts = np.zeros(2, dtype=si.PART_DTYPE)
    parts["x"] = [[0.40, 0.5, 0.5], [0.45, 0.5, 0.5]]
    parts["h"], parts["mass"] = 0.1, 2.0
    ps, cells, tasks, ns, npair = sort_grid(parts, 3)
    orc.density_cycle(ps, cells, tasks)
    assert ps["rho"][0] * 0.1 ** 3 / 2.0 == pytest.approx(0.5470951168783903, rel=3e-7)
    assert ps["rho"][1] == ps["rho"][0]
    assert ps["wcount"][0] * 2.0 == pytest.approx(ps["rho"][0], rel=3e-7)


def test_two_particles_across_periodic_boundary():
    # same pair, one particle wrapped around x = 0: the frame shift of side j must be right
    parts = np.zeros(2, dtype=si.PART_DTYPE)
    parts["x"] = [[0.98, 0.5, 0.01], [0.03, 0.5, 0.99]]
    parts["h"], parts["mass"] = 0.1, 1.0
    r = math.sqrt(0.05 ** 2 + 0.02 ** 2)
    ps, cells, tasks, _, _ = sort_grid(parts, 4)
    orc.density_cycle(ps, cells, tasks)
    expect = (1.0 + orc.w(r / 0.1)) / (math.pi * 1e-3)
    assert ps["rho"][0] == pytest.approx(expect, rel=3e-7) and ps["rho"][1] == pytest.approx(expect, rel=3e-7)


def test_config0_equal_mass_invariant_and_brute_force():
    parts = si.config0(seed=1)
    ps, cells, tasks, ns, npair = sort_grid(parts, 4)
    assert (ns, npair) == (64, 832) and np.all(cells["count"] == 64)
    orc.density_cycle(ps, cells, tasks)
    m = np.float32(1.0 / 4096)
    # equal masses: rho = m wcount, rho_dh = m wcount_dh to rounding
    assert np.max(np.abs(ps["rho"] - m * ps["wcount"]) / ps["rho"]) < 1e-6
    assert np.max(scaled_err(ps["rho_dh"], m * ps["wcount_dh"], ps["rho"] / ps["h"])) < 1e-6
    # O(N^2) minimum-image sums on the original f64 positions: every neighbour reached exactly once
    ref = orc.brute_density(ps)
    assert np.max(np.abs(ps["rho"] - ref[:, 0]) / ref[:, 0]) < 5e-6
    assert np.max(np.abs(ps["wcount"] - ref[:, 2]) / ref[:, 2]) < 5e-6
    assert np.max(scaled_err(ps["rho_dh"], ref[:, 1], ref[:, 0] / ps["h"])) < 5e-6
    assert np.max(scaled_err(ps["wcount_dh"], ref[:, 3], ref[:, 2] / ps["h"])) < 5e-6


def _variable_case(seed, n_side=10, cpd=3):
    parts = si.jittered_lattice(n_side, seed, jitter=0.6, eta=1.2348, sigma_v=0.3, h_spread=0.25, mass_spread=0.5, u_spread=0.4)
    return sort_grid(parts, cpd)


@pytest.mark.parametrize("seed,batch", [(2, 0), (3, 7)])
def test_variable_h_mass_pipeline_vs_brute_force(seed, batch):
    ps, cells, tasks, ns, npair = _variable_case(seed)
    assert 2.0 * ps["h"].max() <= cells["width"][0]
    orc.density_cycle(ps, cells, tasks, batch=batch)
    ref = orc.brute_density(ps)
    assert np.max(np.abs(ps["rho"] - ref[:, 0]) / ref[:, 0]) < 5e-6
    assert np.max(scaled_err(ps["rho_dh"], ref[:, 1], ref[:, 0] / ps["h"])) < 5e-6
    orc.ghost(ps, GAMMA)
    orc.force_cycle(ps, cells, tasks, batch=batch)
    ref5 = orc.brute_force(ps)
    amax = np.abs(ref5[:, :3]).max()
    assert np.max(np.abs(ps["a"] - ref5[:, :3])) < 5e-6 * amax
    assert np.max(np.abs(ps["du_dt"] - ref5[:, 3])) < 5e-6 * np.abs(ref5[:, 3]).max()
    assert np.max(np.abs(ps["v_sig"] - ref5[:, 4]) / ref5[:, 4]) < 1e-6


# ------------------------------------------------------------------ ghost

def test_ghost_closed_form():
    parts = np.zeros(3, dtype=si.PART_DTYPE)
    parts["rho"], parts["u"] = [1.0, 2.0, 0.5], [1.0, 3.0, 0.25]
    orc.ghost(parts, GAMMA)
    assert np.allclose(parts["P"], [2 / 3, 4.0, 1 / 12], rtol=1e-7)
    assert np.allclose(parts["c_s"], [math.sqrt(10 / 9), math.sqrt(10 / 3), math.sqrt(10 / 36)], rtol=1e-7)


# ------------------------------------------------------------------ force

def test_static_lattice_zero_force():
    ps, cells, tasks, _, _ = sort_grid(lattice(12, 1.2348), 3)
    orc.density_cycle(ps, cells, tasks)
    orc.ghost(ps, GAMMA)
    orc.force_cycle(ps, cells, tasks)
    # symmetric neighbours cancel; the per-term size is ~ m A |G| ~ 1e1, f32 partial sums leave ~1e-6 of that
    assert np.abs(ps["a"]).max() < 2e-5
    assert np.all(ps["du_dt"] == 0.0)
    assert np.allclose(ps["v_sig"], 2.1081851067789197, rtol=2e-7)     # 2 c_s, c_s = sqrt(10/9)


def test_force_two_particles_hand_worked():
    # FORCE_IN records written by hand; every factor of the formula is a number chosen here.
    # i at origin, j at (0.05, 0, 0); h_i = h_j = 0.1 -> q = 0.5, w' = -0.9375, G = w'/(pi h^4)
    # rho_dh = 0 -> Omega = 1;  A_i = P_i/rho_i^2 = 2/4, A_j = 3/9;  v_ij.r_hat = (v_i - v_j).(-1,0,0)
    rec = np.zeros((2, 13), dtype=np.float32)
    #          xr0   xr1 xr2  h    m    rho  rho_dh v0   v1 v2  u    P    cs
    rec[0] = [0.00, 0.0, 0.0, 0.1, 1.5, 2.0, 0.0, 0.3, 0.0, 0.0, 1.0, 2.0, 1.0]
    rec[1] = [0.05, 0.0, 0.0, 0.1, 2.5, 3.0, 0.0, -0.1, 0.0, 0.0, 1.0, 3.0, 1.25]
    cells = np.zeros(1, dtype=orc.CELL_DTYPE)
    cells["count"], cells["width"] = 2, 1.0
    tasks = np.zeros(1, dtype=orc.TASK_DTYPE)
    tasks["cj"] = -1
    buf = np.zeros(128, dtype=np.uint8)
    buf[:104] = rec.view(np.uint8).ravel()
    out = orc.force(cells, tasks, buf, alpha=0.8, beta=3.0)[:40].view(np.float32).reshape(2, 5)
    G = -0.9375 / (math.pi * 1e-4)
    vr = (0.3 - (-0.1)) * (-1.0)                 # approaching: -0.4
    mu = vr
    vs = 1.0 + 1.25 - 3.0 * mu                   # 3.45
    visc = -0.5 * 0.8 * vs * mu / 2.5            # > 0
    F = 0.5 * G + (1.0 / 3.0) * G + visc * G
    assert out[0, 0] == pytest.approx(-2.5 * F * (-1.0), rel=1e-6)     # i is pushed towards -x (G < 0)
    assert out[0, 0] < 0 < out[1, 0]
    assert out[1, 0] == pytest.approx(-1.5 * F * (+1.0), rel=1e-6)
    assert out[0, 3] == pytest.approx(2.5 * (0.5 * G + 0.5 * visc * G) * vr, rel=1e-6)
    assert out[1, 3] == pytest.approx(1.5 * ((1.0 / 3.0) * G + 0.5 * visc * G) * vr, rel=1e-6)
    assert out[0, 4] == pytest.approx(vs, rel=1e-6) and out[1, 4] == pytest.approx(vs, rel=1e-6)
    # receding pair: no viscosity (mu = 0), v_sig = c_i + c_j
    rec[0, 7], rec[1, 7] = -0.1, 0.3
    buf[:104] = rec.view(np.uint8).ravel()
    out2 = orc.force(cells, tasks, buf)[:40].view(np.float32).reshape(2, 5)
    assert out2[0, 0] == pytest.approx(2.5 * (0.5 + 1.0 / 3.0) * G, rel=1e-6)
    assert out2[0, 4] == pytest.approx(2.25, rel=1e-6)
    # classic Monaghan form with beta' = 3 alpha / 2: Pi = (-alpha cbar mu + beta' mu^2) / rhobar  (C1)
    cbar, rhobar = 0.5 * (1.0 + 1.25), 2.5
    assert visc == pytest.approx((-0.8 * cbar * mu + 1.2 * mu * mu) / rhobar, rel=1e-12)


def test_force_grad_h_factor():
    # rho_dh != 0 must enter as Omega = 1 + h rho_dh / (3 rho) in the denominator of A
    rec = np.zeros((2, 13), dtype=np.float32)
    rec[0] = [0.00, 0.0, 0.0, 0.1, 1.0, 2.0, 12.0, 0, 0, 0, 1.0, 2.0, 1.0]
    rec[1] = [0.05, 0.0, 0.0, 0.1, 1.0, 2.0, -6.0, 0, 0, 0, 1.0, 2.0, 1.0]
    cells = np.zeros(1, dtype=orc.CELL_DTYPE)
    cells["count"], cells["width"] = 2, 1.0
    tasks = np.zeros(1, dtype=orc.TASK_DTYPE)
    tasks["cj"] = -1
    buf = np.zeros(128, dtype=np.uint8)
    buf[:104] = rec.view(np.uint8).ravel()
    out = orc.force(cells, tasks, buf)[:40].view(np.float32).reshape(2, 5)
    G = -0.9375 / (math.pi * 1e-4)
    om_i, om_j = 1 + 0.1 * 12.0 / 6.0, 1 - 0.1 * 6.0 / 6.0           # 1.2, 0.9
    F = (2.0 / (om_i * 4.0) + 2.0 / (om_j * 4.0)) * G
    assert out[0, 0] == pytest.approx(F, rel=1e-6) and out[1, 0] == pytest.approx(-F, rel=1e-6)


@pytest.mark.parametrize("seed", [4, 5])
def test_force_momentum_and_energy_invariants(seed):
    # sum m a = 0 (pairwise antisymmetry) and sum m (v.a + du/dt) = 0 (C13): a wrong sign, a swapped i/j
    # or a missing factor 1/2 in the viscous heating breaks one of them
    ps, cells, tasks, _, _ = _variable_case(seed)
    orc.density_cycle(ps, cells, tasks)
    orc.ghost(ps, GAMMA)
    f = orc.brute_force(ps)                        # f64 sums: the identity holds to rounding
    m = ps["mass"].astype(np.float64)
    mom = (m[:, None] * f[:, :3]).sum(axis=0)
    assert np.abs(mom).max() <= 1e-12 * np.abs(m[:, None] * f[:, :3]).sum()
    en = m * (np.einsum("ij,ij->i", ps["v"].astype(np.float64), f[:, :3]) + f[:, 3])
    assert abs(en.sum()) <= 1e-12 * np.abs(m * f[:, 3]).sum()
    # and the f32 pipeline result keeps them to the north_star's 1e-6
    orc.force_cycle(ps, cells, tasks)
    a = ps["a"].astype(np.float64)
    assert np.abs((m[:, None] * a).sum(axis=0)).max() <= 1e-6 * np.abs(m[:, None] * a).sum()
    en = m * (np.einsum("ij,ij->i", ps["v"].astype(np.float64), a) + ps["du_dt"])
    assert abs(en.sum()) <= 1e-6 * np.abs(m * ps["du_dt"].astype(np.float64)).sum()


def test_force_continuum_limit_pressure_gradient():
    # lattice, v = 0, u = 1 + eps sin(2 pi x): a_x -> -(1/rho) dP/dx = -(gamma-1) eps 2 pi cos(2 pi x)
    n_side, eps = 16, 0.01
    parts = lattice(n_side, 1.2348)
    parts["u"] = 1.0 + eps * np.sin(2 * np.pi * parts["x"][:, 0])
    ps, cells, tasks, _, _ = sort_grid(parts, 4)
    orc.density_cycle(ps, cells, tasks)
    orc.ghost(ps, GAMMA)
    orc.force_cycle(ps, cells, tasks)
    expect = -(GAMMA - 1.0) * eps * 2 * np.pi * np.cos(2 * np.pi * ps["x"][:, 0])
    amp = np.dot(ps["a"][:, 0], expect) / np.dot(expect, expect)       # least-squares amplitude ratio
    assert 0.9 < amp < 1.1
    assert np.abs(ps["a"][:, 1:]).max() < 1e-4 * np.abs(expect).max() + 2e-5


# ------------------------------------------------------------------ cells and tasks

def _morton_code(x, origin, width):
    """reading C26, restated: 5 bits per axis of floor((x - origin) / width * 32), x most significant in every bit triple"""
    q = np.clip(np.floor((x - origin) / width * 32.0), 0, 31).astype(np.int64)
    code = np.zeros(x.shape[0], dtype=np.int64)
    for b in range(5):
        for d in range(3):
            code |= ((q[:, d] >> b) & 1) << (3 * b + (2 - d))
    return code


def test_order_inside_a_cell_is_morton_and_compact():
    # hand-placed points in one cell of a 3^3 grid: the order is fixed by the definition (octant 4bx + 2by + bz first, then
    # the same rule inside the octant), whatever order they were generated in
    w = 1.0 / 3.0
    rel = np.array([[0.9, 0.9, 0.9], [0.1, 0.1, 0.1], [0.1, 0.1, 0.9], [0.9, 0.1, 0.1], [0.1, 0.9, 0.1], [0.3, 0.1, 0.1], [0.1, 0.1, 0.3],
                    [0.1, 0.1, 0.1]])
    parts = np.zeros(rel.shape[0], dtype=si.PART_DTYPE)
    parts["x"] = (1.0 + rel) * w                       # all in cell (1, 1, 1)
    parts["id"] = np.arange(rel.shape[0])
    perm, cells = orc.cells_build_grid(parts["x"], 3)
    c = 13
    assert cells["count"][c] == rel.shape[0] and cells["count"].sum() == rel.shape[0]
    # octant 0: (.1,.1,.1) twice in generator order [1, 7], then z-neighbour (.1,.1,.3) [6], x-neighbour (.3,.1,.1) [5];
    # then octants 1 (z high) [2], 2 (y high) [4], 4 (x high) [3], 7 [0]
    assert perm.tolist() == [1, 7, 6, 5, 2, 4, 3, 0]
    # a jittered lattice: any 8 consecutive particles of a 64-particle cell form one octant of it
    parts = si.jittered_lattice(12, 3, jitter=0.2)
    perm, cells = orc.cells_build_grid(parts["x"], 3)
    ps = parts[perm.astype(np.int64)]
    for c in (0, 13, 26):
        f = int(cells["first"][c])
        assert cells["count"][c] == 64
        for o in range(8):
            x = (ps["x"][f + 8 * o:f + 8 * o + 8] - cells["origin"][c]) / cells["width"][c]
            assert np.all((x >= 0.5) == np.array([(o >> 2) & 1, (o >> 1) & 1, o & 1], dtype=bool))


def test_grid_cells_and_tasks_structure():
    parts = si.jittered_lattice(12, 7)
    perm, cells = orc.cells_build_grid(parts["x"], 4)
    assert sorted(perm.tolist()) == list(range(12 ** 3))
    ps = parts[perm.astype(np.int64)]
    # particles inside their cell's box, cells contiguous, Morton order inside a cell with ties in generator order (C26)
    for c in range(64):
        f, k = int(cells["first"][c]), int(cells["count"][c])
        x = ps["x"][f:f + k]
        assert np.all(x >= cells["origin"][c]) and np.all(x < cells["origin"][c] + cells["width"][c])
        code = _morton_code(x, cells["origin"][c], cells["width"][c])
        key = code.astype(np.int64) * (1 << 32) + ps["id"][f:f + k]
        assert np.all(np.diff(key) > 0)
    assert cells["first"][0] == 0 and np.all(cells["first"][1:] == np.cumsum(cells["count"])[:-1])
    tasks, ns, npair = orc.tasks_build(cells, orc.cell_hmax(ps, cells))
    assert (ns, npair) == (64, 64 * 13)
    assert np.all(tasks["ci"][:64] == np.arange(64)) and np.all(tasks["cj"][:64] == -1)
    pr = tasks[64:]
    assert np.all(pr["ci"] < pr["cj"])
    key = pr["ci"].astype(np.int64) * 64 + pr["cj"]
    assert np.all(np.diff(key) > 0)
    # every cell has exactly 26 distinct neighbours
    nb = np.bincount(np.concatenate([pr["ci"], pr["cj"]]), minlength=64)
    assert np.all(nb == 26)
    # frames: both sides land in one frame anchored at ci: xr_i in [0, w), xr_j in [-w, 2w)
    w = cells["width"][0]
    for t in pr[::37]:
        ci, cj = int(t["ci"]), int(t["cj"])
        assert np.all(t["frame_i"] == cells["origin"][ci])
        xj = ps["x"][int(cells["first"][cj]):int(cells["first"][cj]) + int(cells["count"][cj])] - t["frame_j"]
        assert np.all(xj >= -w) and np.all(xj < 2 * w)
        shift = cells["origin"][ci] - t["frame_j"]
        assert np.all(np.isin(shift, [-1.0, 0.0, 1.0]))


def test_task_rule_depends_on_hmax():
    # a pair exists only if the box gap is below max(2 hmax_A, 2 hmax_B): with tiny h only touching cells pair up,
    # with h > width/2 second neighbours do too (6^3 grid so that images stay unique)
    parts = lattice(12, 0.4)
    ps, cells, tasks, ns, npair = sort_grid(parts, 6)
    assert npair == 216 * 13
    parts["h"] = 1.1 / 12       # 2h = 2.2 dx > width = 2 dx  -> gap of one cell width (2 dx) is inside the cut-off
    ps, cells, tasks, ns, npair = sort_grid(parts, 6)
    # offsets (a, b, c) in [-2, 2]^3 with gap = 2 dx * |(max(0,|a|-1), ...)| < 2.2 dx: the 26 touching ones plus the
    # 3 * 2 * 9 with exactly one |offset| = 2 (gap 2 dx); two such axes give 2.83 dx -> 80 neighbours, 40 pairs per cell
    assert npair == 216 * 40
    orc.density_cycle(ps, cells, tasks)
    ref = orc.brute_density(ps)
    assert np.max(np.abs(ps["rho"] - ref[:, 0]) / ref[:, 0]) < 5e-6


def test_octree_cells():
    parts = si.clumpy_mixture(20000, seed=3, n_clumps=4, frac_clumps=0.7, sigma=0.03, h_cap=1.0 / 32)
    perm, cells = orc.cells_build_octree(parts["x"], parts["h"], 100)
    assert sorted(perm.tolist()) == list(range(20000))
    ps = parts[perm.astype(np.int64)]
    assert cells["count"].sum() == 20000 and np.all(cells["count"] > 0)
    assert np.all(cells["first"][1:] == np.cumsum(cells["count"])[:-1])
    hmax = orc.cell_hmax(ps, cells)
    for c in range(cells.shape[0]):
        f, k = int(cells["first"][c]), int(cells["count"][c])
        x = ps["x"][f:f + k]
        assert np.all(x >= cells["origin"][c]) and np.all(x < cells["origin"][c] + cells["width"][c])
        # a leaf is either small enough or could not be split: one of its non-empty octants would be narrower than
        # 2 hmax of the particles in that octant (the octants are recomputed here from the positions)
        if k > 100:
            half = 0.5 * cells["width"][c]
            octant = ((x >= cells["origin"][c] + half) * np.array([4, 2, 1])).sum(axis=1)
            hh = ps["h"][f:f + k].astype(np.float64)
            assert any(half < 2.0 * hh[octant == o].max() for o in np.unique(octant))
        assert cells["width"][c] >= 2 * hmax[c] or cells["width"][c] == 1.0
    assert len(set(cells["width"].tolist())) > 1            # really adaptive
    assert cells["count"].max() <= 100 or np.any(cells["width"] / 2 < 2 * hmax)


def test_octree_pipeline_vs_brute_force():
    parts = si.clumpy_mixture(6000, seed=5, n_clumps=3, frac_clumps=0.6, sigma=0.05, h_cap=1.0 / 24)
    ps, cells, tasks, ns, npair = sort_octree(parts, 60)
    assert ns == cells.shape[0] and npair > 0
    orc.density_cycle(ps, cells, tasks, batch=50)
    ref = orc.brute_density(ps)
    assert np.max(np.abs(ps["rho"] - ref[:, 0]) / ref[:, 0]) < 5e-6
    assert np.max(scaled_err(ps["wcount_dh"], ref[:, 3], ref[:, 2] / ps["h"])) < 5e-6


# ------------------------------------------------------------------ pack

def _pattern_store(n):
    """every scalar of particle p, field f, component c holds a value that encodes (p, f, c)."""
    parts = np.zeros(n, dtype=si.PART_DTYPE)
    p = np.arange(n)
    for f, name in enumerate(si.FIELDS):
        nc = si.FIELD_NCOMP[f]
        for c in range(nc):
            code = p * 1000 + f * 10 + c
            if name == "x":
                parts[name][:, c] = code + 0.25
            elif name == "id":
                parts[name] = code
            elif name == "time_bin":
                parts[name] = (p % 100).astype(np.int8)
            elif nc == 3:
                parts[name][:, c] = code.astype(np.float32)
            else:
                parts[name] = code.astype(np.float32)
    return parts


def _one_cell_setup(n):
    cells = np.zeros(2, dtype=orc.CELL_DTYPE)
    cells["first"], cells["count"], cells["width"] = [0, n // 2], [n // 2, n - n // 2], 0.5
    tasks = np.zeros(3, dtype=orc.TASK_DTYPE)
    tasks["ci"], tasks["cj"] = [0, 1, 0], [-1, -1, 1]
    tasks["frame_i"][2] = [1.0, 2.0, 3.0]
    tasks["frame_j"][2] = [-4.0, 0.5, 8.0]
    return cells, tasks


def test_pack_puts_the_right_bytes_at_the_right_offsets():
    n = 13
    parts = _pattern_store(n)
    cells, tasks = _one_cell_setup(n)
    attrset = ([(orc.V, 1, 2), (orc.X, 0, 3), (orc.ID, 0, 1), (orc.TIME_BIN, 0, 1), (orc.ROT_V, 2, 1), (orc.CS, 0, 1)], 0)
    rec = orc.record_bytes(attrset)
    assert rec == 8 + 24 + 8 + 4 + 4 + 4
    buf = orc.pack(parts, cells, tasks, attrset, fill=0xEE)
    off, total = orc.block_offsets(cells, tasks, rec)
    # layout: blocks start at multiples of 128, in task order, side i then side j
    assert np.all(off[[0, 2, 4, 5]] % 128 == 0) and off[0] == 0 and off[1] == off[3] == 2 ** 64 - 1
    assert off[2] == -(-6 * rec // 128) * 128 and total % 128 == 0
    for t, side, c in [(0, 0, 0), (1, 0, 1), (2, 0, 0), (2, 1, 1)]:
        first, count = int(cells["first"][c]), int(cells["count"][c])
        blk = buf[int(off[2 * t + side]):int(off[2 * t + side]) + count * rec].reshape(count, rec)
        p = np.arange(first, first + count)
        assert np.array_equal(blk[:, 0:8].copy().view(np.float32), np.stack([p * 1000 + 11, p * 1000 + 12], 1).astype(np.float32))
        assert np.array_equal(blk[:, 8:32].copy().view(np.float64), np.stack([p * 1000 + c2 + 0.25 for c2 in range(3)], 1))
        assert np.array_equal(blk[:, 32:40].copy().view(np.int64).ravel(), p * 1000 + 160)
        assert np.array_equal(blk[:, 40], (p % 100).astype(np.uint8)) and np.all(blk[:, 41:44] == 0)
        assert np.array_equal(blk[:, 44:48].copy().view(np.float32).ravel(), (p * 1000 + 122).astype(np.float32))
        assert np.array_equal(blk[:, 48:52].copy().view(np.float32).ravel(), (p * 1000 + 140).astype(np.float32))
        # pad bytes after the block are untouched
        end = int(off[2 * t + side]) + count * rec
        nxt = -(-end // 128) * 128
        assert np.all(buf[end:nxt] == 0xEE)


def test_pack_relative_coordinates_one_subtraction_one_rounding():
    n = 13
    parts = _pattern_store(n)
    rng = np.random.default_rng(11)
    parts["x"] = rng.random((n, 3)) * 3.0
    cells, tasks = _one_cell_setup(n)
    buf = orc.pack(parts, cells, tasks, orc.DENSITY_IN)
    off, _ = orc.block_offsets(cells, tasks, 20)
    blk = buf[int(off[5]):int(off[5]) + 7 * 20].copy().view(np.float32).reshape(7, 5)
    xl = parts["x"][6:13].astype(np.longdouble) - tasks["frame_j"][2].astype(np.longdouble)
    assert np.array_equal(blk[:, :3], xl.astype(np.float64).astype(np.float32))     # f64 subtract is exact enough: see below
    assert np.array_equal(blk[:, :3], (parts["x"][6:13] - tasks["frame_j"][2]).astype(np.float32))
    assert np.array_equal(blk[:, 3], parts["h"][6:13]) and np.array_equal(blk[:, 4], parts["mass"][6:13])
    # side i of the same task uses frame_i
    blk_i = buf[int(off[4]):int(off[4]) + 6 * 20].copy().view(np.float32).reshape(6, 5)
    assert np.array_equal(blk_i[:, :3], (parts["x"][0:6] - tasks["frame_i"][2]).astype(np.float32))


def test_self_task_coordinates_inside_cell():
    parts = si.config0(seed=2)
    ps, cells, tasks, ns, _ = sort_grid(parts, 4)
    buf = orc.pack(ps, cells, tasks[:ns], orc.DENSITY_IN)
    off, _ = orc.block_offsets(cells, tasks[:ns], 20)
    for t in range(ns):
        xr = buf[int(off[2 * t]):int(off[2 * t]) + 64 * 20].copy().view(np.float32).reshape(64, 5)[:, :3]
        assert xr.min() >= 0.0 and xr.max() < 0.25


def test_attrset_validation():
    assert orc.record_bytes(orc.DENSITY_IN) == 20 and orc.record_bytes(orc.DENSITY_OUT) == 16
    assert orc.record_bytes(orc.FORCE_IN) == 52 and orc.record_bytes(orc.FORCE_OUT) == 20
    assert orc.record_bytes(([(orc.V, 0, 2), (orc.V, 1, 1)], 0)) == -1          # component listed twice
    assert orc.record_bytes(([(orc.MASS, 0, 2)], 0)) == -1                      # scalar has one component
    assert orc.record_bytes(([(18, 0, 1)], 0)) == -1


# ------------------------------------------------------------------ unpack

def test_pack_then_unpack_identity_assign():
    n = 29
    parts = _pattern_store(n)
    cells, tasks = _one_cell_setup(n)
    attrset = ([(orc.X, 0, 3), (orc.V, 0, 3), (orc.RHO, 0, 1), (orc.ID, 0, 1), (orc.TIME_BIN, 0, 1), (orc.ROT_V, 1, 1)], 0)
    buf = orc.pack(parts, cells, tasks, attrset)
    scr = raw_copy(parts)
    for name in ("x", "v", "rho", "id", "time_bin", "rot_v", "mass", "P"):
        scr[name] = (scr[name] * 0 + 77).astype(scr[name].dtype)
    orc.unpack(scr, cells, tasks, attrset, buf, orc.MODE_ASSIGN)
    for name in ("x", "v", "rho", "id", "time_bin"):
        assert np.array_equal(scr[name], parts[name])
    assert np.array_equal(scr["rot_v"][:, 1], parts["rot_v"][:, 1])
    # untouched members and pad bytes keep the scrambled / original content
    assert np.all(scr["rot_v"][:, [0, 2]] == 77) and np.all(scr["mass"] == 77) and np.all(scr["P"] == 77)
    raw_a, raw_b = scr.view(np.uint8).reshape(n, 128), parts.view(np.uint8).reshape(n, 128)
    assert np.array_equal(raw_a[:, 108:112], raw_b[:, 108:112]) and np.array_equal(raw_a[:, 121:], raw_b[:, 121:])


def test_unpack_reduce_operators_and_order():
    n = 10
    cells, tasks = _one_cell_setup(n)          # cell 0 occurs in tasks 0 and 2, cell 1 in tasks 1 and 2
    attrset = ([(orc.RHO, 0, 1), (orc.V_SIG, 0, 1), (orc.U, 0, 1), (orc.A, 0, 3), (orc.DU_DT, 0, 1)], 0)
    rec = orc.record_bytes(attrset)
    off, total = orc.block_offsets(cells, tasks, rec)
    buf = np.zeros(total, dtype=np.uint8)
    rng = np.random.default_rng(5)
    blocks = {}
    for t, side, c in [(0, 0, 0), (1, 0, 1), (2, 0, 0), (2, 1, 1)]:
        vals = rng.integers(-1000, 1000, size=(5, 7)).astype(np.float32)       # integer-valued: sums are exact
        blocks[(t, c)] = vals
        o = int(off[2 * t + side])
        buf[o:o + 5 * rec] = vals.view(np.uint8).ravel()
    parts = np.zeros(n, dtype=si.PART_DTYPE)
    parts["rho"], parts["v_sig"], parts["u"] = 3.0, -5000.0, 9.0
    orc.unpack(parts, cells, tasks, attrset, buf, orc.MODE_REDUCE)
    for c, (ta, tb) in [(0, (0, 2)), (1, (1, 2))]:
        sl = slice(5 * c, 5 * c + 5)
        a, b = blocks[(ta, c)], blocks[(tb, c)]
        assert np.array_equal(parts["rho"][sl], 3.0 + a[:, 0] + b[:, 0])                    # sum
        assert np.array_equal(parts["v_sig"][sl], np.maximum(a[:, 1], b[:, 1]))             # max (initial -5000 loses)
        assert np.array_equal(parts["u"][sl], b[:, 2])                                      # not a sum field: last task wins
        assert np.array_equal(parts["a"][sl], a[:, 3:6] + b[:, 3:6])
        assert np.array_equal(parts["du_dt"][sl], a[:, 6] + b[:, 6])
    # f32 addition order: ((s + a) + b) in task order, checked with values whose f32 sum depends on the order
    buf2 = np.zeros(total, dtype=np.uint8)
    one = np.zeros((5, 7), dtype=np.float32)
    big, small = one.copy(), one.copy()
    big[:, 0], small[:, 0] = 2.0 ** 24, 1.0
    for (t, side), vals in {(0, 0): small, (2, 0): big, (1, 0): big, (2, 1): small}.items():
        o = int(off[2 * t + side])
        buf2[o:o + 5 * rec] = vals.view(np.uint8).ravel()
    parts["rho"] = 1.0
    orc.unpack(parts, cells, tasks, attrset, buf2, orc.MODE_REDUCE)
    assert np.all(parts["rho"][:5] == np.float32(2.0 ** 24 + 2.0))      # (1 + 1) + 2^24 is exact
    assert np.all(parts["rho"][5:] == np.float32(2.0 ** 24))            # (1 + 2^24) rounds to 2^24, then + 1 rounds back


def test_zero_clears_the_listed_components_and_nothing_else():
    # a store whose every member is non-zero: after zero(set) the listed components are +0.0, every other byte is unchanged
    # (catches a zero that does nothing, one that clears whole fields instead of components, one that touches neighbours)
    n = 23
    parts = _pattern_store(n)
    raw0 = parts.view(np.uint8).reshape(n, 128).copy()
    assert np.all(parts["rho"] != 0) and np.all(parts["a"] != 0) and np.all(parts["v_sig"] != 0)
    orc.zero(parts, ([(orc.RHO, 0, 1), (orc.A, 1, 2), (orc.V_SIG, 0, 1)], 0))
    raw1 = parts.view(np.uint8).reshape(n, 128)
    cleared = np.zeros(128, dtype=bool)
    for off in (64, 36 + 4, 36 + 8, 104):            # rho @64, a[1] @40, a[2] @44, v_sig @104 (reading C16)
        cleared[off:off + 4] = True
    assert np.all(raw1[:, cleared] == 0)
    assert np.array_equal(raw1[:, ~cleared], raw0[:, ~cleared])
    # the canonical output sets: every output of the loop about to run is zero, inputs are untouched
    parts = _pattern_store(n)
    keep = {k: parts[k].copy() for k in ("x", "v", "mass", "h", "u", "P", "c_s", "id", "time_bin", "div_v", "rot_v")}
    orc.zero(parts, orc.DENSITY_OUT)
    for k in ("rho", "rho_dh", "wcount", "wcount_dh"):
        assert np.all(parts[k] == 0)
    assert np.all(parts["a"] != 0) and np.all(parts["du_dt"] != 0) and np.all(parts["v_sig"] != 0)
    orc.zero(parts, orc.FORCE_OUT)
    for k in ("a", "du_dt", "v_sig"):
        assert np.all(parts[k] == 0)
    for k, v in keep.items():
        assert np.array_equal(parts[k], v)
    with pytest.raises(ValueError):
        orc.zero(parts, ([(orc.X, 0, 3)], 0))          # not an f32 member


def test_cycles_start_from_zero_whatever_the_store_held():
    # density_cycle / force_cycle zero their outputs first: running them on a store that already holds results (or
    # garbage) gives the same bits as on a fresh store -- and not twice the sums
    parts = si.jittered_lattice(12, seed=11, h_spread=0.1, mass_spread=0.2, u_spread=0.2)
    ps, cells, tasks, ns, npair = sort_grid(parts, 4)
    fresh = raw_copy(ps)
    orc.density_cycle(fresh, cells, tasks)
    orc.ghost(fresh, GAMMA)
    orc.force_cycle(fresh, cells, tasks)
    again = raw_copy(fresh)                             # outputs of a whole step are in the store
    again["v_sig"] = 1.0e6                              # a max that did not restart from 0 would keep this
    orc.density_cycle(again, cells, tasks)
    orc.ghost(again, GAMMA)
    orc.force_cycle(again, cells, tasks)
    assert np.array_equal(again.view(np.uint8), fresh.view(np.uint8))
    assert np.all(fresh["rho"] > 0) and np.all(fresh["v_sig"] > 0)


def test_unpack_rejects_relative_coordinates():
    cells, tasks = _one_cell_setup(4)
    with pytest.raises(ValueError):
        orc.unpack(np.zeros(4, dtype=si.PART_DTYPE), cells, tasks, orc.DENSITY_IN, np.zeros(1024, np.uint8))


# ------------------------------------------------------------------ h iteration (C20)

def test_h_iteration_on_lattice():
    n_side = 12
    parts = lattice(n_side, 1.2)
    h, bad = orc.iterate_h(parts["x"], parts["h"], h_cap=1.0 / 6.0, tol=1e-6, max_iter=60)
    assert bad == 0
    assert np.allclose(h * n_side, 1.12574487, rtol=0, atol=2e-6)
    # and the result satisfies the condition through the independent pipeline
    parts["h"] = h
    ps, cells, tasks, _, _ = sort_grid(parts, 4)
    orc.density_cycle(ps, cells, tasks)
    nngb = 4.0 / 3.0 * math.pi * (2.0 * ps["h"].astype(np.float64)) ** 3 * ps["wcount"]
    assert np.allclose(nngb, 48.0, atol=1e-3)


# ------------------------------------------------------------------ gradient loop and Balsara switch (reading C34, row f2)

def _gold_omega(h_over_dx):
    for row in _gold_rows():
        if abs(row[0] - h_over_dx) < 1e-12:
            rho_n, rho_dh_n = row[2], row[3]              # rho dx^3 / m and rho_dh dx^4 / m
            return 1.0 + h_over_dx * rho_dh_n / (3.0 * rho_n)
    raise KeyError(h_over_dx)


def _velocity_field(parts, A, box=1.0):
    """v = A (x - centre), kept linear across the periodic wrap by using only particles far from the box faces in the checks"""
    parts["v"] = ((parts["x"] - 0.5) @ np.asarray(A, dtype=np.float64).T).astype(np.float32)
    return parts


@pytest.mark.parametrize("h_over_dx", [1.2348, 1.0, 1.5])
def test_gradient_of_a_linear_field_on_a_lattice(h_over_dx):
    # For v = A x on an unperturbed lattice the estimator gives A's trace (divergence) and antisymmetric part (curl) times
    # S = -(1/3) sum_j (m_j / rho_j) r dW/dr.  Because dW/dh = -(3 W + r dW/dr) / h, S = 1 + h rho_dh / (3 rho) = Omega: the grad-h
    # factor of the SAME lattice, whose value comes from the independent lattice sums of tests/golden/ (0.981238565203 at 1.2348).
    n_side = 16
    omega_l = _gold_omega(h_over_dx)
    A = np.array([[0.3, -0.2, 0.5], [0.7, -0.1, 0.05], [-0.4, 0.6, 0.9]])
    parts = _velocity_field(lattice(n_side, h_over_dx), A)
    ps, cells, tasks, _, _ = sort_grid(parts, 4)
    orc.density_cycle(ps, cells, tasks)
    orc.gradient_cycle(ps, cells, tasks)
    inner = np.all(np.abs(ps["x"] - 0.5) < 0.5 - 2.1 * h_over_dx / n_side, axis=1)      # the field is linear inside their support
    assert inner.sum() > 500
    curl = np.array([A[2, 1] - A[1, 2], A[0, 2] - A[2, 0], A[1, 0] - A[0, 1]])
    assert np.allclose(ps["div_v"][inner], np.trace(A) * omega_l, rtol=0, atol=3e-6)
    assert np.allclose(ps["rot_v"][inner], curl * omega_l, rtol=0, atol=3e-6)
    # a transposed operand (A^T gives -curl), a wrong sign of e or dv, or rho_i instead of rho_j would all show:
    # rigid rotation about z: div = 0, rot = 2 w z; pure strain: rot = 0
    w = 0.37
    parts = _velocity_field(lattice(n_side, h_over_dx), [[0, -w, 0], [w, 0, 0], [0, 0, 0]])
    ps, cells, tasks, _, _ = sort_grid(parts, 4)
    orc.density_cycle(ps, cells, tasks)
    orc.gradient_cycle(ps, cells, tasks)
    assert np.allclose(ps["rot_v"][inner], np.array([0, 0, 2 * w]) * omega_l, atol=3e-6) and np.allclose(ps["div_v"][inner], 0, atol=3e-6)
    parts = _velocity_field(lattice(n_side, h_over_dx), [[0.5, 0.2, 0], [0.2, -0.5, 0.1], [0, 0.1, 0]])
    ps, cells, tasks, _, _ = sort_grid(parts, 4)
    orc.density_cycle(ps, cells, tasks)
    orc.gradient_cycle(ps, cells, tasks)
    assert np.allclose(ps["rot_v"][inner], 0, atol=3e-6) and np.allclose(ps["div_v"][inner], 0, atol=3e-6)


def test_gradient_uses_the_neighbours_volume_and_the_targets_h():
    # two isolated particles, hand-worked: i at the origin (h_i = 0.1), j at distance 0.05 along x (h_j = 0.3 must not matter for i)
    parts = np.zeros(2, dtype=si.PART_DTYPE)
    parts["x"] = [[0.40, 0.5, 0.5], [0.45, 0.5, 0.5]]
    parts["h"], parts["mass"], parts["rho"], parts["u"] = [0.1, 0.3], [2.0, 3.0], [5.0, 7.0], 1.0
    parts["v"] = [[0.0, 0.0, 0.0], [0.2, 0.6, -0.4]]
    parts["id"] = [0, 1]
    cells = np.zeros(1, dtype=orc.CELL_DTYPE)
    cells["count"], cells["width"] = 2, 1.0
    tasks = np.zeros(1, dtype=orc.TASK_DTYPE)
    tasks["cj"] = -1
    out = orc.gradient(cells, tasks, orc.pack(parts, cells, tasks, orc.GRADIENT_IN)).view(np.float32)[:8].reshape(2, 4)
    # i: q = 0.5, w'(0.5) = -0.9375, dW/dr = w' / (pi h^4); e = (x_i - x_j) / r = (-1, 0, 0); dv = v_j - v_i
    g = 3.0 / 7.0 * (-0.9375) / (math.pi * 0.1 ** 4)
    assert np.allclose(out[0], [g * (-0.2), 0.0, g * (-0.4), g * (-0.6)], rtol=1e-6)       # e x dv = (0, dvz, -dvy) for e = -x
    # j: h_j = 0.3, q = 1/6 < 1: w' = -3q + 2.25 q^2; neighbour's volume m_i / rho_i; e = (+1, 0, 0); dv = v_i - v_j
    q = 0.05 / 0.3
    g = 2.0 / 5.0 * (-3 * q + 2.25 * q * q) / (math.pi * 0.3 ** 4)
    assert np.allclose(out[1], [g * (-0.2), 0.0, g * (-0.4), g * (-0.6)], rtol=1e-6)      # e = +x, dv = -v_j: e x dv = (0, -dvz, dvy)


def test_gradient_pipeline_vs_brute_force():
    parts = si.jittered_lattice(12, 9, jitter=0.5, sigma_v=0.2, h_spread=0.15, mass_spread=0.3)
    ps, cells, tasks, _, _ = sort_grid(parts, 4)
    orc.density_cycle(ps, cells, tasks)
    orc.gradient_cycle(ps, cells, tasks, batch=31)
    ref = orc.brute_gradient(ps)
    scale = np.abs(ref).max()
    assert np.max(np.abs(ps["div_v"] - ref[:, 0])) < 5e-6 * scale and np.max(np.abs(ps["rot_v"] - ref[:, 1:])) < 5e-6 * scale
    assert np.abs(ps["div_v"]).max() > 0.1 and np.abs(ps["rot_v"]).max() > 0.1


def _three_loop_state(seed):
    parts = si.jittered_lattice(12, seed, jitter=0.5, sigma_v=0.3, h_spread=0.15, mass_spread=0.3, u_spread=0.3)
    ps, cells, tasks, _, _ = sort_grid(parts, 4)
    orc.density_cycle(ps, cells, tasks)
    orc.ghost(ps, GAMMA)
    return ps, cells, tasks


def test_balsara_switch_limits():
    ps, cells, tasks = _three_loop_state(21)
    plain = raw_copy(ps)
    orc.force_cycle(plain, cells, tasks)
    off = raw_copy(ps)
    orc.force_cycle(off, cells, tasks, alpha=0.0)
    assert np.abs(plain["a"] - off["a"]).max() > 1e-3 * np.abs(plain["a"]).max()         # the viscosity matters in this state
    # pure compression (rot v = 0, |div v| overwhelming the c_s / h floor): B = 1 exactly, the three-loop force IS the plain force
    comp = raw_copy(ps)
    comp["div_v"], comp["rot_v"] = -1.0e30, 0.0
    orc.force3_cycle(comp, cells, tasks)
    for k in ("a", "du_dt", "v_sig"):
        assert np.array_equal(comp[k], plain[k]), k
    # pure shear (div v = 0): B = 0, the viscous term vanishes -- the plain force with alpha = 0 (v_sig is not switched)
    shear = raw_copy(ps)
    shear["div_v"], shear["rot_v"] = 0.0, [[0.3, -2.0, 1.0]]
    orc.force3_cycle(shear, cells, tasks)
    assert np.array_equal(shear["a"], off["a"]) and np.array_equal(shear["du_dt"], off["du_dt"]) and np.array_equal(shear["v_sig"], plain["v_sig"])
    # B = 1/2 everywhere (|div| = |rot|, floor negligible): exactly the plain force at half the alpha
    half = raw_copy(ps)
    half["div_v"], half["rot_v"] = 2.0e20, [[0.0, 2.0e20, 0.0]]
    orc.force3_cycle(half, cells, tasks)
    ref = raw_copy(ps)
    orc.force_cycle(ref, cells, tasks, alpha=0.4)
    assert np.allclose(half["a"], ref["a"], rtol=1e-6, atol=1e-6 * np.abs(ref["a"]).max())


def test_three_loop_step_conserves_momentum_and_energy():
    ps, cells, tasks = _three_loop_state(22)
    orc.gradient_cycle(ps, cells, tasks)
    orc.force3_cycle(ps, cells, tasks)
    B = np.abs(ps["div_v"]) / (np.abs(ps["div_v"]) + np.linalg.norm(ps["rot_v"], axis=1) + 1e-4 * ps["c_s"] / ps["h"])
    assert B.min() < 0.2 and 0.8 < B.max() <= 1.0 and 0.2 < B.std()                        # the switch really varies from particle to particle
    m, a = ps["mass"].astype(np.float64), ps["a"].astype(np.float64)
    assert np.abs((m[:, None] * a).sum(0)).max() <= 1e-6 * np.abs(m[:, None] * a).sum()
    en = m * (np.einsum("ij,ij->i", ps["v"].astype(np.float64), a) + ps["du_dt"])
    assert abs(en.sum()) <= 1e-6 * np.abs(m * ps["du_dt"].astype(np.float64)).sum()


def test_three_loop_record_layouts():
    # Table 1: p-g = x, v, mass, h, u, rho; p-f adds time_bin
    assert orc.record_bytes(orc.GRADIENT_IN) == 40 and orc.record_bytes(orc.GRADIENT_OUT) == 16 and orc.record_bytes(orc.FORCE3_IN) == 72
    parts = _pattern_store(6)
    cells, tasks = _one_cell_setup(6)
    rec = orc.pack(parts, cells, tasks, orc.FORCE3_IN)[:72].view(np.float32)
    f = {name: i for i, name in enumerate(si.FIELDS)}
    assert rec[3] == f["h"] * 10 and rec[13] == f["div_v"] * 10 and list(rec[14:17]) == [f["rot_v"] * 10 + c for c in range(3)]
    assert rec[17:18].view(np.uint32)[0] == 0                                              # time_bin of particle 0: one byte, zero-extended
    # div_v and rot_v are neighbour sums: REDUCE adds them up over the tasks
    buf = np.zeros(orc.block_offsets(cells, tasks, 16)[1], dtype=np.uint8)
    off, _ = orc.block_offsets(cells, tasks, 16)
    for t, side in ((0, 0), (2, 0)):
        buf[int(off[2 * t + side]):int(off[2 * t + side]) + 16 * 3].view(np.float32)[:] = 1.5
    p2 = np.zeros(6, dtype=si.PART_DTYPE)
    orc.unpack(p2, cells, tasks, orc.GRADIENT_OUT, buf, orc.MODE_REDUCE)
    assert np.all(p2["div_v"][:3] == 3.0) and np.all(p2["rot_v"][:3] == 3.0) and np.all(p2["div_v"][3:] == 0)


# ------------------------------------------------------------------ pins of the test-support functions and of the Balsara floor

def test_compare_blocks_finds_the_first_differing_record_byte_and_skips_pad_bytes():
    """orc.compare_blocks is the only comparator of four GPU tests: it must say -1 for equal block bytes whatever the pad bytes
    hold, and the smallest differing offset otherwise -- on side i and side j, in the first and in a later task."""
    cells = np.zeros(3, dtype=orc.CELL_DTYPE)
    cells["count"], cells["first"], cells["width"] = [3, 5, 2], [0, 3, 8], 1.0
    tasks = np.zeros(4, dtype=orc.TASK_DTYPE)
    tasks["ci"], tasks["cj"] = [0, 1, 0, 2], [-1, -1, 1, -1]
    rec = 20
    off, total = orc.block_offsets(cells, tasks, rec)
    # blocks of 60, 100, 60, 100, 40 bytes, each starting on a 128-byte line
    assert [int(o) for o in off[[0, 2, 4, 5, 6]]] == [0, 128, 256, 384, 512] and total == 640
    rng = np.random.default_rng(3)
    a = rng.integers(0, 256, total).astype(np.uint8)
    b = a.copy()
    assert orc.compare_blocks(cells, tasks, rec, a, b) == -1
    b[60:128] ^= 0xFF                                            # the pad bytes behind the first block, all of them
    b[484:512] ^= 0xFF                                           # ... and behind side j of the pair task
    assert orc.compare_blocks(cells, tasks, rec, a, b) == -1
    for where in (0, 59, 128 + 99, 256 + 17, 384, 384 + 99, 512 + 39):      # first / last byte of blocks, side i and side j of the pair task
        c = b.copy()
        c[where] ^= 0x01
        assert orc.compare_blocks(cells, tasks, rec, a, c) == where, where
        assert orc.compare_blocks(cells, tasks, rec, c, a) == where, where
    c = b.copy()
    c[512 + 5] ^= 0x80
    c[384 + 70] ^= 0x80
    c[256 + 59] ^= 0x80
    assert orc.compare_blocks(cells, tasks, rec, a, c) == 256 + 59      # the smallest offset, whichever thread finds which


def _force3_pair(div_i, rot_i, div_j, rot_j):
    """the two-particle FORCE_IN case of test_force_two_particles_hand_worked as FORCE3_IN records (18 words)"""
    rec = np.zeros((2, 18), dtype=np.float32)
    #            xr0   xr1  xr2  h    m    rho  rho_dh v0    v1   v2   u    P    cs
    rec[0, :13] = [0.00, 0.0, 0.0, 0.1, 1.5, 2.0, 0.0, 0.3, 0.0, 0.0, 1.0, 2.0, 1.0]
    rec[1, :13] = [0.05, 0.0, 0.0, 0.1, 2.5, 3.0, 0.0, -0.1, 0.0, 0.0, 1.0, 3.0, 1.25]
    rec[0, 13], rec[0, 14:17] = div_i, rot_i
    rec[1, 13], rec[1, 14:17] = div_j, rot_j
    cells = np.zeros(1, dtype=orc.CELL_DTYPE)
    cells["count"], cells["width"] = 2, 1.0
    tasks = np.zeros(1, dtype=orc.TASK_DTYPE)
    tasks["cj"] = -1
    buf = np.zeros(256, dtype=np.uint8)
    buf[:144] = rec.view(np.uint8).ravel()
    return orc.force3(cells, tasks, buf, alpha=0.8, beta=3.0)[:40].view(np.float32).reshape(2, 5)


def test_balsara_floor_hand_worked():
    """B = |div v| / (|div v| + |rot v| + 1e-4 c_s / h) (reading C34; Table 1 column p-f) with the floor term a
    quarter of the denominator, every factor a number chosen here: a floor of 1e-3 or 1e-5, c_s h instead of c_s / h, or the
    rotation entering by a component instead of its norm all miss the expected values by far more than the tolerance."""
    # i: c_s / h = 1.0 / 0.1 -> floor 1.0e-3;  |div| = 2.0e-3, |rot| = 0.5e-3  -> B_i = 2 / (2 + 0.5 + 1)        = 4/7
    # j: c_s / h = 1.25 / 0.1 -> floor 1.25e-3; |div| = 3.0e-3, |rot| = |(0.75, 0, 1) e-3| = 1.25e-3 -> B_j = 3 / 5.5 = 6/11
    out = _force3_pair(-2.0e-3, [0.0, 0.0, 0.5e-3], 3.0e-3, [0.75e-3, 0.0, 1.0e-3])
    Bbar = 0.5 * (4.0 / 7.0 + 6.0 / 11.0)                      # 43/77
    assert Bbar == pytest.approx(43.0 / 77.0, rel=1e-15)
    G = -0.9375 / (math.pi * 1e-4)
    vr = mu = -0.4
    vs = 1.0 + 1.25 - 3.0 * mu                                   # 3.45: the signal velocity is not switched
    visc = Bbar * (-0.5 * 0.8 * vs * mu / 2.5)
    F = 0.5 * G + (1.0 / 3.0) * G + visc * G
    assert out[0, 0] == pytest.approx(2.5 * F, rel=2e-6) and out[1, 0] == pytest.approx(-1.5 * F, rel=2e-6)
    assert out[0, 3] == pytest.approx(2.5 * (0.5 * G + 0.5 * visc * G) * vr, rel=2e-6)
    assert out[1, 3] == pytest.approx(1.5 * ((1.0 / 3.0) * G + 0.5 * visc * G) * vr, rel=2e-6)
    assert out[0, 4] == pytest.approx(vs, rel=1e-6) and out[1, 4] == pytest.approx(vs, rel=1e-6)
    # what the same pair gives without the floor (B_i = 2 / 2.5, B_j = 3 / 4.25) is 40 % away in the viscous term: the pin is sharp
    no_floor = 0.5 * (0.8 + 3.0 / 4.25)
    assert abs(no_floor / Bbar - 1.0) > 0.3
    assert abs(out[0, 0] / (2.5 * (0.5 * G + G / 3.0 + no_floor * (visc / Bbar) * G)) - 1.0) > 0.02
    # with div v and rot v a million times larger the floor vanishes and B_i = 0.8, B_j = 3 / 4.25
    big = _force3_pair(-2.0e3, [0.0, 0.0, 0.5e3], 3.0e3, [0.75e3, 0.0, 1.0e3])
    F_big = 0.5 * G + (1.0 / 3.0) * G + no_floor * (visc / Bbar) * G
    assert big[0, 0] == pytest.approx(2.5 * F_big, rel=2e-6)


def _force_in_records(rows):
    rec = np.zeros((len(rows), 13), dtype=np.float32)
    for k, (x, h) in enumerate(rows):
        rec[k, :3], rec[k, 3], rec[k, 4], rec[k, 5] = x, h, 1.0, 1.0
    return rec


@pytest.mark.parametrize("h_pair", [(0.1, 0.07), (0.07, 0.1)])
def test_flag_cutoff_pairs_marks_exactly_the_pairs_on_the_cutoff(h_pair):
    """reading C31: a particle is exempt from the v_sig comparison iff it has a partner with |r - R_cut| < 1e-5 R_cut,
    R_cut = max(2 h_i, 2 h_j) -- whichever of the two has the larger h, in self tasks and across the two sides of a pair task."""
    hi, hj = (np.float32(h) for h in h_pair)
    cut = max(2.0 * float(hi), 2.0 * float(hj))
    tasks = np.zeros(1, dtype=orc.TASK_DTYPE)
    for delta, expect in ((5e-6, True), (-5e-6, True), (5e-5, False), (-5e-5, False)):
        r = cut * (1.0 + delta)
        # self task, three particles: the pair along y, a bystander 0.05 away from the first (well inside, not on any cut-off)
        rec = _force_in_records([((0.3, 0.1, 0.2), hi), ((0.3, 0.1 + r, 0.2), hj), ((0.35, 0.1, 0.2), np.float32(0.02))])
        cells = np.zeros(1, dtype=orc.CELL_DTYPE)
        cells["count"], cells["width"] = 3, 1.0
        tasks["ci"], tasks["cj"] = 0, -1
        buf = np.zeros(256, dtype=np.uint8)
        buf[:156] = rec.view(np.uint8).ravel()
        assert orc.flag_cutoff_pairs(cells, tasks, buf).tolist() == [expect, expect, False], (delta, h_pair)
        # pair task: two particles on side i (cell 1: store particles 2, 3), two on side j (cell 0: particles 0, 1); the pair is (i1, j0)
        cells = np.zeros(2, dtype=orc.CELL_DTYPE)
        cells["count"], cells["first"], cells["width"] = 2, [0, 2], 1.0
        tasks["ci"], tasks["cj"] = 1, 0
        side_i = _force_in_records([((0.9, 0.9, 0.9), np.float32(0.01)), ((0.0, 0.0, 0.0), hi)])
        side_j = _force_in_records([((0.0, 0.0, -r), hj), ((0.5, 0.5, 0.5), np.float32(0.01))])
        buf = np.zeros(256, dtype=np.uint8)
        buf[:104], buf[128:232] = side_i.view(np.uint8).ravel(), side_j.view(np.uint8).ravel()
        assert orc.flag_cutoff_pairs(cells, tasks, buf).tolist() == [expect, False, False, expect], (delta, h_pair)
