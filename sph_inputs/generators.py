"""Counter-based seeded particle generators for BASELINE.json:configs[0..4].

PRNG: SplitMix64 evaluated as a pure function of (seed, stream, index), so any
element can be drawn independently and every array is reproducible on any box.
uniform = (u64 >> 11) * 2^-53, normal by Box-Muller on two streams.

Every function returns particles in GENERATOR order (not sorted by cell): the
cell builders of the oracle and of the library each sort them.  `id` is the
generator index, `time_bin` is 1, all loop outputs are 0.

Nothing here is part of the method (no packing, no SPH sums, no cells/tasks).
"""
import numpy as np

from .format import PART_DTYPE

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """n raw 64-bit draws: element i is mix(state0 + (start+i+1)*golden)."""
    with np.errstate(over="ignore"):
        state0 = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) ^ (np.uint64(stream) * _GOLDEN)
        idx = np.arange(start + 1, start + n + 1, dtype=np.uint64)
        z = state0 + idx * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """n doubles in [0, 1)."""
    return (splitmix64(seed, stream, n, start) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def normal01(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """n standard normals (Box-Muller on streams 2*stream+1000, 2*stream+1001)."""
    u1 = uniform01(seed, 2 * stream + 1000, n, start)
    u2 = uniform01(seed, 2 * stream + 1001, n, start)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


def _finish(parts: np.ndarray) -> np.ndarray:
    n = parts.shape[0]
    parts["id"] = np.arange(n, dtype=np.int64)
    parts["time_bin"] = 1
    return parts


def config0(seed: int = 1) -> np.ndarray:
    """configs[0]: 4,096 particles, exactly 64 uniform points in each of 4^3 cells.

    m = 1/N, h = 1.2348 N^(-1/3), v = 0, u = 1.  Particle p sits in cell p % 64
    so that generator order is NOT cell order.
    """
    n, cpd = 4096, 4
    parts = np.zeros(n, dtype=PART_DTYPE)
    p = np.arange(n)
    cell = p % 64
    cxyz = np.stack([cell // 16, (cell // 4) % 4, cell % 4], axis=1).astype(np.float64)
    u = np.stack([uniform01(seed, d, n) for d in range(3)], axis=1)
    parts["x"] = (cxyz + u) / cpd
    parts["mass"] = np.float32(1.0 / n)
    parts["h"] = np.float32(1.2348 * n ** (-1.0 / 3.0))
    parts["u"] = 1.0
    return _finish(parts)


def jittered_lattice(n_side: int, seed: int, jitter: float = 0.2, eta: float = 1.2348,
                     sigma_v: float = 0.1, h_spread: float = 0.0, mass_spread: float = 0.0,
                     u_spread: float = 0.0) -> np.ndarray:
    """n_side^3 lattice points plus uniform jitter of +-jitter/2 spacings, unit periodic box.

    h = eta*dx*(1 + h_spread*(U-0.5)), m = (1/N)*(1 + mass_spread*(U-0.5)),
    u = 1 + u_spread*(U-0.5), v ~ N(0, sigma_v) per component.
    With the defaults and n_side=64 this is BASELINE.json:configs[1].
    """
    n = n_side ** 3
    parts = np.zeros(n, dtype=PART_DTYPE)
    p = np.arange(n)
    ijk = np.stack([p // (n_side * n_side), (p // n_side) % n_side, p % n_side], axis=1).astype(np.float64)
    u = np.stack([uniform01(seed, d, n) for d in range(3)], axis=1)
    parts["x"] = (ijk + 0.5 + jitter * (u - 0.5)) / n_side
    parts["v"] = np.stack([sigma_v * normal01(seed, 10 + d, n) for d in range(3)], axis=1).astype(np.float32)
    parts["mass"] = ((1.0 / n) * (1.0 + mass_spread * (uniform01(seed, 20, n) - 0.5))).astype(np.float32)
    parts["h"] = ((eta / n_side) * (1.0 + h_spread * (uniform01(seed, 21, n) - 0.5))).astype(np.float32)
    parts["u"] = (1.0 + u_spread * (uniform01(seed, 22, n) - 0.5)).astype(np.float32)
    return _finish(parts)


def config1(seed: int = 1) -> np.ndarray:
    """configs[1]: 262,144 particles, 64^3 glass-like lattice, v ~ N(0, 0.1), u = 1."""
    return jittered_lattice(64, seed)


def config2_positions(seed: int = 1, n_yz: int = 128, n_left: int = 102, n_right: int = 26,
                      jitter: float = 0.05) -> np.ndarray:
    """configs[2] before the h iteration: Sod-like two-density lattice.

    n_yz x n_yz lattice in (y, z); n_left x-planes equally spaced in [0, 0.5),
    n_right in [0.5, 1) (102 + 26 = 128 planes keeps N = 2^21 exactly; ratio 3.92,
    DESIGN.md reading C18).  Equal masses 1/N, v ~ N(0, 0.01).  `h` holds the
    continuum first guess 1.12725 n^(-1/3) from the local number density; the
    48-neighbour iteration, rho and u (P = 1 | 0.1) are set by the caller.
    """
    n_planes = n_left + n_right
    n = n_planes * n_yz * n_yz
    parts = np.zeros(n, dtype=PART_DTYPE)
    p = np.arange(n)
    ip = p // (n_yz * n_yz)
    jy = (p // n_yz) % n_yz
    kz = p % n_yz
    left = ip < n_left
    dx_l, dx_r, dyz = 0.5 / n_left, 0.5 / n_right, 1.0 / n_yz
    u = np.stack([uniform01(seed, d, n) for d in range(3)], axis=1)
    x = np.where(left, (ip + 0.5 + jitter * (u[:, 0] - 0.5)) * dx_l,
                 0.5 + (ip - n_left + 0.5 + jitter * (u[:, 0] - 0.5)) * dx_r)
    parts["x"][:, 0] = x
    parts["x"][:, 1] = (jy + 0.5 + jitter * (u[:, 1] - 0.5)) * dyz
    parts["x"][:, 2] = (kz + 0.5 + jitter * (u[:, 2] - 0.5)) * dyz
    parts["v"] = np.stack([0.01 * normal01(seed, 10 + d, n) for d in range(3)], axis=1).astype(np.float32)
    parts["mass"] = np.float32(1.0 / n)
    dens = np.where(left, 1.0 / (dx_l * dyz * dyz), 1.0 / (dx_r * dyz * dyz))
    parts["h"] = (1.12725 * dens ** (-1.0 / 3.0)).astype(np.float32)
    parts["u"] = 1.0
    return _finish(parts)


def _min_image(d: np.ndarray) -> np.ndarray:
    return d - np.round(d)


def mixture_density(x: np.ndarray, centres: np.ndarray, n_total: int, frac_clumps: float,
                    sigma: float, chunk: int = 1 << 18) -> np.ndarray:
    """Analytic number density of the uniform + Gaussian-clump mixture (nearest image).

    A clump's term is dropped beyond 6.25 sigma (exp(-19.5) = 3e-9 of its peak): the points are binned on a
    coarse periodic grid once and every clump visits only the bins within reach, which is what makes the
    2^26-particle workload generate in seconds instead of minutes.
    """
    n_c = centres.shape[0]
    norm = (2.0 * np.pi) ** -1.5 / sigma ** 3
    reach = 6.25 * sigma
    nb = max(1, min(32, int(np.floor(1.0 / reach))))            # bins per dimension, bin width >= reach
    acc = np.zeros(x.shape[0])
    if nb < 3 or x.shape[0] < (1 << 16):                         # small problem or wide clumps: every clump sees every point
        for s in range(0, x.shape[0], chunk):
            xs = x[s:s + chunk]
            a = np.zeros(xs.shape[0])
            for c in range(n_c):
                d = _min_image(xs - centres[c])
                r2 = np.einsum("ij,ij->i", d, d)
                a += np.where(r2 < reach * reach, np.exp(-0.5 * r2 / sigma ** 2), 0.0)
            acc[s:s + chunk] = a
    else:
        b = np.minimum((x * nb).astype(np.int64), nb - 1)
        key = (b[:, 0] * nb + b[:, 1]) * nb + b[:, 2]
        order = np.argsort(key, kind="stable")
        start = np.searchsorted(key[order], np.arange(nb ** 3 + 1))
        xo = x[order]
        ao = np.zeros(x.shape[0])
        for c in range(n_c):
            cb = np.minimum((centres[c] * nb).astype(np.int64), nb - 1)
            for da in (-1, 0, 1):
                for db in (-1, 0, 1):
                    k0 = (((cb[0] + da) % nb) * nb + (cb[1] + db) % nb) * nb
                    for dc in (-1, 0, 1):
                        k = k0 + (cb[2] + dc) % nb
                        lo, hi = start[k], start[k + 1]
                        if hi > lo:
                            d = _min_image(xo[lo:hi] - centres[c])
                            r2 = np.einsum("ij,ij->i", d, d)
                            ao[lo:hi] += np.where(r2 < reach * reach, np.exp(-0.5 * r2 / sigma ** 2), 0.0)
        acc[order] = ao
    return n_total * ((1.0 - frac_clumps) + frac_clumps / n_c * norm * acc)


def clumpy_mixture(n: int, seed: int, n_clumps: int = 64, frac_clumps: float = 0.7,
                   sigma: float = 0.02, h_cap: float = 1.0 / 64.0) -> np.ndarray:
    """Gaussian clumps over a uniform background (Eagle25-like occupancy spread).

    Each clump holds floor(frac_clumps*n/n_clumps) points ~ N(centre, sigma^2) wrapped
    into the unit box, the rest is uniform.  h = 1.12725 n(x)^(-1/3) from the analytic
    mixture density, clipped to h_cap.  m = 1/N, v ~ N(0, 0.1), u = 1.
    """
    parts = np.zeros(n, dtype=PART_DTYPE)
    centres = np.stack([uniform01(seed, 100 + d, n_clumps) for d in range(3)], axis=1)
    per = int(frac_clumps * n / n_clumps)
    n_cl = per * n_clumps
    x = np.empty((n, 3))
    for d in range(3):
        g = normal01(seed, 30 + d, n_cl)
        x[:n_cl, d] = np.repeat(centres[:, d], per) + sigma * g
        x[n_cl:, d] = uniform01(seed, d, n - n_cl)
    x -= np.floor(x)
    x[x >= 1.0] = 0.0
    # interleave clump and background particles so generator order is not spatial
    perm = np.argsort(splitmix64(seed, 200, n), kind="stable")
    x = x[perm]
    parts["x"] = x
    dens = mixture_density(x, centres, n, frac_clumps if n_cl else 0.0, sigma)
    parts["h"] = np.minimum(1.12725 * dens ** (-1.0 / 3.0), h_cap).astype(np.float32)
    parts["v"] = np.stack([0.1 * normal01(seed, 10 + d, n) for d in range(3)], axis=1).astype(np.float32)
    parts["mass"] = np.float32(1.0 / n)
    parts["u"] = 1.0
    return _finish(parts)


def config3(seed: int = 1, n: int = 1 << 24) -> np.ndarray:
    """configs[3]: 64 Gaussian clumps (sigma 0.02) over a 30 % uniform background."""
    return clumpy_mixture(n, seed, n_clumps=64, frac_clumps=0.7, sigma=0.02)


def config4(seed: int = 1, n: int = 1 << 26) -> np.ndarray:
    """configs[4]: uniform-plus-clumps mix, 50 % uniform + 50 % in 256 clumps (reading)."""
    return clumpy_mixture(n, seed, n_clumps=256, frac_clumps=0.5, sigma=0.02)


def eagle_like_counts(seed: int, n_cells: int, n_min: int = 5, n_max: int = 125113,
                      median: float = 109.0, mean: float = 184.0) -> np.ndarray:
    """Per-cell occupancies with the spread the paper reports for Eagle25 (per-cell min 5,
    max 125,113, mean 184, median 109): a lognormal body with that median and mean (sigma^2 = 2 ln(mean / median)),
    clipped below at n_min, plus a short geometric tail -- n_max, n_max / 2, n_max / 4, ... down to ten times the
    median -- placed in seeded cells (the outliers a lognormal of that width does not produce: dense galaxy cores).
    """
    sigma = np.sqrt(2.0 * np.log(mean / median))
    z = normal01(seed, 40, n_cells)
    counts = np.maximum(np.floor(median * np.exp(sigma * z)), n_min).astype(np.int64)
    counts[0] = n_min                                  # the stated minimum is present whatever the draw
    tail = []
    c = float(n_max)
    while c > 10.0 * median and len(tail) < max(1, n_cells // 8):
        tail.append(int(c))
        c *= 0.5
    where = np.argsort(splitmix64(seed, 41, n_cells), kind="stable")[: len(tail)]
    where = where[where != 0][: len(tail)]
    counts[where] = np.array(tail[: where.shape[0]], dtype=np.int64)
    return counts


def eagle_like(seed: int = 1, cells_per_dim: int = 16, n_max: int = 125113, n_min: int = 5,
               median: float = 109.0, mean: float = 184.0) -> np.ndarray:
    """Extreme-occupancy workload (stand-in for Eagle25's cell statistics).

    A periodic grid of cells_per_dim^3 equal cells whose occupancies are drawn by `eagle_like_counts`; a cell's
    particles are uniform inside it.  h = 1.12725 (volume / count)^(1/3) of the own cell (48-neighbour continuum
    value), clipped to 0.4999 of the cell width -- what a cell with a handful of particles gets in a tree code
    whose leaves cannot grow.  m = 1/N, v ~ N(0, 0.1), u = 1.  Generator order is a seeded shuffle, not cell order.
    """
    n_cells = cells_per_dim ** 3
    counts = eagle_like_counts(seed, n_cells, n_min, n_max, median, mean)
    n = int(counts.sum())
    cell = np.repeat(np.arange(n_cells, dtype=np.int64), counts)
    perm = np.argsort(splitmix64(seed, 200, n), kind="stable")
    cell = cell[perm]
    cxyz = np.stack([cell // (cells_per_dim * cells_per_dim), (cell // cells_per_dim) % cells_per_dim, cell % cells_per_dim], axis=1).astype(np.float64)
    u = np.stack([uniform01(seed, d, n) for d in range(3)], axis=1)
    parts = np.zeros(n, dtype=PART_DTYPE)
    parts["x"] = np.minimum((cxyz + u) / cells_per_dim, np.nextafter(1.0, 0.0))
    width = 1.0 / cells_per_dim
    parts["h"] = np.minimum(1.12725 * width * counts[cell].astype(np.float64) ** (-1.0 / 3.0), 0.4999 * width).astype(np.float32)
    parts["v"] = np.stack([0.1 * normal01(seed, 10 + d, n) for d in range(3)], axis=1).astype(np.float32)
    parts["mass"] = np.float32(1.0 / n)
    parts["u"] = 1.0
    return _finish(parts)


def synthetic_trace(n_tasks, n_self, seed, steps=5, bundle_lo=128, bundle_hi=1024):
    """A seeded stand-in for a recorded trace of offload actions: per simulation step the self tasks, then
    the pair tasks, are cut into bundles of seeded sizes; every bundle is packed and later unpacked, density before force.
    -> list of (step, loop, action, first task, task count)"""
    rng = np.random.default_rng(seed)
    trace = []
    for st in range(steps):
        cuts = []
        for lo, hi in ((0, n_self), (n_self, n_tasks)):
            t = lo
            while t < hi:
                m = int(min(hi - t, rng.integers(bundle_lo, bundle_hi + 1)))
                cuts.append((t, m))
                t += m
        for loop in ("density", "force"):
            for t0, m in cuts:
                trace.append((st, loop, "pack", t0, m))
                trace.append((st, loop, "unpack", t0, m))
    return trace
