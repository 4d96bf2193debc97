"""Seeded synthetic duct workloads (BASELINE.json `configs`).

This module is the *input generator only*: sphere placement, the VOF liquid fraction F
sampled on 4^3 sub-points per cell, and a zero-mean right-hand side.  It holds none of the
solver's arithmetic (no density, no coefficients, no stencil) and is the one piece of code
the CPU oracle tests and the CUDA path share: both receive the same host arrays.

The fields stand in for the paper's workload, a 192x192x768 duct with 864 spherical bubbles
of 8 cells diameter at 0.82 % void fraction and rho_l/rho_g = 1000/1.2
(§4, §4), whose own data are not available.

Layout: every field is a C-contiguous float64 array of shape (nz, ny, nx), i.e. the linear
index is n = i + nx*(j + ny*k) with x fastest (SURVEY.md §8 notation).

Random numbers: a counter-based SplitMix64 (u depends on (seed, stream, index) only), so any
cell's value can be regenerated alone.  Stream 0 = sphere placement, stream 1 = rhs noise.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 2104016360          # seed = SEED_BASE + cfg, cfg = 1..5
RHO_L = 1000.0                  # PAPER.md:220 (liquid density, kg/m^3)
RHO_G = 1.2                     # PAPER.md:220 (gas density, kg/m^3)

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_MIX1 = np.uint64(0xBF58476D1CE4E5B9)
_MIX2 = np.uint64(0x94D049BB133111EB)
_STREAM = 0xD1B54A32D192ED03
_MASK = (1 << 64) - 1


def splitmix64(seed: int, stream: int, index) -> np.ndarray:
    """64-bit output number `index` (0-based) of SplitMix64 started at seed ^ (stream*c)."""
    state = np.uint64((seed ^ ((stream * _STREAM) & _MASK)) & _MASK)
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = state + (idx + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _MIX1
        z = (z ^ (z >> np.uint64(27))) * _MIX2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, stream: int, index) -> np.ndarray:
    """u in [0,1): top 53 bits of splitmix64 times 2^-53 (exact in fp64)."""
    return (splitmix64(seed, stream, index) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _mean(a: np.ndarray) -> float:
    """Mean by chunked math.fsum (correctly rounded partial sums; deterministic)."""
    flat = a.reshape(-1)
    parts = [math.fsum(flat[s:s + (1 << 20)].tolist()) for s in range(0, flat.size, 1 << 20)]
    return math.fsum(parts) / flat.size


# ----------------------------------------------------------------------------- spheres
def place_spheres(nx: int, ny: int, nz: int, count: int, diameter: int, seed: int,
                  gap: int = 2, wall: int = 2) -> np.ndarray:
    """Random sequential rejection of `count` equal spheres.

    Centres lie on the integer cell-corner lattice; cx, cy in [R+wall, n-R-wall], cz in
    [0, nz-1].  A candidate is accepted iff its distance to every accepted centre is at
    least diameter+gap, the z distance taken periodically.  Returns int64 (count, 3) as
    (cx, cy, cz).
    """
    if diameter % 2:
        raise ValueError("diameter must be even (centres sit on cell corners)")
    R = diameter // 2
    lo, hix, hiy = R + wall, nx - R - wall, ny - R - wall
    if hix < lo or hiy < lo:
        raise ValueError("duct too narrow for the requested spheres")
    centres = np.zeros((count, 3), dtype=np.int64)
    n_acc, attempt, dmin2 = 0, 0, (diameter + gap) ** 2
    max_attempts = 1000 * max(count, 1)
    while n_acc < count:
        if attempt >= max_attempts:
            raise RuntimeError("sphere placement did not finish (too dense)")
        u = uniform01(seed, 0, np.arange(3 * attempt, 3 * attempt + 3, dtype=np.uint64))
        attempt += 1
        c = np.array([lo + int(u[0] * (hix - lo + 1)),
                      lo + int(u[1] * (hiy - lo + 1)),
                      int(u[2] * nz)], dtype=np.int64)
        if n_acc:
            d = np.abs(centres[:n_acc] - c)
            d[:, 2] = np.minimum(d[:, 2], nz - d[:, 2])
            if int((d * d).sum(axis=1).min()) < dmin2:
                continue
        centres[n_acc] = c
        n_acc += 1
    return centres


def regular_array(nx: int, ny: int, nz: int, mx: int, my: int, mz: int) -> np.ndarray:
    """The paper's initial layout: a regular mx x my x mz array (6x6x24)."""
    cx = [(2 * a + 1) * nx // (2 * mx) for a in range(mx)]
    cy = [(2 * b + 1) * ny // (2 * my) for b in range(my)]
    cz = [(2 * c + 1) * nz // (2 * mz) for c in range(mz)]
    return np.array([(x, y, z) for z in cz for y in cy for x in cx], dtype=np.int64)


def sphere_stencil(diameter: int, sub: int = 4) -> np.ndarray:
    """Number of the sub^3 sample points of each cell of the bounding box that lie inside.

    In units of 1/(2*sub) cell the sample points of cell offset o (o = i - cx in [-R, R-1])
    sit at 2*sub*o + 2a + 1, a = 0..sub-1; inside iff the squared distance is < (2*sub*R)^2.
    Pure integer arithmetic; ties cannot occur.  Shape (2R, 2R, 2R), z first.
    """
    R = diameter // 2
    o = np.arange(-R, R, dtype=np.int64)
    a = np.arange(sub, dtype=np.int64)
    coord = (2 * sub * o[:, None] + 2 * a[None, :] + 1).reshape(-1)      # (2R*sub,)
    sq = coord * coord
    inside = (sq[:, None, None] + sq[None, :, None] + sq[None, None, :]) < (2 * sub * R) ** 2
    n = 2 * R
    return inside.reshape(n, sub, n, sub, n, sub).sum(axis=(1, 3, 5)).astype(np.int64)


def liquid_fraction(nx: int, ny: int, nz: int, centres: np.ndarray, diameter: int,
                    sub: int = 4) -> np.ndarray:
    """F = 1 - (sample points inside a sphere)/sub^3 per cell; z wraps periodically."""
    cnt = np.zeros((nz, ny, nx), dtype=np.int64)
    if len(centres):
        R = diameter // 2
        st = sphere_stencil(diameter, sub)
        for cx, cy, cz in np.asarray(centres, dtype=np.int64):
            if cx - R < 0 or cx + R > nx or cy - R < 0 or cy + R > ny:
                raise ValueError("sphere crosses a duct wall")
            kz = (np.arange(cz - R, cz + R) % nz)
            cnt[kz[:, None, None], np.arange(cy - R, cy + R)[None, :, None],
                np.arange(cx - R, cx + R)[None, None, :]] += st
    if cnt.max(initial=0) > sub ** 3:
        raise ValueError("overlapping spheres")
    return 1.0 - cnt.astype(np.float64) / float(sub ** 3)


# ----------------------------------------------------------------------------- rhs
def noise_rhs(nx: int, ny: int, nz: int, seed: int, amplitude: float = 1.0) -> np.ndarray:
    """amplitude * (2u - 1), u = uniform01(seed, stream 1, n); not yet mean-free."""
    out = np.empty((nz, ny, nx), dtype=np.float64)
    plane = nx * ny
    step = max(1, (1 << 22) // plane)
    for k0 in range(0, nz, step):
        k1 = min(nz, k0 + step)
        idx = np.arange(k0 * plane, k1 * plane, dtype=np.uint64)
        out[k0:k1] = (amplitude * (2.0 * uniform01(seed, 1, idx) - 1.0)).reshape(k1 - k0, ny, nx)
    return out


def eigenmode(nx: int, ny: int, nz: int, kx: int, ky: int, kz: int) -> np.ndarray:
    """cos(pi kx (i+1/2)/nx) cos(pi ky (j+1/2)/ny) cos(2 pi kz k/nz)."""
    i = np.arange(nx, dtype=np.float64)
    j = np.arange(ny, dtype=np.float64)
    k = np.arange(nz, dtype=np.float64)
    vx = np.cos(math.pi * kx * (i + 0.5) / nx)
    vy = np.cos(math.pi * ky * (j + 0.5) / ny)
    vz = np.cos(2.0 * math.pi * kz * k / nz)
    return vz[:, None, None] * vy[None, :, None] * vx[None, None, :]


def remove_mean(a: np.ndarray) -> np.ndarray:
    """Compatibility of the pure Neumann/periodic problem needs sum(rhs) = 0."""
    return a - _mean(a)


# ----------------------------------------------------------------------------- configs
@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    rho_l: float
    rho_g: float
    omega: float
    max_sweeps: int            # fixed-sweep run of the config (0 = to tolerance only)
    tol: float                 # relative residual target (0 = fixed sweeps only)
    seed: int
    diameter: int
    centres: np.ndarray
    F: np.ndarray = field(repr=False)
    rhs: np.ndarray = field(repr=False)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz


# cfg: (nx, ny, nz, spheres, diameter, omega, fixed sweeps, tol)   -- BASELINE.json configs[0..4]
CONFIGS = {
    1: ("tiny_duct_32x32x64", 32, 32, 64, 1, 8, 1.5, 200, 0.0),
    2: ("unladen_duct_64x64x128", 64, 64, 128, 0, 0, 1.7, 0, 1e-8),
    3: ("bubbly_duct_128x128x256", 128, 128, 256, 108, 12, 1.6, 0, 1e-8),
    4: ("paper_scale_duct_256x256x512", 256, 256, 512, 864, 16, 1.6, 500, 1e-8),
    5: ("large_duct_384x384x1024", 384, 384, 1024, 2048, 16, 1.6, 300, 0.0),
}


def make_config(cfg: int, seed_offset: int = 0) -> Workload:
    """Build BASELINE.json config `cfg` (1..5).  `seed_offset` varies the seed per replica."""
    name, nx, ny, nz, count, diam, omega, sweeps, tol = CONFIGS[cfg]
    seed = SEED_BASE + cfg + seed_offset
    h = 1.0 / nx                                   # duct width 1
    if cfg == 1:
        centres = np.array([[16, 16, 32]], dtype=np.int64)
    elif count:
        centres = place_spheres(nx, ny, nz, count, diam, seed)
    else:
        centres = np.zeros((0, 3), dtype=np.int64)
    F = liquid_fraction(nx, ny, nz, centres, diam)
    if cfg == 2:
        rhs0 = eigenmode(nx, ny, nz, 1, 2, 3) + noise_rhs(nx, ny, nz, seed, 1e-3)
    else:
        rhs0 = noise_rhs(nx, ny, nz, seed)
    return Workload(name, nx, ny, nz, h, h, h, RHO_L, RHO_G, omega, sweeps, tol, seed, diam,
                    centres, F, remove_mean(rhs0))


def make_custom(nx: int, ny: int, nz: int, count: int, diameter: int, seed: int,
                omega: float = 1.6, dx: float | None = None, dy: float | None = None,
                dz: float | None = None, rho_l: float = RHO_L, rho_g: float = RHO_G) -> Workload:
    """Same recipe on an arbitrary grid (parity cases with ragged tiles, anisotropic h)."""
    centres = (place_spheres(nx, ny, nz, count, diameter, seed) if count
               else np.zeros((0, 3), dtype=np.int64))
    F = liquid_fraction(nx, ny, nz, centres, diameter)
    rhs = remove_mean(noise_rhs(nx, ny, nz, seed))
    h = 1.0 / nx
    return Workload(f"custom_{nx}x{ny}x{nz}", nx, ny, nz, dx or h, dy or h, dz or h, rho_l, rho_g,
                    omega, 0, 0.0, seed, diameter, centres, F, rhs)


def random_fraction(nx: int, ny: int, nz: int, seed: int, sub: int = 4) -> np.ndarray:
    """F drawn per cell from {m/sub^3}: the hardest coefficient field (no smooth regions)."""
    idx = np.arange(nx * ny * nz, dtype=np.uint64)
    m = (uniform01(seed, 2, idx) * (sub ** 3 + 1)).astype(np.int64)
    return (m.astype(np.float64) / float(sub ** 3)).reshape(nz, ny, nx)


# ----------------------------------------------------------------------------- SSF inputs
SIGMA = 0.072                   # surface tension of air-water, N/m (PAPER.md:220 fluid pair)


def curvature_field(nx: int, ny: int, nz: int, centres: np.ndarray, diameter: int,
                    h: float) -> np.ndarray:
    """Exact interface curvature kappa = 2/R of every sphere (R = diameter/2 cells of size h),
    stored in all cells of the sphere's bounding box grown by one cell (z wrapped); 0 elsewhere.
    This is the "exact analytical curvature" case of PAPER.md:78; the height-function estimate of
    step 5 is out of scope.  Input generator only: no solver arithmetic."""
    kappa = np.zeros((nz, ny, nx), dtype=np.float64)
    if len(centres):
        R = diameter // 2
        val = 2.0 / (R * h)
        for cx, cy, cz in np.asarray(centres, dtype=np.int64):
            kz = (np.arange(cz - R - 1, cz + R + 1) % nz)
            ys = np.arange(max(cy - R - 1, 0), min(cy + R + 1, ny))
            xs = np.arange(max(cx - R - 1, 0), min(cx + R + 1, nx))
            kappa[kz[:, None, None], ys[None, :, None], xs[None, None, :]] = val
    return kappa
