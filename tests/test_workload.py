"""The seeded input generator (pin P12)."""
import json
import math
import os

import numpy as np
import pytest

from paper_2104_01636_b200 import workload as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_rng_is_counter_based_and_uniform():
    idx = np.arange(100000, dtype=np.uint64)
    u = wl.uniform01(123, 1, idx)
    assert u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 5e-3 and abs(u.var() - 1.0 / 12.0) < 2e-3
    assert wl.uniform01(123, 1, np.uint64(4711)) == u[4711]           # value depends on n only
    assert not np.array_equal(u, wl.uniform01(123, 2, idx))           # streams differ
    assert not np.array_equal(u, wl.uniform01(124, 1, idx))           # seeds differ
    # reference SplitMix64 (Steele, Lea, Flood 2014) written with Python integers
    s, M = 123 ^ ((1 * 0xD1B54A32D192ED03) & (2 ** 64 - 1)), 2 ** 64 - 1
    for n in (0, 1, 99999):
        z = (s + (n + 1) * 0x9E3779B97F4A7C15) & M
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
        z ^= z >> 31
        assert int(wl.splitmix64(123, 1, np.uint64(n))) == z


def brute_force_inside_count(R, sub=4):
    """Sample points of one sphere of radius R cells centred on a cell corner, counted one by one."""
    total = 0
    for i in range(-R, R):
        for j in range(-R, R):
            for k in range(-R, R):
                for a in range(sub):
                    for b in range(sub):
                        for c in range(sub):
                            x = i + (2 * a + 1) / (2.0 * sub)
                            y = j + (2 * b + 1) / (2.0 * sub)
                            z = k + (2 * c + 1) / (2.0 * sub)
                            total += (x * x + y * y + z * z) < R * R
    return total


def test_sphere_stencil_against_brute_force_and_volume():
    st = wl.sphere_stencil(8)
    assert st.shape == (8, 8, 8) and st.min() == 0 and st.max() == 64
    assert int(st.sum()) == brute_force_inside_count(4)
    vol = st.sum() / 64.0
    assert vol == 269.625                                   # SURVEY.md §8.d probe value for R = 4
    assert abs(vol - 4.0 / 3.0 * math.pi * 4 ** 3) < 0.01 * vol
    # mirror symmetry in every axis and under axis permutation
    assert np.array_equal(st, st[::-1]) and np.array_equal(st, st[:, ::-1])
    assert np.array_equal(st, st.transpose(2, 1, 0))


def test_paper_layout_reproduces_printed_void_fraction():
    """864 bubbles of 8 cells in a regular 6x6x24 array on 192x192x768 give
    a void fraction of 'approximately 0.82 %'.  One periodic unit cell of that array is
    32x32x32 with one bubble; and the full layout is checked for count and spacing."""
    with open(os.path.join(GOLDEN, "paper_constants.json")) as f:
        g = json.load(f)
    nx, ny, nz = g["grid"]
    c = wl.regular_array(nx, ny, nz, *g["array"])
    assert len(c) == g["bubbles"] and len({tuple(r) for r in c}) == g["bubbles"]
    F = wl.liquid_fraction(32, 32, 32, np.array([[16, 16, 16]]), g["diameter_cells"])
    void = 100.0 * (1.0 - F).sum() / F.size
    assert round(void, 2) == g["void_fraction_percent"]
    d = np.diff(np.unique(c[:, 0]))
    assert np.all(d == nx // g["array"][0])


@pytest.mark.parametrize("cfg", [1, 3])
def test_config_fields(cfg):
    w = wl.make_config(cfg)
    name, nx, ny, nz, count, diam, omega, sweeps, tol = wl.CONFIGS[cfg]
    assert w.F.shape == w.rhs.shape == (nz, ny, nx) and w.F.dtype == np.float64
    assert w.F.flags["C_CONTIGUOUS"] and w.rhs.flags["C_CONTIGUOUS"]
    assert np.array_equal(w.F * 64, np.round(w.F * 64)) and w.F.min() >= 0 and w.F.max() == 1
    gas = (1.0 - w.F).sum()
    assert gas == count * wl.sphere_stencil(diam).sum() / 64.0        # no overlap, nothing clipped
    assert abs(gas - count * 4.0 / 3.0 * math.pi * (diam / 2) ** 3) < 0.01 * gas
    assert abs(math.fsum(w.rhs.reshape(-1))) < 1e-9 and np.abs(w.rhs).max() <= 1.0 + 1e-2
    assert w.dx == w.dy == w.dz == 1.0 / nx
    R = diam // 2
    c = w.centres
    assert len(c) == count
    assert c[:, 0].min() >= R + 2 and c[:, 0].max() <= nx - R - 2     # >= 2 cells from the walls
    assert c[:, 1].min() >= R + 2 and c[:, 1].max() <= ny - R - 2
    for a in range(len(c)):                                           # gaps >= 2 cells, periodic z
        d = np.abs(c[a + 1:] - c[a])
        d[:, 2] = np.minimum(d[:, 2], nz - d[:, 2])
        if len(d):
            assert (d * d).sum(axis=1).min() >= (diam + 2) ** 2


def test_config1_is_the_stated_sphere():
    w = wl.make_config(1)
    assert w.centres.tolist() == [[16, 16, 32]] and w.diameter == 8 and w.omega == 1.5
    assert w.max_sweeps == 200
    assert w.F[32, 16, 16] == 0.0 and w.F[31, 15, 15] == 0.0 and w.F[0, 0, 0] == 1.0
    assert w.F[32, 16, 11] == 1.0 and w.F[32, 16, 12] < 1.0           # radius 4 from x = 16


def test_config2_rhs_is_the_eigenmode_plus_noise():
    w = wl.make_config(2)
    assert w.F.min() == 1.0
    mode = wl.eigenmode(64, 64, 128, 1, 2, 3)
    assert np.abs(w.rhs - mode).max() <= 1e-3 + 1e-5        # noise + the removed mean
    assert abs(w.rhs.mean()) < 1e-17 + 1e-16


def test_seeds_reproduce_and_replicas_differ():
    a, b = wl.make_config(1), wl.make_config(1)
    assert np.array_equal(a.rhs, b.rhs) and np.array_equal(a.F, b.F)
    c = wl.make_config(1, seed_offset=1000)
    assert not np.array_equal(a.rhs, c.rhs)


def test_periodic_wrap_of_spheres_in_z():
    F = wl.liquid_fraction(16, 16, 8, np.array([[8, 8, 0]]), 6)
    assert F[0, 8, 8] == 0.0 and F[7, 8, 8] == 0.0                    # both sides of the seam
    assert (1.0 - F).sum() == wl.sphere_stencil(6).sum() / 64.0
    with pytest.raises(ValueError):
        wl.liquid_fraction(16, 16, 8, np.array([[2, 8, 0]]), 6)       # would cross a wall
