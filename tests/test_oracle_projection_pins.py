"""Pins of the oracle's steps 10-12 (readings P1-P3 of DESIGN.md §13): the
right-hand side div(u_f)/dt, the velocity correction and the divergence of the corrected face
velocity.  Pinned by closed forms (uniform and linear fields, walls, periodic z), telescoping
(the rhs is always compatible), and the projection identity div(u_f^{n+1}) = dt (rhs - A p) that
ties all three to the already pinned operator A -- a wrong sign, face, spacing or wall rule in any
of them breaks one of these.
"""
import numpy as np
import pytest

from paper_2104_01636_b200 import workload as wl

H = (0.1, 0.07, 0.13)


def rnd(shape, seed, stream=13):
    n = int(np.prod(shape))
    return (2.0 * wl.uniform01(seed, stream, np.arange(n, dtype=np.uint64)) - 1.0).reshape(shape)


def fields(nx, ny, nz, seed):
    return tuple(rnd((nz, ny, nx), seed + q) for q in range(3))


def test_rhs_of_uniform_flow_only_sees_the_walls(ora):
    nx, ny, nz, dt = 6, 5, 8, 0.01
    u = (np.full((nz, ny, nx), 2.0), np.full((nz, ny, nx), -3.0), np.full((nz, ny, nx), 5.0))
    rhs = ora.rhs_from_velocity(u, H, dt)
    want = np.zeros((nz, ny, nx))
    want[:, :, 0] += 2.0 / H[0] / dt          # x- wall face carries 0, x+ face carries U
    want[:, :, -1] -= 2.0 / H[0] / dt
    want[:, 0, :] += -3.0 / H[1] / dt
    want[:, -1, :] -= -3.0 / H[1] / dt        # uniform uz: periodic, no contribution
    assert np.max(np.abs(rhs - want)) <= 1e-12 * np.max(np.abs(want))


def test_rhs_of_linear_and_periodic_fields(ora):
    nx, ny, nz, dt = 8, 6, 12, 0.5
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    ux = 3.0 * (i + 0.5) * H[0]               # du/dx = 3 in the interior
    uz = np.sin(2 * np.pi * k / nz)           # central difference of a periodic mode
    zero = np.zeros_like(ux)
    rhs = ora.rhs_from_velocity((ux, zero, zero), H, dt)
    assert np.max(np.abs(rhs[:, :, 1:-1] - 3.0 / dt)) <= 1e-12 * 3.0 / dt
    rhs = ora.rhs_from_velocity((zero, zero, uz), H, dt)
    want = (np.sin(2 * np.pi * (k + 1) / nz) - np.sin(2 * np.pi * (k - 1) / nz)) / (2 * H[2]) / dt
    assert np.max(np.abs(rhs - want)) <= 1e-12 * np.max(np.abs(want))


def test_rhs_is_always_compatible(ora):
    """Wall faces carry no flux and z is periodic, so the fluxes telescope: sum(rhs) = 0 -- the
    compatibility condition of the singular Neumann/periodic problem (S6)."""
    u = fields(10, 6, 8, 3)
    rhs = ora.rhs_from_velocity(u, H, 0.01)
    assert abs(rhs.sum()) <= 1e-12 * np.abs(rhs).sum()


def test_correction_of_a_linear_pressure_in_constant_density(ora):
    nx, ny, nz, dt, rho = 8, 6, 8, 0.02, 1000.0
    coef = ora.coefficients(np.ones((nz, ny, nx)), 1000.0, 1.2, *H)
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    p = 7.0 * (i + 0.5) * H[0] - 4.0 * (j + 0.5) * H[1]
    u = [np.zeros((nz, ny, nx)) for _ in range(3)]
    ora.correct_velocity(coef, p, u, H, dt)
    assert np.max(np.abs(u[0][:, :, 1:-1] + dt * 7.0 / rho)) <= 1e-12 * dt * 7.0 / rho
    assert np.max(np.abs(u[1][:, 1:-1, :] - dt * 4.0 / rho)) <= 1e-12 * dt * 4.0 / rho
    assert np.all(u[2] == 0.0)
    # at a wall the wall face contributes nothing: half the interior correction
    assert np.max(np.abs(u[0][:, :, 0] + 0.5 * dt * 7.0 / rho)) <= 1e-12 * dt * 7.0 / rho


def test_projection_identity_ties_all_three_to_the_operator(ora):
    """div(u_f - dt (grad p/rho)_f) = dt (rhs - A p) for ANY u, p and variable density."""
    nx, ny, nz, dt = 10, 6, 8, 0.013
    coef = ora.coefficients(wl.random_fraction(nx, ny, nz, 5), 1000.0, 1.2, *H)
    u, p = fields(nx, ny, nz, 7), rnd((nz, ny, nx), 11)
    rhs = ora.rhs_from_velocity(u, H, dt)
    div = ora.face_divergence(coef, u, p, H, dt)
    want = dt * (rhs - ora.apply(coef, p))
    assert np.max(np.abs(div - want)) <= 1e-11 * np.max(np.abs(want))
    # with p = 0 it is the divergence of the uncorrected face velocity
    div0 = ora.face_divergence(coef, u, np.zeros_like(p), H, dt)
    assert np.max(np.abs(div0 - dt * rhs)) <= 1e-13 * np.max(np.abs(dt * rhs))


def test_cell_correction_is_the_mean_of_the_face_corrections(ora):
    """f->c: with uz = 0 and a z-only pressure, the cell correction equals minus dt times the mean
    of the two z-face gradients, which P3 exposes through the face divergence."""
    nx, ny, nz, dt = 4, 4, 8, 0.1
    coef = ora.coefficients(wl.random_fraction(nx, ny, nz, 9), 1000.0, 1.2, *H)
    p = np.broadcast_to(rnd((nz, 1, 1), 15), (nz, ny, nx)).copy()
    u = [np.zeros((nz, ny, nx)) for _ in range(3)]
    ora.correct_velocity(coef, p, u, H, dt)
    az = coef[2]
    gp = az * H[2] * (np.roll(p, -1, axis=0) - p)          # (grad p / rho) on the z+ face
    want = -dt * 0.5 * (np.roll(gp, 1, axis=0) + gp)
    assert np.max(np.abs(u[2] - want)) <= 1e-13 * np.max(np.abs(want))
    assert np.all(u[0] == 0.0) and np.all(u[1] == 0.0)


def test_full_projection_makes_the_face_velocity_divergence_free(ora):
    w = wl.make_custom(16, 16, 32, 1, 8, 3)
    h, dt = (w.dx, w.dy, w.dz), 1e-3
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, *h)
    u = fields(w.nx, w.ny, w.nz, 21)
    rhs = ora.rhs_from_velocity(u, h, dt)
    p = np.zeros_like(rhs)
    info = ora.mg_solve(coef, rhs, p, 200, 1e-10, levels=3, nu1=2, nu2=2, coarse_sweeps=100,
                        omega_s=1.5, nu_growth=4, nu_max=16)
    assert info.converged
    div0 = ora.face_divergence(coef, u, np.zeros_like(p), h, dt)
    div1 = ora.face_divergence(coef, u, p, h, dt)
    assert np.linalg.norm(div1) <= 2e-10 * np.linalg.norm(div0)
