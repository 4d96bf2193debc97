"""Parity of the CUDA kernels of steps 10-12 against the oracle's P1-P3,
element by element on the same seeded inputs.  Same expressions, same order, --fmad=false /
-ffp-contract=off: the expectation is zero differing doubles.
"""
import numpy as np
import pytest

from paper_2104_01636_b200 import workload as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2104_01636_b200 import binding, build
    build.build()
    binding.load()
    return binding


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rnd(shape, seed, stream=17):
    n = int(np.prod(shape))
    return (2.0 * wl.uniform01(seed, stream, np.arange(n, dtype=np.uint64)) - 1.0).reshape(shape)


def same(got, want, what):
    nbad = int(np.count_nonzero(got != want))
    scale = np.max(np.abs(want)) or 1.0
    assert nbad == 0, f"{what}: {nbad} doubles differ (max-rel {np.max(np.abs(got - want)) / scale:.3e})"


SHAPES = [(16, 12, 20, (0.1, 0.07, 0.13)), (1, 1, 8, None), (5, 7, 6, None), (2, 3, 2, None),
          (72, 52, 34, (1 / 72, 1 / 60, 1 / 50)), (132, 20, 10, None),
          # boundary shapes of the z-marching tiles (64 cells x 8 rows, z chunks of >= 4 planes)
          (64, 1, 8, None), (66, 2, 4, None), (2, 1, 2, None), (130, 9, 6, None), (256, 3, 2, None),
          (62, 15, 4, None), (64, 8, 40, None), (4, 5, 256, None)]


@pytest.mark.parametrize("shape", SHAPES)
def test_rhs_correction_and_face_divergence_bitwise(torch_cuda, B, ora, shape):
    nx, ny, nz, h = shape
    kw = dict(dx=h[0], dy=h[1], dz=h[2]) if h else {}
    w = wl.make_custom(nx, ny, nz, 0, 0, 3, **kw)
    w.F = wl.random_fraction(nx, ny, nz, 3)
    hh, dt = (w.dx, w.dy, w.dz), 0.0137
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, *hh)
    u = [rnd((nz, ny, nx), 5 + q) for q in range(3)]
    p = rnd((nz, ny, nx), 9)
    with B.PoissonSolver(nx, ny, nz, *hh) as s:
        u_d = [dev(torch_cuda, a) for a in u]
        p_d = dev(torch_cuda, p)
        same(s.rhs_from_velocity(*u_d, dt).cpu().numpy(), ora.rhs_from_velocity(u, hh, dt), "rhs")
        with pytest.raises(B.PsError):                      # needs coefficients
            s.correct_velocity(p_d, dt, *u_d)
        with pytest.raises(B.PsError):
            s.rhs_from_velocity(*u_d, 0.0)
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        same(s.face_divergence(*u_d, p_d, dt).cpu().numpy(),
             ora.face_divergence(coef, u, p, hh, dt), "face divergence")
        s.correct_velocity(p_d, dt, *u_d)
        v = [a.copy() for a in u]
        ora.correct_velocity(coef, p, v, hh, dt)
        for name, g, want in zip("xyz", u_d, v):
            same(g.cpu().numpy(), want, f"corrected u{name}")


def test_projection_step_on_a_bubbly_duct(torch_cuda, B, ora):
    """Steps 10-12 end to end on the GPU (config-1-shaped duct): rhs from a random u^, multigrid
    solve, correction; the corrected face velocity is divergence free to the solver tolerance,
    and the rhs and the correction are bitwise the oracle's for the GPU's p."""
    w = wl.make_config(1)
    hh, dt = (w.dx, w.dy, w.dz), 1e-3
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, *hh)
    u = [rnd(w.rhs.shape, 31 + q) for q in range(3)]
    with B.PoissonSolver(w.nx, w.ny, w.nz, *hh) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        u_d = [dev(torch_cuda, a) for a in u]
        rhs_d = s.rhs_from_velocity(*u_d, dt)
        rhs = ora.rhs_from_velocity(u, hh, dt)
        same(rhs_d.cpu().numpy(), rhs, "rhs")
        assert abs(rhs.sum()) <= 1e-12 * np.abs(rhs).sum()          # compatible by construction
        s.mg_setup()
        p_d = torch_cuda.zeros_like(rhs_d)
        info = s.mg_solve(rhs_d, p_d, 300, 1e-9)
        assert info.converged
        div0 = s.face_divergence(*u_d, torch_cuda.zeros_like(p_d), dt).cpu().numpy()
        div1 = s.face_divergence(*u_d, p_d, dt).cpu().numpy()
        assert np.linalg.norm(div1) <= 2e-9 * np.linalg.norm(div0)
        p = p_d.cpu().numpy()
        same(div1, ora.face_divergence(coef, u, p, hh, dt), "face divergence at the solution")
        s.correct_velocity(p_d, dt, *u_d)
        v = [a.copy() for a in u]
        ora.correct_velocity(coef, p, v, hh, dt)
        for name, g, want in zip("xyz", u_d, v):
            same(g.cpu().numpy(), want, f"corrected u{name}")
