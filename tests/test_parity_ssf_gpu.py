"""Parity of ps_ssf_rhs against the oracle (bitwise), and the p~ solve as a second right-hand side
on the same coefficient set."""
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


@pytest.mark.parametrize("shape", [(24, 24, 32, 1, 8), (40, 36, 24, 2, 8), (72, 52, 34, 3, 12),
                                   (5, 7, 6, 0, 0)])
def test_ssf_rhs_bitwise(torch_cuda, B, ora, shape):
    nx, ny, nz, count, D = shape
    w = wl.make_custom(nx, ny, nz, count, D, 3)
    if count == 0:
        w.F = wl.random_fraction(nx, ny, nz, 3)
        kappa = np.abs(w.rhs) * 10.0
    else:
        kappa = wl.curvature_field(nx, ny, nz, w.centres, D, w.dx)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    want = ora.ssf_rhs(coef, w.F, kappa, wl.SIGMA)
    with B.PoissonSolver(nx, ny, nz, w.dx, w.dy, w.dz) as s:
        F_d = dev(torch_cuda, w.F)
        with pytest.raises(B.PsError):
            s.ssf_rhs(F_d, dev(torch_cuda, kappa), wl.SIGMA)
        s.set_fraction(F_d, w.rho_l, w.rho_g)
        got = s.ssf_rhs(F_d, dev(torch_cuda, kappa), wl.SIGMA).cpu().numpy()
    assert int(np.count_nonzero(got != want)) == 0


def test_two_right_hand_sides_on_one_coefficient_set(torch_cuda, B, ora):
    """Config 1: p~ (steps 6-7) and p (step 11) solved back to back with one ps_set_fraction and
    one ps_mg_setup; p~ shows the Laplace jump 2 sigma / R; a warm start from the converged p~
    needs no further cycle."""
    w = wl.make_config(1)
    R = 4 * w.dx
    kappa = wl.curvature_field(w.nx, w.ny, w.nz, w.centres, 8, w.dx)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        F_d = dev(torch_cuda, w.F)
        s.set_fraction(F_d, w.rho_l, w.rho_g)
        s.mg_setup()
        rhs_t = s.ssf_rhs(F_d, dev(torch_cuda, kappa), wl.SIGMA)
        pt = torch_cuda.zeros_like(rhs_t)
        it = s.mg_solve(rhs_t, pt, 300, 1e-10)
        assert it.converged
        p = torch_cuda.zeros_like(rhs_t)
        ip = s.mg_solve(dev(torch_cuda, w.rhs), p, 300, 1e-8)
        assert ip.converged
        again = s.mg_solve(rhs_t, pt, 300, 1e-10)          # warm start: converged at cycle 1
        assert again.converged and again.sweeps == 1
    q = pt.cpu().numpy()
    jump = q[w.F == 0.0].mean() - q[w.F == 1.0].mean()
    assert abs(jump - 2.0 * wl.SIGMA / R) <= 1e-7 * 2.0 * wl.SIGMA / R
