"""Parity at the run lengths BASELINE.json's configs state, and the oracle's own norm on every
to-tolerance result of the CUDA path (SURVEY.md §8.d "Timing the oracle beside it": config 3
"parity of p and norms at a fixed 2,000 sweeps always", config 5 "oracle runs the 300 sweeps",
long runs pinned by "oracle O5 evaluated on the GPU's p, one pass").

Config 4's 500 sweeps and config 5's 300 sweeps are compared element by element in
tests/test_parity_gpu.py::test_full_size_configs; this file adds
  * config 3 at 2,000 sweeps (bitwise) and its plain-SOR solve to 1e-8 (oracle norm of the GPU's p),
  * the multigrid path with the BINDING DEFAULTS (6 levels, V(0,2), fused residual + restriction +
    norm pass on the finest level, streaming sweeps on the large levels and the resident kernel on
    the small ones) on configs 3, 4 and 5: cycles bitwise against oracle M1-M6, then the solve to
    1e-8 with the oracle's O5 norm evaluated on the GPU's final p.
All calls go through the C ABI (binding.PoissonSolver).
"""
import functools

import numpy as np
import pytest

from paper_2104_01636_b200 import workload as wl

pytestmark = pytest.mark.gpu

P_TOL, NORM_TOL, TOL = 1e-12, 1e-10, 1e-8


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2104_01636_b200 import binding, build
    build.build()
    binding.load()          # fails loudly if the CUDA extension is missing
    return binding


@functools.lru_cache(maxsize=1)
def config(cfg):
    return wl.make_config(cfg)


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def same(got, want, what):
    scale = np.max(np.abs(want)) or 1.0
    diff = np.max(np.abs(got - want)) / scale
    nbad = int(np.count_nonzero(got != want))
    assert diff <= P_TOL, f"{what}: max-rel diff {diff:.3e}"
    assert nbad == 0, f"{what}: {nbad} doubles differ (max-rel {diff:.3e})"


def check_against_oracle_norm(ora, coef, w, p_gpu, info, what):
    """O5 on the GPU's final p: the oracle must call the result converged too, and its norm
    must be the one the CUDA path reported (1e-10 relative; long double vs fixed tree)."""
    ra, rr, bn = ora.residual(coef, w.rhs, p_gpu)
    assert info.converged, f"{what}: CUDA path did not converge (res_rel {info.res_rel:.3e})"
    assert rr <= TOL, f"{what}: oracle norm of the GPU's p is {rr:.3e} > {TOL}"
    assert abs(info.res_rel - rr) <= NORM_TOL * rr, (what, info.res_rel, rr)
    assert abs(info.res_abs - ra) <= NORM_TOL * ra and abs(info.rhs_norm - bn) <= NORM_TOL * bn
    return rr


def test_config3_2000_sweeps_bitwise_and_sor_to_tolerance(torch_cuda, B, ora):
    """configs[2] (128x128x256, 108 spheres of 12 cells, omega 1.6): p and norms after 2,000
    sweeps against the oracle (kernel AUTO, the launch configuration `report` times); then the
    row-(a5) loop to 1e-8 (326,850 sweeps in round 1) with the oracle's O5 norm on the result."""
    w = config(3)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    io = ora.solve(coef, w.rhs, p_ora, w.omega, 2000, 0.0)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        rhs_d = dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros_like(rhs_d)
        ig = s.solve(rhs_d, p_d, w.omega, 2000, 0.0)
        same(p_d.cpu().numpy(), p_ora, "config 3 after 2,000 sweeps")
        assert ig.sweeps == io.sweeps == 2000
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
        assert abs(ig.res_abs - io.res_abs) <= NORM_TOL * io.res_abs
        # continue the same iterate to the tolerance (p is in/out): sweep counts add up
        ig2 = s.solve(rhs_d, p_d, w.omega, 1_000_000, w.tol)
        assert ig2.sweeps % 50 == 0 and ig2.sweeps > 100_000
        check_against_oracle_norm(ora, coef, w, p_d.cpu().numpy(), ig2, "config 3 plain SOR")


@pytest.mark.parametrize("cfg,cycles", [(3, 3), (4, 3), (5, 2)])
def test_default_multigrid_bitwise_and_to_tolerance(torch_cuda, B, ora, cfg, cycles):
    """The multigrid path exactly as bench.py runs it (binding defaults; on config 4 the fused
    residual + restriction + norm kernel works on 8,192 partials, levels 0-2 run the streaming
    sweep and levels 3-5 the resident kernel): `cycles` cycles bitwise against the oracle, then
    to 1e-8 from p = 0 with the oracle's norm of the GPU's final p."""
    w = config(cfg)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_o = np.zeros_like(w.rhs)
    io = ora.mg_solve(coef, w.rhs, p_o, cycles, 0.0, **B.MG_DEFAULTS)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        assert s.mg_setup() == B.MG_DEFAULTS["levels"] == 6       # the defaults
        rhs_d = dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros_like(rhs_d)
        ig = s.mg_solve(rhs_d, p_d, cycles, 0.0)
        same(p_d.cpu().numpy(), p_o, f"config {cfg}: p after {cycles} default cycles")
        del p_o
        assert ig.sweeps == io.sweeps == cycles
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
        assert abs(ig.rhs_norm - io.rhs_norm) <= NORM_TOL * io.rhs_norm
        p_d.zero_()
        it = s.mg_solve(rhs_d, p_d, 1000, TOL)
        check_against_oracle_norm(ora, coef, w, p_d.cpu().numpy(), it,
                                  f"config {cfg} multigrid ({it.sweeps} cycles)")
