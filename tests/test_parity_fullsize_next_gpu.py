"""Parity of the kernels around the solve at the FULL size of configs 4 and 5, in the launch
geometry they run with there.

tests/test_parity_projection_gpu.py and tests/test_parity_ssf_gpu.py compare steps 10-12
 and the p~ right-hand side (eqs (6)-(7)) with the oracle on
grids of up to 127 k cells, where every grid-stride loop makes one trip and the z-marching pair
kernels launch a few dozen blocks.  At 33.5 M cells (config 4) and 151 M cells (config 5) the
grid-stride kernels make 2-4 trips (the block count is capped at 32 waves of the device), the
z-marching kernels launch thousands of blocks, and the 32-bit index arithmetic of the streaming
kernels is near its range.  Here each of ps_rhs_from_velocity, ps_face_divergence,
ps_correct_velocity, ps_ssf_rhs and ps_export_coefficients is compared with one oracle pass at
those sizes, bitwise, through the C ABI: seeded random u^ and p, the config's own F and the exact
curvature of its spheres.  One kernel at a time, host arrays released in between (config 5 is
1.2 GB per field).
"""
import gc

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
    if nbad:
        where = np.argwhere(got != want)[0]
        raise AssertionError(f"{what}: {nbad} doubles differ, first at (k,j,i) = {tuple(where)}: "
                             f"{got[tuple(where)]!r} vs {want[tuple(where)]!r}")


@pytest.mark.parametrize("cfg", [4, 5])
def test_next_rows_at_full_size(torch_cuda, B, ora, cfg):
    torch = torch_cuda
    w = wl.make_config(cfg)
    sh, hh, dt = w.rhs.shape, (w.dx, w.dy, w.dz), 0.0137
    w.rhs = None                                           # not needed here
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, *hh)
    with B.PoissonSolver(w.nx, w.ny, w.nz, *hh) as s:
        F_d = dev(torch, w.F)
        s.set_fraction(F_d, w.rho_l, w.rho_g)

        # (a1) the coefficient arrays themselves (so far compared at this size only through p)
        for name, got, want in zip(("ax", "ay", "az"), s.export_coefficients(), coef):
            same(got.cpu().numpy(), np.asarray(want).reshape(sh), name)
            del got
        torch.cuda.empty_cache()

        # NEXT-3: rhs of the p~ system from F and the exact curvature of the spheres
        kappa = wl.curvature_field(w.nx, w.ny, w.nz, w.centres, w.diameter, w.dx)
        assert np.count_nonzero(kappa) > 0
        got = s.ssf_rhs(F_d, dev(torch, kappa), wl.SIGMA).cpu().numpy()
        want = ora.ssf_rhs(coef, w.F, kappa, wl.SIGMA)
        assert np.count_nonzero(want) > 0
        same(got, want, "ssf rhs")
        del kappa, got, want, F_d
        gc.collect()
        torch.cuda.empty_cache()

        # NEXT-2: steps 10-12 on a random u^ and a random p
        u = [rnd(sh, 5 + q) for q in range(3)]
        u_d = [dev(torch, a) for a in u]
        got = s.rhs_from_velocity(*u_d, dt).cpu().numpy()
        same(got, ora.rhs_from_velocity(u, hh, dt), "rhs from velocity")
        del got
        p = rnd(sh, 9)
        p_d = dev(torch, p)
        got = s.face_divergence(*u_d, p_d, dt).cpu().numpy()
        same(got, ora.face_divergence(coef, u, p, hh, dt), "face divergence")
        del got
        gc.collect()
        torch.cuda.empty_cache()
        s.correct_velocity(p_d, dt, *u_d)
        ora.correct_velocity(coef, p, u, hh, dt)           # in place on the host copies
        for name, g, want in zip("xyz", u_d, u):
            same(g.cpu().numpy(), want, f"corrected u{name}")
