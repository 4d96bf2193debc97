"""ps_residual_noalloc against ps_residual (the existing path), on the GPU.

ps_residual_noalloc is the entry point for callers that cannot allocate device memory when they
call into the library: a flow solver whose own memory pool already owns the board (a cudaMalloc
inside it may fail, and it stalls every stream of the device while it runs), or a plug-in that is
given pointers and a stream but no allocator.  It keeps the reduction's scratch in a fixed array
inside the library, which every call on the device shares and which keeps the last call's
contents.  So the thing to check is not one call but calls in a row: a big grid first (fills
thousands of scratch slots), then smaller ones (which must not see what the big one left), then
the big one again -- each against ps_residual on the same data.  Both paths add in the same
order, so the numbers must be bitwise equal; the suite's norm tolerance is asserted as well.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It builds everything it needs itself, so it passes alone in
a fresh process as well as after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

from paper_2104_01636_b200 import workload as wl

pytestmark = pytest.mark.gpu

NORM_TOL = 1e-10    # the suite's bar for norms (tests/test_parity_gpu.py)


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


class Case:
    """One grid with coefficients, a right-hand side and a partly relaxed p on the device, and
    the three norms ps_residual returns for them."""

    def __init__(self, torch, B, nx, ny, nz, count, diam, seed, sweeps):
        w = wl.make_custom(nx, ny, nz, count, diam, seed)
        if count == 0:
            w.F = wl.random_fraction(nx, ny, nz, seed)
        self.w = w
        self.rhs = torch.from_numpy(np.ascontiguousarray(w.rhs)).cuda()
        self.p = torch.zeros_like(self.rhs)
        self.existing_path(torch, B, sweeps)
        self.out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")

    def existing_path(self, torch, B, sweeps=0):
        w = self.w
        with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
            s.set_fraction(torch.from_numpy(np.ascontiguousarray(w.F)).cuda(), w.rho_l, w.rho_g)
            s.sweeps(self.rhs, self.p, w.omega, sweeps)
            self.ax, self.ay, self.az = s.export_coefficients()
            self.expect = s.residual(self.rhs, self.p)

    def check(self, torch, B, what):
        self.out.fill_(float("nan"))
        B.residual_noalloc(self.ax, self.ay, self.az, self.rhs, self.p, self.out)
        torch.cuda.synchronize()
        got = tuple(self.out.cpu().tolist())
        for g, e, name in zip(got, self.expect, ("res_abs", "res_rel", "rhs_norm")):
            assert abs(g - e) <= NORM_TOL * abs(e), f"{what}: {name} {g!r} vs {e!r}"
        assert got == self.expect, f"{what}: not bitwise: {got!r} vs {self.expect!r}"


def test_calls_in_a_row_match_ps_residual(torch_cuda, B):
    torch = torch_cuda
    big = Case(torch, B, 128, 96, 160, 6, 12, 5, 7)        # 480 chunks, even nx (pair loads)
    odd = Case(torch, B, 37, 21, 10, 0, 0, 6, 3)           # 2 chunks, ragged, odd nx (scalar loads)
    tiny = Case(torch, B, 2, 3, 2, 0, 0, 7, 2)             # one partly filled chunk
    assert big.expect[0] > 0.0 and odd.expect[0] > 0.0
    big.check(torch, B, "first call, big grid")
    big.check(torch, B, "second call, same data")
    odd.check(torch, B, "small odd grid after the big one")
    tiny.check(torch, B, "12 cells after the others")
    big.p.mul_(1.5)                                        # other data, same slots
    big.existing_path(torch, B)
    big.check(torch, B, "big grid again, changed p")


def test_back_to_back_without_a_sync_in_between(torch_cuda, B):
    """Two calls enqueued on one stream with no host synchronisation between them: stream order
    is all the ordering the shared array needs."""
    torch = torch_cuda
    a = Case(torch, B, 64, 48, 40, 2, 8, 8, 4)
    b = Case(torch, B, 40, 36, 24, 2, 8, 9, 4)
    B.residual_noalloc(a.ax, a.ay, a.az, a.rhs, a.p, a.out)
    B.residual_noalloc(b.ax, b.ay, b.az, b.rhs, b.p, b.out)
    torch.cuda.synchronize()
    assert tuple(a.out.cpu().tolist()) == a.expect
    assert tuple(b.out.cpu().tolist()) == b.expect


def test_size_limit_and_bad_arguments_are_refused(torch_cuda, B):
    torch = torch_cuda
    lib = B.load()
    t = torch.zeros(64, dtype=torch.float64, device="cuda")     # never touched by a refused call
    q = ctypes.c_void_p(t.data_ptr())
    assert 1024 * 1024 * 256 == B.NOALLOC_MAX_CELLS
    rc = lib.ps_residual_noalloc(1024, 1024, 258, q, q, q, q, q, None, q)
    assert rc == B.PS_ETOOBIG
    assert b"PS_NOALLOC_MAX_CELLS" in lib.ps_strerror(rc)
    assert lib.ps_residual_noalloc(4, 4, 3, q, q, q, q, q, None, q) == B.PS_EINVAL      # odd nz
    assert lib.ps_residual_noalloc(4, 4, 4, q, q, None, q, q, None, q) == B.PS_EINVAL   # NULL
    off = ctypes.c_void_p(t.data_ptr() + 8)
    assert lib.ps_residual_noalloc(4, 4, 4, q, q, q, off, q, None, q) == B.PS_EINVAL    # alignment
    torch.cuda.synchronize()
    assert float(t.abs().sum()) == 0.0
