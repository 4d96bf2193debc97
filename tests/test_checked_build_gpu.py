"""The repo's own memory and race checks of the CUDA path (compute-sanitizer is closed on the B200
pool -- profiles/r02_sanitizer.md quotes the pool's answer, which asks for "bounds checks and
asserts of your own, small cases, and a comparison with the CPU reference"):

1. libps_poisson_checked.so (-DPS_CHECKED): the fused sweep kernel checks every shared-memory
   address it forms, every TMA destination, every global store, and its mbarrier ring protocol
   through plane / stage / red-step tags (ps_kernels_zmarch.cuh "checked build"); it counts
   violations in a device record.  The cases below must leave the record at zero AND reproduce the
   oracle bit for bit; a deliberately broken protocol (the row warps skip the red-barrier wait) must
   be noticed -- the negative control of the checks.
2. Guard bands with the PRODUCT library: every array a kernel may touch (F, rhs, p, velocities,
   outputs, the workspace, the multigrid level block, the host-staging block) is carved from one
   arena pre-filled with NaNs, each array between two guard zones.  A stray write lands in a guard
   (checked afterwards, bit for bit); a stray read of a guard or of uninitialised workspace brings
   a NaN into a result that is compared with the oracle.
"""
import ctypes

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


@pytest.fixture(scope="module")
def checked(B):
    from paper_2104_01636_b200 import build
    lib = B.load(build.build(checked=True))
    assert lib.ps_checked_build() == 1 and B.load().ps_checked_build() == 0
    return lib


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def workload(nx, ny, nz, seed=3):
    w = wl.make_custom(nx, ny, nz, 0, 0, seed)
    w.F = wl.random_fraction(nx, ny, nz, seed)
    return w


CASES = [
    # nx, ny, nz, sweeps, (kernel, z_chunks) list
    (32, 32, 64, 6),        # config-1 shape: one tile across (narrow boxes, no ring warp)
    (64, 64, 128, 4),       # config-2 shape
    (186, 46, 8, 5),        # ragged tiles in x and y, ring columns on both sides
    (256, 20, 12, 5),       # four full tiles across
    (130, 44, 4, 3),        # a one-pair last tile
    (2, 2, 2, 3),
]


@pytest.mark.parametrize("nx,ny,nz,nsweeps", CASES)
def test_checked_kernel_counts_no_violation_and_matches_oracle(torch_cuda, B, checked, ora, nx, ny,
                                                               nz, nsweeps):
    w = workload(nx, ny, nz)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p_ora, w.omega, nsweeps)
    for kernel in (B.KERNEL_FUSED, B.KERNEL_FUSED_OTF):
        for chunks in (0, 1, 2, 3):
            if chunks > nz // 2:
                continue
            with B.PoissonSolver(nx, ny, nz, w.dx, w.dy, w.dz, lib=checked) as s:
                s.set_kernel(kernel)
                s.set_tuning(1, chunks)
                s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
                p_d = torch_cuda.zeros(w.rhs.shape, dtype=torch_cuda.float64, device="cuda")
                s.sweeps(dev(torch_cuda, w.rhs), p_d, w.omega, nsweeps)
                rec = s.debug_read()
                assert rec[0] == 0, f"kernel {kernel} chunks {chunks}: {rec[0]} violations, first {rec[1:6]}"
                assert int(np.count_nonzero(p_d.cpu().numpy() != p_ora)) == 0


def test_checked_kernel_long_run_and_multigrid(torch_cuda, B, checked, ora):
    """config 3 (18 tiles, all SMs, rounds + re-cut leftover): 300 sweeps and three default
    multigrid cycles (fused kernel on levels 0-2) without a violation, p bitwise the oracle's."""
    w = wl.make_config(3)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p_ora, w.omega, 300)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, lib=checked) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        rhs_d = dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros_like(rhs_d)
        s.sweeps(rhs_d, p_d, w.omega, 300)
        assert s.debug_read()[0] == 0, s.debug_read()
        assert int(np.count_nonzero(p_d.cpu().numpy() != p_ora)) == 0
        # the launch options the library would not pick by itself: dependent launches and pacing
        # both on, both off (the producer then waits on the pacing counter / the grid dependency
        # before it issues the p planes; the ring tags still have to come out right)
        for dep, window in ((1, 2), (1, 1), (0, 0)):
            s.set_launch_options(dep, window)
            p_d.zero_()
            s.sweeps(rhs_d, p_d, w.omega, 300)
            assert s.debug_read()[0] == 0, (dep, window, s.debug_read())
            assert int(np.count_nonzero(p_d.cpu().numpy() != p_ora)) == 0, (dep, window)
        s.set_launch_options(-1, -1)
        prm = dict(B.MG_DEFAULTS)
        q_ora = np.zeros_like(w.rhs)
        ora.mg_solve(coef, w.rhs, q_ora, 3, 0.0, **prm)
        s.mg_setup(**prm)
        p_d.zero_()
        s.mg_solve(rhs_d, p_d, 3, 0.0)
        assert s.debug_read()[0] == 0, s.debug_read()
        assert int(np.count_nonzero(p_d.cpu().numpy() != q_ora)) == 0


def test_checks_notice_a_broken_protocol(torch_cuda, B, checked):
    """Negative control: with the red-barrier wait of the row warps switched off the black update
    may read a neighbour's red value before it is written; the red-step tags (code 6) must catch
    it at least once in 200 sweeps on a grid that keeps every SM busy.  Harmless to memory."""
    w = wl.make_config(3)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, lib=checked) as s:
        assert checked.ps_debug_sabotage(s._h, 1) == B.PS_OK
        s.set_kernel(B.KERNEL_FUSED)
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        rhs_d = dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros_like(rhs_d)
        s.sweeps(rhs_d, p_d, w.omega, 200)
        rec = s.debug_read()
        assert rec[0] > 0 and rec[1] == 6, rec
    with B.PoissonSolver(8, 8, 8, 1.0, 1.0, 1.0) as s:               # product build: no such switch
        assert B.load().ps_debug_sabotage(s._h, 1) == B.PS_EINVAL
        assert s.debug_read() == [0] * 8


def test_pacing_gives_up_instead_of_deadlocking(torch_cuda, B, checked, ora):
    """Pacing assumes that all CTAs of the persistent grid are resident at once.  If one of them
    never shows up in the pacing counter (sabotage 2: CTA 0 does not claim its stages until it
    is done -- what a CTA kept off the SMs by foreign work looks like to the others) the others
    must not wait for ever: each gives up after about a millisecond and runs free.  The give-up is
    remembered on the device, so the launches after it do not wait at all; setting the launch
    options again re-arms the pacing.  The paced launches come after an unpaced batch on the same
    context: the host's base of the counter must not have moved during it (it once did, and no
    paced launch after an unpaced one ever waited).  p is bitwise right, no ring violation."""
    import time
    w = workload(128, 128, 64)                     # 18 tiles x 1 z chunk: 18 CTAs of 67 stages;
                                                   # without CTA 0 the mean falls behind at stage 40
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p_ora, w.omega, 5)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, lib=checked) as s:
        s.set_kernel(B.KERNEL_FUSED)
        s.set_tuning(1, 1)
        assert s.get_tuning()[3] == 18
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        rhs_d = dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros_like(rhs_d)
        s.set_launch_options(0, 0)
        s.sweeps(rhs_d, p_d, w.omega, 7)             # unpaced batch (and the warm-up)
        p_d.zero_()
        s.set_launch_options(0, 2)
        assert checked.ps_debug_sabotage(s._h, 2) == B.PS_OK

        def one_sweep():
            torch_cuda.cuda.synchronize()
            t0 = time.perf_counter()
            s.sweeps(rhs_d, p_d, w.omega, 1)
            torch_cuda.cuda.synchronize()
            return time.perf_counter() - t0

        t = [one_sweep() for _ in range(4)]
        s.set_launch_options(0, 2)                   # re-arm
        t.append(one_sweep())
        free = min(t[1:4])
        assert max(t) < 5.0, t
        assert t[0] > free + 0.4e-3, t               # the first paced launch waited for CTA 0 ...
        assert max(t[1:4]) < free + 0.3e-3, t        # ... the next three did not ...
        assert t[4] > free + 0.4e-3, t               # ... and the re-armed one did again
        assert s.debug_read()[0] == 0, s.debug_read()
        assert int(np.count_nonzero(p_d.cpu().numpy() != p_ora)) == 0


# ------------------------------------------------------------------------------- guard bands
GUARD = 4096          # doubles per guard zone (32 KB)


class Arena:
    """One NaN-filled device buffer; arrays are carved out between guard zones."""

    def __init__(self, torch, doubles):
        self.torch = torch
        self.buf = torch.full((doubles,), float("nan"), dtype=torch.float64, device="cuda")
        self.pos = GUARD
        self.used = []

    def take(self, n, shape=None):
        n_al = (n + 31) // 32 * 32                      # keep every array 256-byte aligned
        assert self.pos + n_al + GUARD <= self.buf.numel(), "arena too small"
        t = self.buf[self.pos:self.pos + n]
        self.used.append((self.pos, self.pos + n))
        self.pos += n_al + GUARD
        return t.view(shape) if shape else t

    def guards_intact(self):
        mask = self.torch.ones(self.buf.numel(), dtype=self.torch.bool, device="cuda")
        for a, b in self.used:
            mask[a:b] = False
        return bool(self.torch.isnan(self.buf[mask]).all())


@pytest.mark.parametrize("shape", [(32, 32, 64), (186, 46, 8), (130, 44, 4), (5, 7, 6)])
def test_guard_bands_stay_intact_and_no_nan_leaks_in(torch_cuda, B, ora, shape):
    torch = torch_cuda
    nx, ny, nz = shape
    w = workload(nx, ny, nz, seed=9)
    n = nx * ny * nz
    sh = (nz, ny, nx)
    lib = B.load()
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    variants = [B.KERNEL_TWOPASS, B.KERNEL_RESIDENT, B.KERNEL_CLUSTER] + ([B.KERNEL_FUSED, B.KERNEL_FUSED_OTF] if nx % 2 == 0 else [])
    for kernel in variants:
        with B.PoissonSolver(nx, ny, nz, w.dx, w.dy, w.dz, workspace=False) as s:
            ws_n = lib.ps_workspace_bytes(s._h) // 8
            mg_n = lib.ps_mg_workspace_bytes(s._h, 3) // 8
            st_n = lib.ps_host_staging_bytes(s._h) // 8
            ar = Arena(torch, 14 * (n + 40 + GUARD) + ws_n + mg_n + st_n + 8 * GUARD)
            F, rhs, p = ar.take(n, sh), ar.take(n, sh), ar.take(n, sh)
            ws, mg, st = ar.take(ws_n), ar.take(max(mg_n, 32)), ar.take(st_n)
            u = [ar.take(n, sh) for _ in range(3)]
            out1, out2, out3, kap = ar.take(n, sh), ar.take(n, sh), ar.take(n, sh), ar.take(n, sh)
            F.copy_(dev(torch, w.F)); rhs.copy_(dev(torch, w.rhs)); p.zero_()
            kap.copy_(dev(torch, wl.noise_rhs(nx, ny, nz, 77)))
            for q in range(3):
                u[q].copy_(dev(torch, wl.noise_rhs(nx, ny, nz, 50 + q)))
            assert lib.ps_set_workspace(s._h, ctypes.c_void_p(ws.data_ptr()), ws_n * 8) == B.PS_OK
            if mg_n:
                assert lib.ps_mg_set_workspace(s._h, ctypes.c_void_p(mg.data_ptr()), mg_n * 8) == B.PS_OK
            assert lib.ps_set_host_staging(s._h, ctypes.c_void_p(st.data_ptr()), st_n * 8) == B.PS_OK
            try:
                s.set_kernel(kernel)
            except B.PsError:
                assert kernel == B.KERNEL_CLUSTER       # the grid does not fit one cluster
                continue
            s.set_fraction(F, w.rho_l, w.rho_g)
            info = s.solve(rhs, p, w.omega, 5, 0.0)
            p_ora = np.zeros_like(w.rhs)
            io = ora.solve(coef, w.rhs, p_ora, w.omega, 5, 0.0)
            assert int(np.count_nonzero(p.cpu().numpy() != p_ora)) == 0, kernel
            assert abs(info.res_rel - io.res_rel) <= 1e-10 * io.res_rel
            # host path through the staging block
            ph = np.zeros_like(w.rhs)
            s.solve_host(w.F, w.rho_l, w.rho_g, w.rhs, ph, w.omega, 5, 0.0)
            assert int(np.count_nonzero(ph != p_ora)) == 0
            # multigrid (levels live in the arena block), projection and surface-tension kernels
            nlev = s.mg_setup(levels=3, nu1=1, nu2=1, coarse_sweeps=4, omega_s=1.3, nu_growth=2, nu_max=4)
            q_ora = p_ora.copy()
            ora.mg_solve(coef, w.rhs, q_ora, 1, 0.0, levels=3, nu1=1, nu2=1, coarse_sweeps=4,
                         omega_s=1.3, nu_growth=2, nu_max=4)
            s.mg_solve(rhs, p, 1, 0.0)
            assert nlev >= 1 and int(np.count_nonzero(p.cpu().numpy() != q_ora)) == 0
            h = (w.dx, w.dy, w.dz)
            uh = [wl.noise_rhs(nx, ny, nz, 50 + q) for q in range(3)]
            s.rhs_from_velocity(*u, 1e-3, out1)
            assert np.array_equal(out1.cpu().numpy(), ora.rhs_from_velocity(uh, h, 1e-3))
            lib_div = lib.ps_face_divergence(s._h, *[ctypes.c_void_p(t.data_ptr()) for t in (*u, p)],
                                             1e-3, ctypes.c_void_p(out2.data_ptr()))
            assert lib_div == B.PS_OK
            assert np.array_equal(out2.cpu().numpy(), ora.face_divergence(coef, uh, q_ora, h, 1e-3))
            assert lib.ps_ssf_rhs(s._h, ctypes.c_void_p(F.data_ptr()), ctypes.c_void_p(kap.data_ptr()),
                                  0.07, ctypes.c_void_p(out3.data_ptr())) == B.PS_OK
            assert np.array_equal(out3.cpu().numpy(),
                                  ora.ssf_rhs(coef, w.F, wl.noise_rhs(nx, ny, nz, 77), 0.07))
            s.correct_velocity(p, 1e-3, *u)
            ora.correct_velocity(coef, q_ora, uh, h, 1e-3)
            for q in range(3):
                assert np.array_equal(u[q].cpu().numpy(), uh[q])
            torch.cuda.synchronize()
            assert ar.guards_intact(), f"kernel {kernel}: a guard zone was written"
