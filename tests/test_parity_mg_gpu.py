"""Parity of the CUDA multigrid path (through the C ABI) against the oracle's M1-M6, element by
element on the same seeded inputs.  Every step is the same expression in the same order on both
sides (--fmad=false / -ffp-contract=off), and red-black SOR is schedule independent, so the
expectation is ZERO differing doubles; the stated bar (BASELINE.json north_star) is 1e-12 on p
and 1e-10 on the norms.
"""
import numpy as np
import pytest

from paper_2104_01636_b200 import workload as wl

pytestmark = pytest.mark.gpu

P_TOL, NORM_TOL = 1e-12, 1e-10


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


def same(got, want, what):
    scale = np.max(np.abs(want)) or 1.0
    diff = np.max(np.abs(got - want)) / scale
    nbad = int(np.count_nonzero(got != want))
    assert diff <= P_TOL, f"{what}: max-rel diff {diff:.3e}"
    assert nbad == 0, f"{what}: {nbad} doubles differ (max-rel {diff:.3e})"


SHAPES = [
    # nx, ny, nz, spheres, diameter, spacing
    (8, 6, 12, 0, 0, (0.1, 0.07, 0.13)),
    (4, 4, 8, 0, 0, None),
    (40, 36, 24, 2, 8, None),                  # ragged tiles, two levels (nz = 24 -> 12 -> stop)
    (72, 52, 32, 3, 12, (1 / 72, 1 / 60, 1 / 50)),
    (136, 24, 16, 0, 0, None),                 # wider than one x tile of the fused kernel
]


def workload(nx, ny, nz, count, diam, h, seed=5):
    kw = dict(dx=h[0], dy=h[1], dz=h[2]) if h else {}
    w = wl.make_custom(nx, ny, nz, count, diam, seed, **kw)
    if count == 0:
        w.F = wl.random_fraction(nx, ny, nz, seed)
    return w


@pytest.mark.parametrize("shape", SHAPES)
def test_transfer_operators_bitwise(torch_cuda, B, ora, shape):
    w = workload(*shape)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p, 1.3, 3)                      # a non-trivial iterate
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        nlev = s.mg_setup(levels=3, nu_growth=1)
        assert nlev == min(3, ora.mg_max_levels(w.nx, w.ny, w.nz))
        c = coef
        for level in range(1, nlev):                       # M1, level by level
            c = ora.mg_coarsen(c)
            got = [t.cpu().numpy() for t in s.mg_export_coarse(level)]
            for g, want, name in zip(got, c, ("ax", "ay", "az")):
                same(g, want, f"{name} level {level}")
        rc = s.mg_residual_restrict(dev(torch_cuda, w.rhs), dev(torch_cuda, p)).cpu().numpy()
        same(rc, ora.mg_restrict(ora.mg_residual_field(coef, w.rhs, p)), "restricted residual")
        p_d = dev(torch_cuda, p)                           # M4
        s.mg_prolong_add(dev(torch_cuda, rc), p_d)
        q = p.copy()
        ora.mg_prolong_add(rc, q)
        same(p_d.cpu().numpy(), q, "prolongation")


PARAMS = [
    dict(levels=99, nu1=2, nu2=2, coarse_sweeps=20, gamma=1, omega_s=1.2, nu_growth=1, nu_max=64),
    dict(levels=2, nu1=1, nu2=3, coarse_sweeps=7, gamma=2, omega_s=1.0, nu_growth=1, nu_max=64),     # odd sweep counts
    dict(levels=3, nu1=2, nu2=2, coarse_sweeps=30, gamma=2, omega_s=1.3, nu_growth=1, nu_max=64),
    dict(levels=1, nu1=0, nu2=0, coarse_sweeps=5, gamma=1, omega_s=1.5, nu_growth=1, nu_max=64),     # plain SOR
    dict(levels=99, nu1=2, nu2=1, coarse_sweeps=40, gamma=1, omega_s=1.6, nu_growth=4, nu_max=16),
    dict(levels=99, nu1=0, nu2=2, coarse_sweeps=30, gamma=1, omega_s=1.75, nu_growth=4, nu_max=16),  # round 1's defaults
    dict(levels=99, nu1=1, nu2=2, coarse_sweeps=9, gamma=1, omega_s=1.45, omega_c=1.9, nu_growth=3, nu_max=12),  # two relaxation factors
    dict(levels=99, nu1=0, nu2=2, coarse_sweeps=6, gamma=1, omega_s=1.4, omega_c=1.9, nu_growth=8, nu_max=16, nu_max_deep=5),  # fewer sweeps below level 1
    None,                                                                                             # binding.MG_DEFAULTS
]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("prm", PARAMS)
def test_cycles_bitwise(torch_cuda, B, ora, shape, prm):
    w = workload(*shape)
    prm = dict(B.MG_DEFAULTS) if prm is None else prm
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_o = np.zeros_like(w.rhs)
    io = ora.mg_solve(coef, w.rhs, p_o, 3, 0.0, **prm)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        s.mg_setup(**prm)
        p_d = torch_cuda.zeros(w.rhs.shape, dtype=torch_cuda.float64, device="cuda")
        ig = s.mg_solve(dev(torch_cuda, w.rhs), p_d, 3, 0.0)
        same(p_d.cpu().numpy(), p_o, f"p after 3 cycles {prm}")
        assert ig.sweeps == io.sweeps == 3
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
        assert s.launch_count() > 0


def test_config1_to_tolerance_same_cycle_count(torch_cuda, B, ora):
    w = wl.make_config(1)
    prm = dict(levels=3, nu1=2, nu2=2, coarse_sweeps=100, gamma=1, omega_s=1.2, nu_growth=1, nu_max=64)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_o = np.zeros_like(w.rhs)
    io = ora.mg_solve(coef, w.rhs, p_o, 200, 1e-8, **prm)
    assert io.converged
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        s.mg_setup(**prm)
        p_d = torch_cuda.zeros(w.rhs.shape, dtype=torch_cuda.float64, device="cuda")
        ig = s.mg_solve(dev(torch_cuda, w.rhs), p_d, 200, 1e-8)
    assert ig.converged and ig.sweeps == io.sweeps
    same(p_d.cpu().numpy(), p_o, "config 1 multigrid solution")
    assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
    # the answer is the solution of the linear system: the oracle's own O5 norm on the GPU's p
    assert ora.residual(coef, w.rhs, p_d.cpu().numpy())[1] <= 1e-8


def test_fused_norm_path_defaults_to_tolerance(torch_cuda, B, ora):
    """With no pre-smoothing on the finest level (the binding defaults, V(0,2)) ps_mg_solve takes
    the norm of every cycle inside the residual + restriction pass of the next one.  The
    (cycle, check)* semantics must not change: same cycle count as the oracle's plain loop, p
    bitwise, norms to 1e-10 (a different fixed summation tree), at least one cycle even from a
    converged start, max_cycles honoured, max_cycles = 0 only measures."""
    w = wl.make_config(1)
    prm = dict(B.MG_DEFAULTS)
    assert prm["nu1"] == 0                                       # the fused-norm path
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_o = np.zeros_like(w.rhs)
    io = ora.mg_solve(coef, w.rhs, p_o, 200, 1e-8, **prm)
    assert io.converged
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        s.mg_setup()                                             # the defaults are prm
        rhs_d = dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros(w.rhs.shape, dtype=torch_cuda.float64, device="cuda")
        ig = s.mg_solve(rhs_d, p_d, 200, 1e-8)
        assert ig.converged and ig.sweeps == io.sweeps
        same(p_d.cpu().numpy(), p_o, "config 1, default multigrid")
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
        ra, rr, bn = s.residual(rhs_d, p_d)                      # the a4 kernel on the same p
        assert abs(ig.res_rel - rr) <= NORM_TOL * rr and abs(ig.rhs_norm - bn) <= NORM_TOL * bn
        # converged start: still one cycle, as in the oracle's loop
        q_o = p_o.copy()
        jo = ora.mg_solve(coef, w.rhs, q_o, 200, 1e-8, **prm)
        jg = s.mg_solve(rhs_d, p_d, 200, 1e-8)
        assert (jg.sweeps, jg.converged) == (jo.sweeps, jo.converged) == (1, 1)
        same(p_d.cpu().numpy(), q_o, "one more cycle from the converged iterate")
        # max_cycles reached without convergence; max_cycles = 0 leaves p alone
        p_d.zero_()
        p3 = np.zeros_like(w.rhs)
        ko = ora.mg_solve(coef, w.rhs, p3, 3, 1e-8, **prm)
        kg = s.mg_solve(rhs_d, p_d, 3, 1e-8)
        assert (kg.sweeps, kg.converged) == (ko.sweeps, ko.converged) == (3, 0)
        same(p_d.cpu().numpy(), p3, "three default cycles")
        zg = s.mg_solve(rhs_d, p_d, 0, 1e-8)
        assert zg.sweeps == 0 and abs(zg.res_rel - kg.res_rel) <= NORM_TOL * kg.res_rel
        same(p_d.cpu().numpy(), p3, "max_cycles = 0")


def test_config3_three_cycles_and_state_errors(torch_cuda, B, ora):
    w = wl.make_config(3)
    prm = dict(levels=4, nu1=2, nu2=2, coarse_sweeps=40, gamma=1, omega_s=1.2, nu_growth=1, nu_max=64)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_o = np.zeros_like(w.rhs)
    io = ora.mg_solve(coef, w.rhs, p_o, 3, 0.0, **prm)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        rhs_d = dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros(w.rhs.shape, dtype=torch_cuda.float64, device="cuda")
        with pytest.raises(B.PsError):                     # no coefficients yet
            s.mg_setup(**prm)
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        with pytest.raises(B.PsError):                     # no hierarchy yet
            s.mg_solve(rhs_d, p_d, 1, 0.0)
        with pytest.raises(B.PsError):
            s.mg_setup(levels=2, gamma=3)
        assert s.mg_setup(**prm) == 4
        ig = s.mg_solve(rhs_d, p_d, 3, 0.0)
        same(p_d.cpu().numpy(), p_o, "config 3, 3 V-cycles")
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)     # invalidates the hierarchy
        with pytest.raises(B.PsError):
            s.mg_solve(rhs_d, p_d, 1, 0.0)


def test_diverging_parameters_stop_early(torch_cuda, B):
    """V(0,2) with 2 / 8 / 16 sweeps per level and one relaxation factor of 1.9 diverges
    (DESIGN.md §12); ps_mg_solve must not grind through max_cycles on infinities: it stops at the
    first cycle whose norm is not finite."""
    w = wl.make_config(1)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        s.mg_setup(levels=6, nu1=0, nu2=2, coarse_sweeps=30, gamma=1, omega_s=1.9, omega_c=1.9,
                   nu_growth=4, nu_max=16, stall_cycles=0)      # safeguard M7 off: let it diverge
        p_d = torch_cuda.zeros(w.rhs.shape, dtype=torch_cuda.float64, device="cuda")
        info = s.mg_solve(dev(torch_cuda, w.rhs), p_d, 100000, 1e-8)
        assert not info.converged and info.sweeps < 100000
        assert not np.isfinite(info.res_rel)


def test_level_memory_is_caller_owned_and_setup_failures_leave_no_half_built_hierarchy(torch_cuda, B, ora):
    """ps_mg_workspace_bytes / ps_mg_set_workspace: the binding hands the level memory over as a
    torch allocation; a block that is too small makes ps_mg_setup fail with PS_EINVAL, drops the
    hierarchy (ps_mg_levels == 0, ps_mg_solve -> PS_ESTATE), and a later set-up with enough memory
    works and gives the oracle's bits; changing the depth re-uses or rebuilds the chain."""
    import ctypes
    w = workload(40, 36, 24, 2, 8, None)
    prm = dict(levels=2, nu1=1, nu2=1, coarse_sweeps=9, gamma=1, omega_s=1.3, nu_growth=1, nu_max=64)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_o = np.zeros_like(w.rhs)
    ora.mg_solve(coef, w.rhs, p_o, 2, 0.0, **prm)
    lib = B.load()
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        need = lib.ps_mg_workspace_bytes(s._h, 2)
        assert need > 7 * (w.nx // 2) * (w.ny // 2) * (w.nz // 2) * 8
        assert lib.ps_mg_workspace_bytes(s._h, 1) == 0
        deepest = ora.mg_max_levels(w.nx, w.ny, w.nz)             # 3 for this grid
        assert lib.ps_mg_workspace_bytes(s._h, 99) == lib.ps_mg_workspace_bytes(s._h, deepest) > need
        small = torch_cuda.empty(need // 2 + 256, dtype=torch_cuda.uint8, device="cuda")
        base = (small.data_ptr() + 255) // 256 * 256
        assert lib.ps_mg_set_workspace(s._h, ctypes.c_void_p(base + 8), need) == B.PS_EINVAL   # misaligned
        assert lib.ps_mg_set_workspace(s._h, ctypes.c_void_p(base), need // 2) == B.PS_OK
        c_prm = B._MgParams(prm["levels"], prm["nu1"], prm["nu2"], prm["nu_growth"], prm["nu_max"],
                            prm["coarse_sweeps"], prm["gamma"], prm["omega_s"], prm["omega_s"],
                            prm["nu_max"])
        assert lib.ps_mg_setup(s._h, ctypes.byref(c_prm)) == B.PS_EINVAL
        assert lib.ps_mg_levels(s._h) == 0
        rhs_d = dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros(w.rhs.shape, dtype=torch_cuda.float64, device="cuda")
        with pytest.raises(B.PsError) as e:
            s.mg_solve(rhs_d, p_d, 1, 0.0)
        assert e.value.code == B.PS_ESTATE
        s._mg_ws = None                       # let the binding allocate a block that fits
        assert s.mg_setup(**prm) == 2
        s.mg_solve(rhs_d, p_d, 2, 0.0)
        same(p_d.cpu().numpy(), p_o, "after a failed set-up")
        assert s.mg_setup(**dict(prm, levels=1)) == 1             # shallower: chain dropped
        assert s.mg_setup(**prm) == 2                             # and rebuilt in the same block
        p_d.zero_()
        s.mg_solve(rhs_d, p_d, 2, 0.0)
        same(p_d.cpu().numpy(), p_o, "after a depth change")
    # library-owned level memory (no torch block): same numbers
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, workspace=False) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        assert s.mg_setup(**prm) == 2
        p_d = torch_cuda.zeros(w.rhs.shape, dtype=torch_cuda.float64, device="cuda")
        s.mg_solve(dev(torch_cuda, w.rhs), p_d, 2, 0.0)
        same(p_d.cpu().numpy(), p_o, "library-owned level memory")


# ---------------------------------------------------------------- M7: safeguard of the solve loop
@pytest.mark.parametrize("h", [(4 / 64, 1 / 64, 1 / 64), (1 / 64, 2 / 64, 4 / 64)])
def test_stall_safeguard_bitwise_on_anisotropic_ducts(torch_cuda, B, ora, h):
    """The binding defaults on a duct with 4:1:1 / 1:2:4 spacing: omega_c = 1.97 diverges there,
    the safeguard (3 cycles without a new best norm -> omega_c - 0.05) brings it back.  Both the
    fused-norm loop (nu1 = 0: the defaults) and the plain loop (nu1 = 1) must take the oracle's
    decisions: p bitwise after 40 cycles, and without the safeguard the same run diverges."""
    w = workload(64, 64, 128, 6, 8, h)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    rhs_d = dev(torch_cuda, w.rhs)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        for extra in ({}, {"nu1": 1}):
            prm = dict(B.MG_DEFAULTS, **extra)
            p_o = np.zeros_like(w.rhs)
            io = ora.mg_solve(coef, w.rhs, p_o, 40, 0.0, **prm)
            s.mg_setup(**prm)
            p_d = torch_cuda.zeros_like(rhs_d)
            ig = s.mg_solve(rhs_d, p_d, 40, 0.0)
            same(p_d.cpu().numpy(), p_o, f"safeguarded cycles {extra}")
            assert abs(ig.res_rel - io.res_rel) <= 1e-10 * io.res_rel
            assert ig.res_rel < 0.1
        s.mg_setup(**dict(B.MG_DEFAULTS, stall_cycles=0))
        p_d = torch_cuda.zeros_like(rhs_d)
        plain = s.mg_solve(rhs_d, p_d, 40, 0.0)
        assert plain.res_rel > 10 * ig.res_rel
        lib = B.load()
        bad = B._MgParams(6, 0, 2, 24, 48, 10, 1, 1.4, 1.97, 48, -1, 0.05)
        import ctypes
        assert lib.ps_mg_setup(s._h, ctypes.byref(bad)) == B.PS_EINVAL
        bad = B._MgParams(6, 0, 2, 24, 48, 10, 1, 1.4, 1.97, 48, 3, float("nan"))
        assert lib.ps_mg_setup(s._h, ctypes.byref(bad)) == B.PS_EINVAL
