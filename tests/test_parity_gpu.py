"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Bar (BASELINE.json north_star): max-rel p <= 1e-12 after N sweeps, residual
norms <= 1e-10 relative.  Because both sides round the same expressions in the same order
(--fmad=false / -ffp-contract=off) and red-black SOR is schedule independent, the expectation is
ZERO differing doubles; both are asserted.
"""
import numpy as np
import pytest

from paper_2104_01636_b200 import workload as wl

pytestmark = pytest.mark.gpu

P_TOL = 1e-12       # max_n |p_gpu - p_ora| / max_n |p_ora|
NORM_TOL = 1e-10    # |res_gpu - res_ora| / res_ora


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


def to_dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_p_parity(p_gpu, p_ora, what=""):
    scale = np.max(np.abs(p_ora))
    diff = np.max(np.abs(p_gpu - p_ora)) / (scale if scale > 0 else 1.0)
    nbad = int(np.count_nonzero(p_gpu != p_ora))
    assert diff <= P_TOL, f"{what}: max-rel p diff {diff:.3e}"
    assert nbad == 0, f"{what}: {nbad} doubles differ (max-rel {diff:.3e})"


def variants_for(B, w, tunings=((1, 0, -1, -1), (1, 1, 0, 0), (1, 2, 1, 0), (1, 3, 0, 4),
                                 (1, 0, 1, 1))):
    """Kernel variants the library accepts for this grid shape (asked of the library itself):
    (kernel, rows_per_thread, z_chunks, dependent_launch, pace_window); the fused kernel is run
    in several launch geometries (z_chunks = 0: the balanced split bench.py times; n > 0: tile x
    chunk items) and with its launch options on and off (-1: the library defaults)."""
    out = []
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, workspace=False) as s:
        for v in (B.KERNEL_TWOPASS, B.KERNEL_RESIDENT, B.KERNEL_CLUSTER, B.KERNEL_FUSED_OTF,
                  B.KERNEL_FUSED):
            try:
                s.set_kernel(v)
            except B.PsError:
                continue
            if v in (B.KERNEL_TWOPASS, B.KERNEL_RESIDENT, B.KERNEL_CLUSTER):
                out.append((v, 0, 0, -1, -1))
                continue
            for rpt, chunks, dep, window in tunings:
                try:
                    s.set_tuning(rpt, chunks)
                    s.set_launch_options(dep, window)
                    out.append((v, rpt, chunks, dep, window))
                except B.PsError:
                    pass
    return out


def make_solver(B, w, variant=None):
    s = B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz)
    if variant is not None:
        kernel, rpt, chunks, dep, window = variant
        s.set_kernel(kernel)
        if kernel not in (B.KERNEL_TWOPASS, B.KERNEL_RESIDENT, B.KERNEL_CLUSTER):
            s.set_tuning(rpt, chunks)
            s.set_launch_options(dep, window)
    return s


SHAPES = [
    # nx, ny, nz, spheres, diameter, (dx, dy, dz)
    (16, 12, 20, 0, 0, (0.1, 0.07, 0.13)),       # anisotropic spacing, tiny
    (1, 1, 8, 0, 0, None),                       # 1-D periodic degenerate case
    (5, 7, 6, 0, 0, None),                       # odd nx, ny
    (2, 3, 2, 0, 0, None),                       # smallest legal nz
    (40, 36, 24, 2, 8, None),                    # spheres, several tiles + ragged tails
    (72, 52, 34, 3, 12, (1 / 72, 1 / 60, 1 / 50)),
    (132, 20, 10, 0, 0, None),                   # wider than one x tile
]


def shape_workload(nx, ny, nz, count, diam, h, seed=11):
    kw = {}
    if h is not None:
        kw = dict(dx=h[0], dy=h[1], dz=h[2])
    w = wl.make_custom(nx, ny, nz, count, diam, seed, **kw)
    if count == 0:                                # hardest coefficients: random F in {m/64}
        w.F = wl.random_fraction(nx, ny, nz, seed)
    return w


# ---------------------------------------------------------------- (a1) coefficient build
@pytest.mark.parametrize("shape", SHAPES)
def test_coefficients_bitwise(torch_cuda, B, ora, shape):
    w = shape_workload(*shape)
    ax, ay, az = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    with make_solver(B, w) as s:
        s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        gx, gy, gz = [t.cpu().numpy() for t in s.export_coefficients()]
    assert np.array_equal(gx, ax) and np.array_equal(gy, ay) and np.array_equal(gz, az)


# ---------------------------------------------------------------- (a2)/(a3) half-sweeps
@pytest.mark.parametrize("shape", SHAPES[:5])
def test_half_sweeps_bitwise(torch_cuda, B, ora, shape):
    w = shape_workload(*shape)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p0 = wl.noise_rhs(w.nx, w.ny, w.nz, 99)       # non-trivial start
    with make_solver(B, w) as s:
        s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        rhs_d = to_dev(torch_cuda, w.rhs)
        for colour in (0, 1):
            p_ora = p0.copy()
            ora.half_sweep(coef, w.rhs, p_ora, w.omega, colour)
            p_d = to_dev(torch_cuda, p0)
            s.half_sweep(rhs_d, p_d, w.omega, colour)
            assert_p_parity(p_d.cpu().numpy(), p_ora, f"colour {colour}")
            other = ((np.add.outer(np.add.outer(np.arange(w.nz), np.arange(w.ny)),
                                   np.arange(w.nx)) & 1) != colour)
            assert np.array_equal(p_d.cpu().numpy()[other], p0[other])   # other colour untouched


# ---------------------------------------------------------------- sweeps, every kernel variant
@pytest.mark.parametrize("nsweeps", [1, 2, 3, 7])
@pytest.mark.parametrize("shape", SHAPES)
def test_sweeps_bitwise_all_variants(torch_cuda, B, ora, shape, nsweeps):
    w = shape_workload(*shape)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p_ora, w.omega, nsweeps)
    ra, rr, bn = ora.residual(coef, w.rhs, p_ora)
    for variant in variants_for(B, w):
        with make_solver(B, w, variant) as s:
            s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
            rhs_d = to_dev(torch_cuda, w.rhs)
            p_d = torch_cuda.zeros_like(rhs_d)
            s.sweeps(rhs_d, p_d, w.omega, nsweeps)
            assert_p_parity(p_d.cpu().numpy(), p_ora, f"variant {variant} x{nsweeps}")
            ga, gr, gb = s.residual(rhs_d, p_d)
        assert abs(ga - ra) <= NORM_TOL * ra and abs(gr - rr) <= NORM_TOL * rr
        assert abs(gb - bn) <= NORM_TOL * bn


# ---------------------------------------------------------------- BASELINE.json configs
def test_config1_200_sweeps(torch_cuda, B, ora):
    """configs[0]: 32x32x64, one D=8 sphere, omega 1.5, 200 sweeps -- p and norms."""
    w = wl.make_config(1)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    io = ora.solve(coef, w.rhs, p_ora, w.omega, w.max_sweeps, 0.0)
    for variant in variants_for(B, w):
        with make_solver(B, w, variant) as s:
            s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
            rhs_d = to_dev(torch_cuda, w.rhs)
            p_d = torch_cuda.zeros_like(rhs_d)
            ig = s.solve(rhs_d, p_d, w.omega, w.max_sweeps, 0.0)
            assert_p_parity(p_d.cpu().numpy(), p_ora, f"config1 variant {variant}")
        assert ig.sweeps == io.sweeps == 200 and not ig.converged
        assert abs(ig.res_abs - io.res_abs) <= NORM_TOL * io.res_abs
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
        assert abs(ig.rhs_norm - io.rhs_norm) <= NORM_TOL * io.rhs_norm


def test_config2_to_tolerance(torch_cuda, B, ora):
    """configs[1]: unladen 64x64x128, omega 1.7, to 1e-8: same sweep count, p, norms; and the
    converged field is the eigenmode / lambda (closed form) up to the 1e-3 noise."""
    w = wl.make_config(2)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    io = ora.solve(coef, w.rhs, p_ora, w.omega, 100000, w.tol)
    assert io.converged
    for variant in variants_for(B, w):
        with make_solver(B, w, variant) as s:
            s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
            rhs_d = to_dev(torch_cuda, w.rhs)
            p_d = torch_cuda.zeros_like(rhs_d)
            ig = s.solve(rhs_d, p_d, w.omega, 100000, w.tol)
            p_gpu = p_d.cpu().numpy()
        assert ig.converged and ig.sweeps == io.sweeps
        assert_p_parity(p_gpu, p_ora, f"config2 variant {variant}")
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
        assert ig.res_rel <= w.tol
    import json, os
    with open(os.path.join(os.path.dirname(__file__), "golden", "eigenvalue_config2.json")) as f:
        lam = json.load(f)["lambda_1_2_3"]
    mode = wl.eigenmode(w.nx, w.ny, w.nz, 1, 2, 3) / lam
    q = p_gpu - p_gpu.mean()
    assert np.max(np.abs(q - mode)) <= 2e-2 * np.max(np.abs(mode))


def test_config3_fixed_sweeps(torch_cuda, B, ora):
    """configs[2]: 128x128x256, 108 spheres D=12, omega 1.6 -- bitwise parity at 60 sweeps."""
    w = wl.make_config(3)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    n = 60
    io = ora.solve(coef, w.rhs, p_ora, w.omega, n, 0.0)
    for variant in variants_for(B, w):
        with make_solver(B, w, variant) as s:
            s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
            gx, gy, gz = [t.cpu().numpy() for t in s.export_coefficients()]
            assert np.array_equal(gx, coef[0]) and np.array_equal(gy, coef[1])
            assert np.array_equal(gz, coef[2])
            rhs_d = to_dev(torch_cuda, w.rhs)
            p_d = torch_cuda.zeros_like(rhs_d)
            ig = s.solve(rhs_d, p_d, w.omega, n, 0.0)
            assert_p_parity(p_d.cpu().numpy(), p_ora, f"config3 variant {variant}")
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel


@pytest.mark.parametrize("cfg,nsweeps", [(4, 500), (5, 300)])
def test_full_size_configs(torch_cuda, B, ora, cfg, nsweeps):
    """configs[3] (256x256x512, 864 spheres, its full 500 sweeps) and configs[4] (384x384x1024,
    2048 spheres, its full 300 sweeps: 4.5e10 oracle updates, about a minute of host time) at full
    size in the launch
    configuration bench.py times (kernel AUTO): full-field bitwise parity of p and the norms, then
    two properties that hold at any size: the norm ps_solve reports equals a fresh ps_residual,
    and rolling the inputs by an even number of z planes rolls p bitwise (pin P7)."""
    w = wl.make_config(cfg)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    io = ora.solve(coef, w.rhs, p_ora, w.omega, nsweeps, 0.0)
    del coef
    with make_solver(B, w) as s:
        F_d, rhs_d = to_dev(torch_cuda, w.F), to_dev(torch_cuda, w.rhs)
        s.set_fraction(F_d, w.rho_l, w.rho_g)
        p_d = torch_cuda.zeros_like(rhs_d)
        ig = s.solve(rhs_d, p_d, w.omega, nsweeps, 0.0)
        assert_p_parity(p_d.cpu().numpy(), p_ora, f"config{cfg}")
        del p_ora
        assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
        assert abs(ig.rhs_norm - io.rhs_norm) <= NORM_TOL * io.rhs_norm
        ra, rr, bn = s.residual(rhs_d, p_d)
        assert ig.sweeps == nsweeps and (ra, rr, bn) == (ig.res_abs, ig.res_rel, ig.rhs_norm)
        shift = 6
        s.set_fraction(torch_cuda.roll(F_d, shift, 0).contiguous(), w.rho_l, w.rho_g)
        q_d = torch_cuda.zeros_like(rhs_d)
        s.solve(torch_cuda.roll(rhs_d, shift, 0).contiguous(), q_d, w.omega, nsweeps, 0.0)
        assert torch_cuda.equal(torch_cuda.roll(p_d, shift, 0), q_d)


# ---------------------------------------------------------------- solve loop and API behaviour
def test_solve_check_cadence_matches_oracle(torch_cuda, B, ora):
    """Stops at the first check (every K sweeps and at max_sweeps) with res_rel <= tol."""
    w = shape_workload(16, 12, 20, 0, 0, None)
    w.F[:] = 1.0
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    for K, max_sweeps, tol in [(7, 1000, 1e-6), (50, 33, 1e-30), (10, 1000, 1e-9), (3, 0, 1e-3)]:
        p_ora = np.zeros_like(w.rhs)
        io = ora.solve(coef, w.rhs, p_ora, 1.5, max_sweeps, tol, check_interval=K)
        with make_solver(B, w) as s:
            s.set_check_interval(K)
            s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
            rhs_d = to_dev(torch_cuda, w.rhs)
            p_d = torch_cuda.zeros_like(rhs_d)
            ig = s.solve(rhs_d, p_d, 1.5, max_sweeps, tol)
            assert (ig.sweeps, ig.converged) == (io.sweeps, io.converged), (K, max_sweeps, tol)
            assert_p_parity(p_d.cpu().numpy(), p_ora)
            assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel


def test_warm_start_and_restart(torch_cuda, B, ora):
    """p is in/out: 5 sweeps + 6 sweeps == 11 sweeps, bitwise, for every variant."""
    w = shape_workload(40, 36, 24, 2, 8, None)
    for variant in variants_for(B, w):
        with make_solver(B, w, variant) as s:
            s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
            rhs_d = to_dev(torch_cuda, w.rhs)
            a = torch_cuda.zeros_like(rhs_d)
            s.sweeps(rhs_d, a, w.omega, 5)
            s.sweeps(rhs_d, a, w.omega, 6)
            b = torch_cuda.zeros_like(rhs_d)
            s.sweeps(rhs_d, b, w.omega, 11)
            assert torch_cuda.equal(a, b)


def test_deterministic_norm(torch_cuda, B):
    """The two-pass reduction has a fixed summation tree: repeated calls agree to the last bit."""
    w = shape_workload(72, 52, 34, 3, 12, None)
    with make_solver(B, w) as s:
        s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        rhs_d = to_dev(torch_cuda, w.rhs)
        p_d = torch_cuda.zeros_like(rhs_d)
        s.sweeps(rhs_d, p_d, w.omega, 3)
        vals = {s.residual(rhs_d, p_d) for _ in range(5)}
    assert len(vals) == 1


def test_zero_rhs_and_state_errors(torch_cuda, B):
    w = shape_workload(16, 12, 20, 0, 0, None)
    with make_solver(B, w) as s:
        rhs_d = torch_cuda.zeros(w.nz, w.ny, w.nx, dtype=torch_cuda.float64, device="cuda")
        p_d = torch_cuda.zeros_like(rhs_d)
        with pytest.raises(B.PsError) as e:
            s.solve(rhs_d, p_d, 1.5, 1, 0.0)          # before set_fraction
        assert e.value.code == B.PS_ESTATE
        s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
        info = s.solve(rhs_d, p_d, 1.5, 3, 1e-8)      # rhs = 0, p = 0: residual 0, rel := abs
        assert info.res_abs == 0.0 and info.res_rel == 0.0 and info.rhs_norm == 0.0
        assert info.converged and float(p_d.abs().max()) == 0.0
        for bad_omega in (0.0, 2.0, -1.0, float("nan")):
            with pytest.raises(B.PsError) as e:
                s.solve(rhs_d, p_d, bad_omega, 1, 0.0)
            assert e.value.code == B.PS_EINVAL
        with pytest.raises(B.PsError):
            s.solve(rhs_d, p_d, 1.5, -1, 0.0)
        with pytest.raises(B.PsError):
            s.set_fraction(to_dev(torch_cuda, w.F), -1.0, 1.2)
        assert s.launch_count() > 0


def test_solve_host_end_to_end(torch_cuda, B, ora):
    """ps_solve_host: host buffers in, host p out -- same numbers as the device-pointer path."""
    w = wl.make_config(1)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    io = ora.solve(coef, w.rhs, p_ora, w.omega, 40, 0.0)
    p = np.zeros_like(w.rhs)
    with make_solver(B, w) as s:
        ig = s.solve_host(w.F, w.rho_l, w.rho_g, w.rhs, p, w.omega, 40, 0.0)
    assert_p_parity(p, p_ora, "solve_host")
    assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel


def test_non_default_stream_and_library_workspace(torch_cuda, B, ora):
    w = shape_workload(40, 36, 24, 2, 8, None)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p_ora, w.omega, 4)
    s = B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, workspace=False)   # cudaMalloc'd ws
    st = torch_cuda.cuda.Stream()
    F_d, rhs_d = to_dev(torch_cuda, w.F), to_dev(torch_cuda, w.rhs)
    p_d = torch_cuda.zeros_like(rhs_d)
    torch_cuda.cuda.synchronize()
    with torch_cuda.cuda.stream(st):
        s.set_fraction(F_d, w.rho_l, w.rho_g)
        s.sweeps(rhs_d, p_d, w.omega, 4)
    st.synchronize()
    assert_p_parity(p_d.cpu().numpy(), p_ora, "side stream")
    s.close()


# ---------------------------------------------------------------- NEXT-4: on-the-fly coefficients
@pytest.mark.parametrize("shape", [(40, 36, 24, 2, 8, None), (72, 52, 34, 3, 12, (1 / 72, 1 / 60, 1 / 50)),
                                   (132, 20, 10, 0, 0, None), (64, 16, 8, 0, 0, None),
                                   (2, 1, 2, 0, 0, None)])
def test_on_the_fly_coefficients_bitwise(torch_cuda, B, ora, shape):
    """PS_KERNEL_FUSED_OTF rebuilds ax, ay, az from rho inside the sweep:
    p must equal the oracle's (which sweeps with stored O2 coefficients) to the last bit, and the
    variant must be chosen before ps_set_fraction (PS_ESTATE otherwise)."""
    w = shape_workload(*shape)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p_ora, w.omega, 7)
    F_d, rhs_d = to_dev(torch_cuda, w.F), to_dev(torch_cuda, w.rhs)
    with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(F_d, w.rho_l, w.rho_g)
        s.set_kernel(B.KERNEL_FUSED_OTF)
        p_d = torch_cuda.zeros_like(rhs_d)
        with pytest.raises(B.PsError) as e:
            s.sweeps(rhs_d, p_d, w.omega, 1)          # rho was not stored by that set_fraction
        assert e.value.code == B.PS_ESTATE
        with pytest.raises(B.PsError):
            s.set_tuning(2, 0)                        # one row per thread only
        s.set_fraction(F_d, w.rho_l, w.rho_g)
        s.sweeps(rhs_d, p_d, w.omega, 7)
        assert_p_parity(p_d.cpu().numpy(), p_ora, "fused_otf x7")
        info = s.solve(rhs_d, p_d, w.omega, 0, 0.0)   # norms still come from the stored coefficients
        assert abs(info.res_rel - ora.residual(coef, w.rhs, p_ora)[1]) <= NORM_TOL * info.res_rel


# ---------------------------------------------------------------- tile-geometry edge cases
@pytest.mark.parametrize("nx,ny,nz", [
    (64, 16, 4),      # exactly one box: both walls of x and of y inside one tile
    (66, 17, 4),      # one pair / one row more than a box: two tiles each way, ring columns live
    (62, 30, 6),      # two wall tiles of the maximum height (15 rows each)
    (128, 31, 4),     # two full 64-column tiles; 15 + 16 rows -> three row tiles
    (130, 44, 4),     # 64 + 64 + 2 columns: a one-pair last tile; 15 + 14 + 15 rows
    (186, 45, 6),     # three ragged x tiles; one row more than 15 + 14 + 15
    (256, 20, 8),     # four full tiles across (the paper-scale width)
    (2, 2, 2),        # smallest grid the fused kernels take
])
def test_fused_tile_edges_bitwise(torch_cuda, B, ora, nx, ny, nz):
    """Fused kernels (stored and on-the-fly coefficients) on grids whose sizes sit on the tile
    capacities (64 owned columns per tile, 15 / 14 rows per wall / middle tile), with the balanced
    split and with 1 and 2 z chunks per tile: p bitwise equal to the oracle after 3 sweeps."""
    w = shape_workload(nx, ny, nz, 0, 0, None, seed=nx + ny)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p0 = wl.noise_rhs(w.nx, w.ny, w.nz, 5)
    p_ora = p0.copy()
    ora.sweep(coef, w.rhs, p_ora, w.omega, 3)
    for kernel in (B.KERNEL_FUSED, B.KERNEL_FUSED_OTF):
        for chunks in (0, 1, 2):
            if chunks > nz // 2:
                continue
            with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
                s.set_kernel(kernel)
                s.set_tuning(1, chunks)
                s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
                p_d = to_dev(torch_cuda, p0)
                s.sweeps(to_dev(torch_cuda, w.rhs), p_d, w.omega, 3)
                assert_p_parity(p_d.cpu().numpy(), p_ora, f"{nx}x{ny}x{nz} kernel {kernel} chunks {chunks}")


def test_wide_dynamic_range_bitwise(torch_cuda, B, ora):
    """IEEE division and rounding outside the comfortable range: |rhs| = 2^k with k drawn from
    [-1070, 400] (subnormal numerators up to huge ones) sends many quotients of the update through
    the GPU's division slow path; every variant must still equal the host's correctly rounded
    arithmetic bit for bit."""
    nx, ny, nz = 40, 36, 24
    w = shape_workload(nx, ny, nz, 2, 8, None)
    rng = np.random.default_rng(2104)
    k = rng.integers(-1070, 401, size=(nz, ny, nx))
    rhs = np.ldexp(rng.choice([-1.0, 1.0], size=k.shape), k)
    assert np.isfinite(rhs).all() and (np.abs(rhs[rhs != 0]) < 2.3e-308).any()   # has subnormals
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    for nsweeps in (1, 2):                        # after 1 sweep red cells still hold subnormals
        p_ora = np.zeros_like(rhs)
        ora.sweep(coef, rhs, p_ora, w.omega, nsweeps)
        assert np.isfinite(p_ora).all()
        if nsweeps == 1:
            assert np.count_nonzero((np.abs(p_ora) < 2.3e-308) & (p_ora != 0)) > 100
        for variant in variants_for(B, w):
            with make_solver(B, w, variant) as s:
                s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
                p_d = torch_cuda.zeros(nz, ny, nx, dtype=torch_cuda.float64, device="cuda")
                s.sweeps(to_dev(torch_cuda, rhs), p_d, w.omega, nsweeps)
                p_gpu = p_d.cpu().numpy()
                assert int(np.count_nonzero(p_gpu != p_ora)) == 0, f"variant {variant} x{nsweeps}"


def test_subnormal_coefficients_bitwise(torch_cuda, B, ora):
    """Densities near the top of the fp64 range with h = 1 give SUBNORMAL face coefficients
    (2 / 1.6e308): the coefficient quotients of the on-the-fly variant leave the fast path of the
    division (its guards ask for a normal quotient) and must fall back to the plain quotient; the
    stored-coefficient kernels get the same subnormals from ps_set_fraction.  All equal the
    oracle bit for bit."""
    nx, ny, nz = 40, 20, 8
    w = wl.make_custom(nx, ny, nz, 0, 0, 3, dx=1.0, dy=1.0, dz=1.0)
    w.F = wl.random_fraction(nx, ny, nz, 3)
    rho_l, rho_g = 8.0e307, 4.0e307
    coef = ora.coefficients(w.F, rho_l, rho_g, 1.0, 1.0, 1.0)
    sub = (coef[2] > 0.0) & (coef[2] < 2.2e-308)
    assert coef[2].min() > 0.0 and sub.mean() > 0.5                # most az are subnormal
    p_ora = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p_ora, w.omega, 2)
    assert np.isfinite(p_ora).all()
    for kernel in (B.KERNEL_TWOPASS, B.KERNEL_FUSED, B.KERNEL_FUSED_OTF):
        with B.PoissonSolver(nx, ny, nz, 1.0, 1.0, 1.0) as s:
            s.set_kernel(kernel)
            s.set_fraction(to_dev(torch_cuda, w.F), rho_l, rho_g)
            if kernel == B.KERNEL_FUSED:
                gz = s.export_coefficients()[2].cpu().numpy()
                assert np.array_equal(gz, coef[2])
            p_d = torch_cuda.zeros(nz, ny, nx, dtype=torch_cuda.float64, device="cuda")
            s.sweeps(to_dev(torch_cuda, w.rhs), p_d, w.omega, 2)
            assert int(np.count_nonzero(p_d.cpu().numpy() != p_ora)) == 0, f"kernel {kernel}"


def test_long_run_repeatable_across_fused_variants(torch_cuda, B):
    """2,000 sweeps on config 3 (18 tiles, every SM busy): the fused kernel twice with the balanced
    split, without dependent launches and pacing, with 5 and with 9 z chunks per tile under other
    pacing windows, and the on-the-fly variant all end on the same bits -- a rare miss in the mbarrier protocol (a stage read before it landed, a red value read
    before it was written) would show up as a difference between runs."""
    w = wl.make_config(3)
    F_d, rhs_d = to_dev(torch_cuda, w.F), to_dev(torch_cuda, w.rhs)
    ref = None
    # (kernel, rows per thread, z chunks, dependent launches, pacing window; -1 = library default)
    for kernel, rpt, chunks, dep, window in [
            (B.KERNEL_FUSED, 1, 0, -1, -1), (B.KERNEL_FUSED, 1, 0, -1, -1),
            (B.KERNEL_FUSED, 1, 0, 0, 0), (B.KERNEL_FUSED, 1, 5, 1, 1), (B.KERNEL_FUSED, 1, 9, 0, 8),
            (B.KERNEL_FUSED_OTF, 1, 0, -1, -1)]:
        with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
            s.set_kernel(kernel)
            s.set_tuning(rpt, chunks)
            s.set_launch_options(dep, window)
            s.set_fraction(F_d, w.rho_l, w.rho_g)
            p_d = torch_cuda.zeros_like(rhs_d)
            s.sweeps(rhs_d, p_d, w.omega, 2000)
            if ref is None:
                ref = p_d.clone()
            else:
                assert torch_cuda.equal(p_d, ref), (kernel, rpt, chunks, dep, window)


def test_unaligned_pointers_are_rejected_everywhere(torch_cuda, B, ora):
    """Every *_dev field pointer must be 16-byte aligned (include/ps_poisson.h "Pointers").  A
    contiguous view at an odd storage offset is 8-byte aligned only: each entry point must return
    PS_EINVAL before launching anything (a 16-byte access or a TMA map on such a pointer would
    fault and poison the CUDA context), the binding must refuse such a tensor, and the context must
    work as before afterwards."""
    import ctypes
    w = shape_workload(40, 36, 24, 2, 8, None)
    n = w.nx * w.ny * w.nz
    shape = (w.nz, w.ny, w.nx)

    def odd(a=None):
        buf = torch_cuda.zeros(n + 1, dtype=torch_cuda.float64, device="cuda")
        v = buf[1:].view(shape)
        if a is not None:
            v.copy_(to_dev(torch_cuda, a))
        assert v.is_contiguous() and v.data_ptr() % 16 == 8
        return v

    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p_ora = np.zeros_like(w.rhs)
    ora.sweep(coef, w.rhs, p_ora, w.omega, 3)
    lib = B.load()
    ptr = lambda t: ctypes.c_void_p(t.data_ptr())
    for kernel in (B.KERNEL_TWOPASS, B.KERNEL_FUSED, B.KERNEL_RESIDENT, B.KERNEL_CLUSTER):
        with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
            s.set_kernel(kernel)                         # 40 x 36 x 24 fits one cluster
            F_d, rhs_d = to_dev(torch_cuda, w.F), to_dev(torch_cuda, w.rhs)
            p_d = torch_cuda.zeros_like(rhs_d)
            bad_F, bad_rhs, bad_p = odd(w.F), odd(w.rhs), odd()
            h = s._h
            assert lib.ps_set_fraction(h, ptr(bad_F), w.rho_l, w.rho_g) == B.PS_EINVAL
            s.set_fraction(F_d, w.rho_l, w.rho_g)
            s.mg_setup(levels=2)
            dbl = ctypes.c_double()
            for rhs_t, p_t in ((bad_rhs, p_d), (rhs_d, bad_p), (bad_rhs, bad_p)):
                assert lib.ps_sweeps(h, ptr(rhs_t), ptr(p_t), w.omega, 1) == B.PS_EINVAL
                assert lib.ps_half_sweep(h, ptr(rhs_t), ptr(p_t), w.omega, 0) == B.PS_EINVAL
                assert lib.ps_solve(h, ptr(rhs_t), ptr(p_t), w.omega, 1, 0.0, None) == B.PS_EINVAL
                assert lib.ps_residual(h, ptr(rhs_t), ptr(p_t), ctypes.byref(dbl), None, None) == B.PS_EINVAL
                assert lib.ps_mg_solve(h, ptr(rhs_t), ptr(p_t), 1, 0.0, None) == B.PS_EINVAL
                assert lib.ps_mg_residual_restrict(h, ptr(rhs_t), ptr(p_t), ptr(p_d)) == B.PS_EINVAL
            assert lib.ps_mg_prolong_add(h, ptr(rhs_d), ptr(bad_p)) == B.PS_EINVAL
            assert lib.ps_rhs_from_velocity(h, ptr(bad_p), ptr(p_d), ptr(p_d), 1e-3, ptr(rhs_d)) == B.PS_EINVAL
            assert lib.ps_correct_velocity(h, ptr(bad_p), 1e-3, ptr(p_d), ptr(p_d), ptr(p_d)) == B.PS_EINVAL
            assert lib.ps_face_divergence(h, ptr(p_d), ptr(p_d), ptr(p_d), ptr(bad_p), 1e-3, ptr(rhs_d)) == B.PS_EINVAL
            assert lib.ps_ssf_rhs(h, ptr(bad_F), ptr(F_d), 0.07, ptr(rhs_d)) == B.PS_EINVAL
            with pytest.raises(TypeError, match="16-byte"):
                s.sweeps(rhs_d, bad_p, w.omega, 1)
            assert float(bad_p.abs().max()) == 0.0 and float(p_d.abs().max()) == 0.0   # untouched
            s.sweeps(rhs_d, p_d, w.omega, 3)                      # the context is still healthy
            assert_p_parity(p_d.cpu().numpy(), p_ora, f"after rejected calls, kernel {kernel}")


def test_odd_check_interval_needs_no_copy_and_matches_oracle(torch_cuda, B, ora):
    """K odd: the fused kernels end every batch in the other ping-pong buffer; ps_solve takes the
    norm on whichever buffer holds the iterate and settles p once at the end.  Same stops, same p."""
    w = shape_workload(72, 52, 34, 3, 12, None)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    for K, max_sweeps, tol in [(7, 64, 1e-30), (3, 40, 0.5), (5, 23, 1e-30), (1, 9, 1e-30)]:
        p_ora = np.zeros_like(w.rhs)
        io = ora.solve(coef, w.rhs, p_ora, w.omega, max_sweeps, tol, check_interval=K)
        for kernel in (B.KERNEL_FUSED, B.KERNEL_FUSED_OTF, B.KERNEL_TWOPASS):
            with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
                s.set_kernel(kernel)
                s.set_check_interval(K)
                s.set_fraction(to_dev(torch_cuda, w.F), w.rho_l, w.rho_g)
                rhs_d = to_dev(torch_cuda, w.rhs)
                p_d = torch_cuda.zeros_like(rhs_d)
                ig = s.solve(rhs_d, p_d, w.omega, max_sweeps, tol)
                assert (ig.sweeps, ig.converged) == (io.sweeps, io.converged), (K, max_sweeps, tol)
                assert_p_parity(p_d.cpu().numpy(), p_ora, f"K={K} kernel {kernel}")
                assert abs(ig.res_rel - io.res_rel) <= NORM_TOL * io.res_rel
                assert s.residual(rhs_d, p_d)[1] == ig.res_rel    # p_dev holds what was measured


EDGE_SHAPES = [(64, 1, 8), (2, 1, 2), (66, 2, 4), (130, 1, 6), (4, 5, 256), (256, 3, 2), (62, 15, 4),
               (64, 16, 2), (128, 14, 2), (70, 29, 6), (2, 2, 2), (6, 1, 4), (68, 30, 12), (192, 17, 8)]


@pytest.mark.parametrize("shape", EDGE_SHAPES)
def test_edge_shapes_all_variants_and_default_multigrid(torch_cuda, B, ora, shape):
    """Degenerate and boundary shapes of the tilings: one row, one pair, exactly one box of rows,
    one row more or fewer than a tile, one column pair more than a tile, the smallest nz, a long
    thin duct -- every kernel variant the library accepts, 1 and 3 sweeps, and two default
    multigrid cycles (as many levels as the shape allows), all bitwise against the oracle."""
    nx, ny, nz = shape
    w = shape_workload(nx, ny, nz, 0, 0, None, seed=5)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    F_d, rhs_d = to_dev(torch_cuda, w.F), to_dev(torch_cuda, w.rhs)
    for nsweeps in (1, 3):
        p_ora = np.zeros_like(w.rhs)
        ora.sweep(coef, w.rhs, p_ora, w.omega, nsweeps)
        for variant in variants_for(B, w, tunings=((1, 0, -1, -1), (1, 1, 1, 2), (1, 2, 0, 0))):
            with make_solver(B, w, variant) as s:
                s.set_fraction(F_d, w.rho_l, w.rho_g)
                p_d = torch_cuda.zeros_like(rhs_d)
                s.sweeps(rhs_d, p_d, w.omega, nsweeps)
                assert_p_parity(p_d.cpu().numpy(), p_ora, f"{shape} variant {variant} x{nsweeps}")
    q_ora = np.zeros_like(w.rhs)
    ora.mg_solve(coef, w.rhs, q_ora, 2, 0.0, **B.MG_DEFAULTS)
    with make_solver(B, w) as s:
        s.set_fraction(F_d, w.rho_l, w.rho_g)
        s.mg_setup()
        q_d = torch_cuda.zeros_like(rhs_d)
        s.mg_solve(rhs_d, q_d, 2, 0.0)
        assert_p_parity(q_d.cpu().numpy(), q_ora, f"{shape} default multigrid")


# ---------------------------------------------------------------- bench.py's bandwidth probe
@pytest.mark.parametrize("reads", [1, 3, 5])
def test_stream_probe_adds_its_streams(torch_cuda, B, reads):
    """ps_stream_probe (the second roofline denominator of bench.py) reads every element of every
    stream and writes every output: ragged sizes, more and fewer elements than threads."""
    import ctypes
    torch = torch_cuda
    lib = B.load()
    for n, blocks in ((2, 1), (1026, 1), (100_000, 3), (3_000_002, 592)):
        src = torch.rand(reads * n, dtype=torch.float64, device="cuda")
        dst = torch.full((n + 2,), -1.0, dtype=torch.float64, device="cuda")
        rc = lib.ps_stream_probe(ctypes.c_void_p(src.data_ptr()), ctypes.c_void_p(dst.data_ptr()),
                                 n, reads, blocks, None)
        assert rc == B.PS_OK
        torch.cuda.synchronize()
        want = src[:n].clone()
        for r in range(1, reads):
            want += src[r * n:(r + 1) * n]
        assert torch.equal(dst[:n], want), (n, blocks)
        assert float(dst[n]) == -1.0 and float(dst[n + 1]) == -1.0
    assert lib.ps_stream_probe(None, None, 4, 5, 1, None) == B.PS_EINVAL
    assert B.stream_probe_gbs(1 << 22, 5, reps=2, warmup=1) > 0.0
