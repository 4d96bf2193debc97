"""Thin ctypes binding of include/ps_poisson.h -- argument marshalling only.

Every step of the path (coefficient build, sweeps, residual, norms) runs in the CUDA kernels
behind libps_poisson.so.  PyTorch is used for device memory and streams: arguments are CUDA
float64 tensors of shape (nz, ny, nx) (linear index n = i + nx*(j + ny*k)), handed over as raw
device pointers; the library enqueues on torch's current stream.

There is no CPU fallback: if the library is not built, `load()` raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

from . import build as _build

PS_OK, PS_EINVAL, PS_ESTATE, PS_ECUDA, PS_ENOMEM = 0, -1, -2, -3, -4
PS_ETOOBIG = -5
NOALLOC_MAX_CELLS = 1 << 28      # PS_NOALLOC_MAX_CELLS of include/ps_poisson.h
KERNEL_AUTO, KERNEL_TWOPASS, KERNEL_FUSED, KERNEL_RESIDENT, KERNEL_FUSED_OTF = 0, 1, 2, 3, 4
KERNEL_CLUSTER = 5
KERNEL_NAMES = {KERNEL_AUTO: "auto", KERNEL_TWOPASS: "twopass", KERNEL_FUSED: "fused",
                KERNEL_RESIDENT: "resident", KERNEL_FUSED_OTF: "fused_otf",
                KERNEL_CLUSTER: "cluster"}

# Multigrid parameters `mg_setup()` uses when none are given (chosen among ~700
# settings scanned on the five configs, profiles/r02_mg_tuning.md): V(0,2) -- no pre-smoothing, 2
# post-smoothing sweeps on the finest level at omega_s = 1.4 --, 48 sweeps at omega_c = 1.97 on
# every coarser level, 10 on the coarsest of 6: 16-21 cycles to 1e-8 on all five configs.
# omega_c = 1.98 is ~10 % faster and 1.985 still converges on every config and seed tried; 1.99 does
# not on all.  The one place they are written down: bench.py, report.py and the parity tests take
# them from here.
# stall_cycles / omega_c_step: the safeguard M7 -- the defaults are tuned on isotropic bubbly ducts
# and omega_c = 1.97 diverges on 4:1:1 or 1:2:4 spacing; three cycles in a row without a new best
# norm lower omega_c by 0.05 (tests/test_mg_heldout_gpu.py, profiles/r03_mg_heldout.md).
MG_DEFAULTS = dict(levels=6, nu1=0, nu2=2, coarse_sweeps=10, gamma=1, omega_s=1.4, omega_c=1.97,
                   nu_growth=24, nu_max=48, nu_max_deep=48, stall_cycles=3, omega_c_step=0.05)

# every symbol include/ps_poisson.h declares (tests check the library exports each one)
SYMBOLS = ("ps_create", "ps_destroy", "ps_workspace_bytes", "ps_set_workspace", "ps_set_stream",
           "ps_set_check_interval", "ps_set_kernel", "ps_get_kernel", "ps_set_tuning",
           "ps_get_tuning", "ps_set_launch_options", "ps_get_launch_options", "ps_fused_plan",
           "ps_set_fraction",
           "ps_export_coefficients", "ps_solve", "ps_sweeps", "ps_half_sweep", "ps_residual",
           "ps_solve_host", "ps_host_staging_bytes", "ps_set_host_staging", "ps_enable_timing",
           "ps_checked_build", "ps_debug_read", "ps_debug_sabotage", "ps_timing", "ps_launch_count", "ps_strerror",
           "ps_mg_workspace_bytes", "ps_mg_set_workspace", "ps_mg_setup", "ps_mg_levels", "ps_mg_solve", "ps_mg_export_coarse",
           "ps_mg_residual_restrict", "ps_mg_prolong_add", "ps_rhs_from_velocity",
           "ps_correct_velocity", "ps_face_divergence", "ps_ssf_rhs", "ps_residual_noalloc", "ps_stream_probe")


class PsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libps_poisson: {msg} (code {code})")
        self.code = code


class _MgParams(ctypes.Structure):
    _fields_ = [("levels", ctypes.c_int), ("nu1", ctypes.c_int), ("nu2", ctypes.c_int),
                ("nu_growth", ctypes.c_int), ("nu_max", ctypes.c_int),
                ("coarse_sweeps", ctypes.c_int), ("gamma", ctypes.c_int),
                ("omega_s", ctypes.c_double), ("omega_c", ctypes.c_double),
                ("nu_max_deep", ctypes.c_int), ("stall_cycles", ctypes.c_int),
                ("omega_c_step", ctypes.c_double)]


class _Info(ctypes.Structure):
    _fields_ = [("sweeps", ctypes.c_int), ("converged", ctypes.c_int),
                ("res_abs", ctypes.c_double), ("res_rel", ctypes.c_double),
                ("rhs_norm", ctypes.c_double)]


@dataclass
class Info:
    sweeps: int
    converged: bool
    res_abs: float
    res_rel: float
    rhs_norm: float


_lib = None


def load(path: str | None = None) -> ctypes.CDLL:
    """dlopen libps_poisson.so and declare the prototypes.  Raises if it is not built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or _build.LIB
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: run `python -m paper_2104_01636_b200.build` "
                           "(the CUDA extension is the only compute path; there is no fallback)")
    import torch  # noqa: F401  -- first, so that the library binds the libcudart torch loaded
    lib = ctypes.CDLL(path)
    vp, i, d, dp = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.POINTER(ctypes.c_double)
    lib.ps_create.argtypes = [ctypes.POINTER(vp), i, i, i, d, d, d]
    lib.ps_destroy.argtypes = [vp]
    lib.ps_workspace_bytes.argtypes = [vp]
    lib.ps_workspace_bytes.restype = ctypes.c_size_t
    lib.ps_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    lib.ps_set_stream.argtypes = [vp, vp]
    lib.ps_set_check_interval.argtypes = [vp, i]
    lib.ps_set_kernel.argtypes = [vp, i]
    lib.ps_get_kernel.argtypes = [vp]
    lib.ps_set_tuning.argtypes = [vp, i, i]
    ip = ctypes.POINTER(ctypes.c_int)
    lib.ps_get_tuning.argtypes = [vp, ip, ip, ip, ip, ip]
    lib.ps_set_launch_options.argtypes = [vp, i, i]
    lib.ps_get_launch_options.argtypes = [vp, ip, ip]
    lib.ps_fused_plan.argtypes = [i, i, i, i, i, ip, i, ip, i, ip, ip, ip]
    lib.ps_set_fraction.argtypes = [vp, vp, d, d]
    lib.ps_export_coefficients.argtypes = [vp, vp, vp, vp]
    lib.ps_solve.argtypes = [vp, vp, vp, d, i, d, ctypes.POINTER(_Info)]
    lib.ps_sweeps.argtypes = [vp, vp, vp, d, i]
    lib.ps_half_sweep.argtypes = [vp, vp, vp, d, i]
    lib.ps_residual.argtypes = [vp, vp, vp, dp, dp, dp]
    lib.ps_solve_host.argtypes = [vp, vp, d, d, vp, vp, d, i, d, ctypes.POINTER(_Info)]
    lib.ps_enable_timing.argtypes = [vp, i]
    lib.ps_host_staging_bytes.argtypes = [vp]
    lib.ps_host_staging_bytes.restype = ctypes.c_size_t
    lib.ps_set_host_staging.argtypes = [vp, vp, ctypes.c_size_t]
    llp = ctypes.POINTER(ctypes.c_longlong)
    lib.ps_timing.argtypes = [vp, dp, llp, llp]
    lib.ps_mg_workspace_bytes.argtypes = [vp, i]
    lib.ps_mg_workspace_bytes.restype = ctypes.c_size_t
    lib.ps_mg_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    lib.ps_checked_build.argtypes = []
    lib.ps_debug_read.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong)]
    lib.ps_debug_sabotage.argtypes = [vp, i]
    lib.ps_launch_count.argtypes = [vp]
    lib.ps_launch_count.restype = ctypes.c_longlong
    lib.ps_mg_setup.argtypes = [vp, ctypes.POINTER(_MgParams)]
    lib.ps_mg_levels.argtypes = [vp]
    lib.ps_mg_solve.argtypes = [vp, vp, vp, i, d, ctypes.POINTER(_Info)]
    lib.ps_mg_export_coarse.argtypes = [vp, i, vp, vp, vp]
    lib.ps_mg_residual_restrict.argtypes = [vp, vp, vp, vp]
    lib.ps_mg_prolong_add.argtypes = [vp, vp, vp]
    lib.ps_rhs_from_velocity.argtypes = [vp, vp, vp, vp, d, vp]
    lib.ps_correct_velocity.argtypes = [vp, vp, d, vp, vp, vp]
    lib.ps_face_divergence.argtypes = [vp, vp, vp, vp, vp, d, vp]
    lib.ps_ssf_rhs.argtypes = [vp, vp, vp, d, vp]
    lib.ps_residual_noalloc.argtypes = [i, i, i, vp, vp, vp, vp, vp, vp, vp]
    lib.ps_stream_probe.argtypes = [vp, vp, ctypes.c_size_t, i, i, vp]
    lib.ps_strerror.argtypes = [i]
    lib.ps_strerror.restype = ctypes.c_char_p
    if path == _build.LIB:
        _lib = lib
    return lib


def _check(lib, rc: int):
    if rc != PS_OK:
        raise PsError(rc, lib.ps_strerror(rc).decode())


def _dev_ptr(t, shape, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64
            and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
        raise TypeError(f"{name}: expected a contiguous CUDA float64 tensor of shape {tuple(shape)}")
    if t.data_ptr() % 16:
        raise TypeError(f"{name}: device pointer must be 16-byte aligned (a view with an odd "
                        "storage offset is not; make it contiguous at an even offset)")
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(a, shape, name):
    import numpy as np
    import torch
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or tuple(a.shape) != tuple(shape):
            raise TypeError(f"{name}: expected a contiguous host float64 tensor of shape {tuple(shape)}")
        return ctypes.c_void_p(a.data_ptr())
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
            and tuple(a.shape) == tuple(shape)):
        raise TypeError(f"{name}: expected a C-contiguous float64 array of shape {tuple(shape)}")
    return ctypes.c_void_p(a.ctypes.data)


def residual_noalloc(ax, ay, az, rhs, p, out, lib=None):
    """ps_residual_noalloc: the three numbers of `PoissonSolver.residual` written to the caller's
    device tensor `out` (3 float64: ||r||, ||r||/||rhs||, ||rhs||), with the reduction's scratch
    taken from a fixed array inside the library instead of a context's workspace.  For callers
    that must not allocate device memory in the call -- a flow solver whose memory pool already
    owns the board, where a cudaMalloc can fail or stalls every stream of the device.  Neither
    this wrapper nor the library allocates: `out` is the caller's.  Enqueued on torch's current
    stream, not synchronised; calls that may overlap on one GPU must be ordered by the caller (they
    share the array).  Grids above NOALLOC_MAX_CELLS raise PsError(PS_ETOOBIG)."""
    import torch
    lib = lib if lib is not None else load()
    nz, ny, nx = rhs.shape
    ptrs = [_dev_ptr(t, rhs.shape, n) for t, n in
            ((ax, "ax"), (ay, "ay"), (az, "az"), (rhs, "rhs"), (p, "p"))]
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64
            and out.is_contiguous() and out.numel() >= 3):
        raise TypeError("out: expected a contiguous CUDA float64 tensor of at least 3 elements")
    s = torch.cuda.current_stream().cuda_stream
    _check(lib, lib.ps_residual_noalloc(nx, ny, nz, *ptrs, ctypes.c_void_p(s),
                                        ctypes.c_void_p(out.data_ptr())))
    return out


def stream_probe_gbs(n: int, reads: int = 5, blocks_per_sm: int = 4, reps: int = 20,
                     warmup: int = 3) -> float:
    """GB/s (read + written bytes over CUDA-event time, mean of `reps` launches after `warmup`)
    of ps_stream_probe on n doubles per stream: the library's own streaming kernel with the fused
    sweep's 5-read / 1-write mix (reads=5) or a plain copy (reads=1).  A measured denominator for
    bench.py's roofline beside the device-copy figure of MEASURED_PEAKS.json."""
    import torch
    lib = load()
    n -= n & 1
    src = torch.rand(reads * n, dtype=torch.float64, device="cuda")
    dst = torch.empty(n, dtype=torch.float64, device="cuda")
    blocks = blocks_per_sm * torch.cuda.get_device_properties(0).multi_processor_count
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    a, b = ctypes.c_void_p(src.data_ptr()), ctypes.c_void_p(dst.data_ptr())
    for _ in range(warmup):
        _check(lib, lib.ps_stream_probe(a, b, n, reads, blocks, st))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        _check(lib, lib.ps_stream_probe(a, b, n, reads, blocks, st))
    e1.record()
    torch.cuda.synchronize()
    if reads > 1:      # the probe really added the streams up
        want = src.view(reads, n)[:, :1024].sum(0)
        assert torch.allclose(dst[:1024], want, rtol=1e-14, atol=0)
    return (reads + 1) * 8.0 * n * reps / (e0.elapsed_time(e1) * 1e-3) / 1e9


def fused_plan(nx: int, ny: int, nz: int, sm_count: int = 148, z_chunks: int = 0):
    """(tiles, items) of the fused kernel's work split (host only): tiles as (xs, xe, ys, ye),
    items as (cta, tile, ks, ke) in launch order."""
    lib = load()
    n = [ctypes.c_int() for _ in range(3)]
    _check(lib, lib.ps_fused_plan(nx, ny, nz, sm_count, z_chunks, None, 0, None, 0,
                                  *[ctypes.byref(x) for x in n]))
    nt, ni = n[0].value, n[1].value
    tiles, items = (ctypes.c_int * (4 * nt))(), (ctypes.c_int * (4 * ni))()
    _check(lib, lib.ps_fused_plan(nx, ny, nz, sm_count, z_chunks, tiles, nt, items, ni,
                                  *[ctypes.byref(x) for x in n]))
    return ([tuple(tiles[4 * q:4 * q + 4]) for q in range(nt)],
            [tuple(items[4 * q:4 * q + 4]) for q in range(ni)])


class PoissonSolver:
    """ps_create / ps_set_fraction / ps_solve / ps_residual with the names of the C ABI."""

    def __init__(self, nx: int, ny: int, nz: int, dx: float, dy: float, dz: float,
                 workspace: bool = True, lib=None):
        import torch
        self._lib = lib if lib is not None else load()
        self._h = ctypes.c_void_p()
        self.nx, self.ny, self.nz = nx, ny, nz
        self.shape = (nz, ny, nx)
        _check(self._lib, self._lib.ps_create(ctypes.byref(self._h), nx, ny, nz, dx, dy, dz))
        self._ws = self._mg_ws = self._st_ws = None
        self._torch_owns = workspace
        if workspace:      # torch owns the device memory (north_star: "PyTorch ... device memory")
            nbytes = self._lib.ps_workspace_bytes(self._h)
            self._ws, base = self._block(nbytes)
            _check(self._lib, self._lib.ps_set_workspace(self._h, base, nbytes))

    @staticmethod
    def _block(nbytes: int):
        """A torch-owned device block and its 256-byte aligned base pointer."""
        import torch
        t = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        return t, ctypes.c_void_p((t.data_ptr() + 255) // 256 * 256)

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.ps_destroy(self._h)
            self._h = ctypes.c_void_p()
        self._ws = self._mg_ws = self._st_ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _sync_stream(self):
        import torch
        s = torch.cuda.current_stream().cuda_stream
        _check(self._lib, self._lib.ps_set_stream(self._h, ctypes.c_void_p(s)))

    # -- options
    def set_check_interval(self, K: int):
        _check(self._lib, self._lib.ps_set_check_interval(self._h, K))

    def set_kernel(self, variant: int):
        _check(self._lib, self._lib.ps_set_kernel(self._h, variant))

    def get_kernel(self) -> int:
        return self._lib.ps_get_kernel(self._h)

    def set_tuning(self, rows_per_thread: int = 0, z_chunks: int = 0):
        _check(self._lib, self._lib.ps_set_tuning(self._h, rows_per_thread, z_chunks))

    def get_tuning(self):
        """(rows_per_thread, z_chunks, tiles, ctas, items) of the fused kernel's launch geometry."""
        v = [ctypes.c_int() for _ in range(5)]
        _check(self._lib, self._lib.ps_get_tuning(self._h, *[ctypes.byref(x) for x in v]))
        return tuple(x.value for x in v)

    def set_launch_options(self, dependent_launch: int = -1, pace_window: int = -1):
        """Fused kernel: dependent launches (0/1) and the pacing window (0 = off); -1 leaves the
        choice to the library."""
        _check(self._lib, self._lib.ps_set_launch_options(self._h, dependent_launch, pace_window))

    def get_launch_options(self):
        v = [ctypes.c_int() for _ in range(2)]
        _check(self._lib, self._lib.ps_get_launch_options(self._h, *[ctypes.byref(x) for x in v]))
        return tuple(x.value for x in v)

    def workspace_bytes(self) -> int:
        return self._lib.ps_workspace_bytes(self._h)

    def enable_timing(self, on: bool = True):
        _check(self._lib, self._lib.ps_enable_timing(self._h, int(on)))

    def timing(self):
        """(sweep_ms, sweep_launches, sweeps) accumulated since the last call; synchronises the
        stream."""
        ms, n, sw = ctypes.c_double(), ctypes.c_longlong(), ctypes.c_longlong()
        _check(self._lib, self._lib.ps_timing(self._h, ctypes.byref(ms), ctypes.byref(n),
                                              ctypes.byref(sw)))
        return ms.value, n.value, sw.value

    def launch_count(self) -> int:
        return self._lib.ps_launch_count(self._h)

    def debug_read(self):
        """Violation record of the self-checking build (all zero in the product build)."""
        out = (ctypes.c_ulonglong * 8)()
        _check(self._lib, self._lib.ps_debug_read(self._h, out))
        return list(out)

    # -- the path
    def set_fraction(self, F, rho_l: float, rho_g: float):
        self._sync_stream()
        _check(self._lib, self._lib.ps_set_fraction(self._h, _dev_ptr(F, self.shape, "F"),
                                                    rho_l, rho_g))

    def export_coefficients(self):
        import torch
        self._sync_stream()
        out = [torch.empty(self.shape, dtype=torch.float64, device="cuda") for _ in range(3)]
        _check(self._lib, self._lib.ps_export_coefficients(
            self._h, *[ctypes.c_void_p(t.data_ptr()) for t in out]))
        return tuple(out)

    def solve(self, rhs, p, omega: float, max_sweeps: int, tol: float) -> Info:
        self._sync_stream()
        info = _Info()
        _check(self._lib, self._lib.ps_solve(self._h, _dev_ptr(rhs, self.shape, "rhs"),
                                             _dev_ptr(p, self.shape, "p"), omega, max_sweeps,
                                             tol, ctypes.byref(info)))
        return Info(info.sweeps, bool(info.converged), info.res_abs, info.res_rel, info.rhs_norm)

    def sweeps(self, rhs, p, omega: float, n: int):
        self._sync_stream()
        _check(self._lib, self._lib.ps_sweeps(self._h, _dev_ptr(rhs, self.shape, "rhs"),
                                              _dev_ptr(p, self.shape, "p"), omega, n))

    def half_sweep(self, rhs, p, omega: float, colour: int):
        self._sync_stream()
        _check(self._lib, self._lib.ps_half_sweep(self._h, _dev_ptr(rhs, self.shape, "rhs"),
                                                  _dev_ptr(p, self.shape, "p"), omega, colour))

    def residual(self, rhs, p):
        """(res_abs, res_rel, rhs_norm)"""
        self._sync_stream()
        ra, rr, bn = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        _check(self._lib, self._lib.ps_residual(self._h, _dev_ptr(rhs, self.shape, "rhs"),
                                                _dev_ptr(p, self.shape, "p"), ctypes.byref(ra),
                                                ctypes.byref(rr), ctypes.byref(bn)))
        return ra.value, rr.value, bn.value

    # -- multigrid acceleration
    def mg_setup(self, levels: int | None = None, nu1: int | None = None, nu2: int | None = None,
                 coarse_sweeps: int | None = None, gamma: int | None = None,
                 omega_s: float | None = None, nu_growth: int | None = None,
                 nu_max: int | None = None, omega_c: float | None = None,
                 nu_max_deep: int | None = None, stall_cycles: int | None = None,
                 omega_c_step: float | None = None) -> int:
        """Build the level hierarchy from the current coefficients; returns the levels in use.
        With no arguments: MG_DEFAULTS.  Any argument given replaces its default, except that
        omega_c follows an explicitly given omega_s when it is not given itself (one relaxation
        factor on every level), and nu_max_deep an explicitly given nu_max (one cap on every
        level)."""
        self._sync_stream()
        if omega_c is None and omega_s is not None:
            omega_c = omega_s
        if nu_max_deep is None and nu_max is not None:
            nu_max_deep = nu_max
        given = dict(levels=levels, nu1=nu1, nu2=nu2, coarse_sweeps=coarse_sweeps, gamma=gamma,
                     omega_s=omega_s, omega_c=omega_c, nu_growth=nu_growth, nu_max=nu_max,
                     nu_max_deep=nu_max_deep, stall_cycles=stall_cycles,
                     omega_c_step=omega_c_step)
        q = dict(MG_DEFAULTS)
        q.update({k: v for k, v in given.items() if v is not None})
        levels = q["levels"]
        prm = _MgParams(q["levels"], q["nu1"], q["nu2"], q["nu_growth"], q["nu_max"],
                        q["coarse_sweeps"], q["gamma"], q["omega_s"], q["omega_c"],
                        q["nu_max_deep"], q["stall_cycles"], q["omega_c_step"])
        if self._torch_owns:               # the level memory is a torch allocation too
            need = self._lib.ps_mg_workspace_bytes(self._h, levels)
            if need and (self._mg_ws is None or self._mg_ws[0].numel() < need + 256):
                self._mg_ws = self._block(need)
                _check(self._lib, self._lib.ps_mg_set_workspace(self._h, self._mg_ws[1], need))
        _check(self._lib, self._lib.ps_mg_setup(self._h, ctypes.byref(prm)))
        return self._lib.ps_mg_levels(self._h)

    def mg_solve(self, rhs, p, max_cycles: int, tol: float) -> Info:
        """Multigrid cycles in place on p; Info.sweeps holds the number of cycles."""
        self._sync_stream()
        info = _Info()
        _check(self._lib, self._lib.ps_mg_solve(self._h, _dev_ptr(rhs, self.shape, "rhs"),
                                                _dev_ptr(p, self.shape, "p"), max_cycles, tol,
                                                ctypes.byref(info)))
        return Info(info.sweeps, bool(info.converged), info.res_abs, info.res_rel, info.rhs_norm)

    def _coarse_shape(self, level: int = 1):
        nz, ny, nx = self.shape
        return (nz >> level, ny >> level, nx >> level)

    def mg_export_coarse(self, level: int = 1):
        import torch
        self._sync_stream()
        out = [torch.empty(self._coarse_shape(level), dtype=torch.float64, device="cuda")
               for _ in range(3)]
        _check(self._lib, self._lib.ps_mg_export_coarse(
            self._h, level, *[ctypes.c_void_p(t.data_ptr()) for t in out]))
        return tuple(out)

    def mg_residual_restrict(self, rhs, p):
        import torch
        self._sync_stream()
        rc = torch.empty(self._coarse_shape(1), dtype=torch.float64, device="cuda")
        _check(self._lib, self._lib.ps_mg_residual_restrict(
            self._h, _dev_ptr(rhs, self.shape, "rhs"), _dev_ptr(p, self.shape, "p"),
            ctypes.c_void_p(rc.data_ptr())))
        return rc

    def mg_prolong_add(self, ec, p):
        self._sync_stream()
        _check(self._lib, self._lib.ps_mg_prolong_add(
            self._h, _dev_ptr(ec, self._coarse_shape(1), "ec"), _dev_ptr(p, self.shape, "p")))

    # -- steps 10-12 of the time step around the solve
    def rhs_from_velocity(self, ux, uy, uz, dt: float, rhs=None):
        import torch
        self._sync_stream()
        if rhs is None:
            rhs = torch.empty(self.shape, dtype=torch.float64, device="cuda")
        _check(self._lib, self._lib.ps_rhs_from_velocity(
            self._h, _dev_ptr(ux, self.shape, "ux"), _dev_ptr(uy, self.shape, "uy"),
            _dev_ptr(uz, self.shape, "uz"), dt, _dev_ptr(rhs, self.shape, "rhs")))
        return rhs

    def correct_velocity(self, p, dt: float, ux, uy, uz):
        self._sync_stream()
        _check(self._lib, self._lib.ps_correct_velocity(
            self._h, _dev_ptr(p, self.shape, "p"), dt, _dev_ptr(ux, self.shape, "ux"),
            _dev_ptr(uy, self.shape, "uy"), _dev_ptr(uz, self.shape, "uz")))

    def face_divergence(self, ux, uy, uz, p, dt: float):
        import torch
        self._sync_stream()
        div = torch.empty(self.shape, dtype=torch.float64, device="cuda")
        _check(self._lib, self._lib.ps_face_divergence(
            self._h, _dev_ptr(ux, self.shape, "ux"), _dev_ptr(uy, self.shape, "uy"),
            _dev_ptr(uz, self.shape, "uz"), _dev_ptr(p, self.shape, "p"), dt,
            _dev_ptr(div, self.shape, "div")))
        return div

    def ssf_rhs(self, F, kappa, sigma: float):
        """rhs of the sharp-surface-force pressure system."""
        import torch
        self._sync_stream()
        rhs = torch.empty(self.shape, dtype=torch.float64, device="cuda")
        _check(self._lib, self._lib.ps_ssf_rhs(
            self._h, _dev_ptr(F, self.shape, "F"), _dev_ptr(kappa, self.shape, "kappa"), sigma,
            _dev_ptr(rhs, self.shape, "rhs")))
        return rhs

    def solve_host(self, F, rho_l: float, rho_g: float, rhs, p, omega: float, max_sweeps: int,
                   tol: float) -> Info:
        """Whole path on HOST arrays (numpy or CPU torch tensors); p is updated in place."""
        self._sync_stream()
        if self._torch_owns and self._st_ws is None:
            need = self._lib.ps_host_staging_bytes(self._h)
            self._st_ws = self._block(need)
            _check(self._lib, self._lib.ps_set_host_staging(self._h, self._st_ws[1], need))
        info = _Info()
        _check(self._lib, self._lib.ps_solve_host(
            self._h, _host_ptr(F, self.shape, "F"), rho_l, rho_g,
            _host_ptr(rhs, self.shape, "rhs"), _host_ptr(p, self.shape, "p"), omega, max_sweeps,
            tol, ctypes.byref(info)))
        return Info(info.sweeps, bool(info.converged), info.res_abs, info.res_rel, info.rhs_norm)
