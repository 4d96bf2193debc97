"""compute-sanitizer record of the CUDA path (SURVEY.md §5 "sanitizers").

    python -m paper_2104_01636_b200.sanitize [--md FILE] [--tools memcheck,initcheck,racecheck,synccheck]
    python -m paper_2104_01636_b200.sanitize --target        (what the tools run; also fine alone)
    python -m paper_2104_01636_b200.sanitize --soak          (long-run repeatability, see soak())

The target drives every kernel family through the C ABI on two small grids -- BASELINE.json's
config 1 (32x32x64, one bubble) and a ragged multi-tile grid (186x46x8 with a random F in
{m/64}: several x and y tiles with ragged last tiles, 4-plane z chunks, an odd-sized coarse
level) -- : coefficient build, the two-pass, fused
(two launch geometries), on-the-fly and resident sweep kernels (each must reproduce the two-pass
kernel's p bit for bit), residual/norm reduction, one multigrid V-cycle (coarsening, fused
residual + restriction + norm, prolongation, smoothing on every level), the projection kernels
and the surface-tension right-hand side.  The driver runs it under `compute-sanitizer` once per
tool of --tools (this pool allows one tool per GPU-box call, so profiles/r02_sanitizer.md is four
calls, `--tools memcheck` ... `--tools synccheck`, each after a plain `--target` run had exited 0),
collects the ERROR SUMMARY lines and the first reports, and prints a markdown summary.  Needs the
B200: there is no CPU path.
"""
from __future__ import annotations

import argparse
import os
import re
import subprocess
import sys
import time

GRIDS = [(1, None), (0, (186, 46, 8))]          # (config, custom shape)


def target() -> int:
    import torch
    from . import binding as B, build, workload as wl
    build.build()
    B.load()
    assert torch.cuda.is_available(), "sanitize --target needs the GPU"
    ran = 0
    for cfg, shape in GRIDS:
        w = wl.make_config(cfg) if cfg else wl.make_custom(*shape, 0, 0, 7)
        if not cfg:
            w.F = wl.random_fraction(*shape, 7)
        F = torch.from_numpy(w.F).cuda()
        rhs = torch.from_numpy(w.rhs).cuda()
        ref = None
        cases = [(B.KERNEL_TWOPASS, 0, 0), (B.KERNEL_FUSED, 1, 0), (B.KERNEL_FUSED, 1, 2),
                 (B.KERNEL_FUSED_OTF, 1, 0), (B.KERNEL_RESIDENT, 0, 0), (B.KERNEL_CLUSTER, 0, 0)]
        for kernel, rpt, chunks in cases:
            with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
                try:
                    s.set_kernel(kernel)
                except B.PsError:
                    if kernel == B.KERNEL_CLUSTER:       # the grid does not fit one cluster
                        continue
                    raise
                if kernel in (B.KERNEL_FUSED, B.KERNEL_FUSED_OTF):
                    s.set_tuning(rpt, chunks)
                s.set_fraction(F, w.rho_l, w.rho_g)
                p = torch.zeros_like(rhs)
                info = s.solve(rhs, p, w.omega, 3, 0.0)
                if ref is None:
                    ref = p.clone()
                assert torch.equal(p, ref), (cfg, shape, kernel, rpt, chunks)
                assert info.res_rel > 0.0
                ran += 1
        with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
            s.set_fraction(F, w.rho_l, w.rho_g)
            # one V(0,2) cycle with the fused residual + restriction + norm pass, one V(1,1) cycle
            for nu1 in (0, 1):
                s.mg_setup(levels=3, nu1=nu1, nu2=2 - nu1, coarse_sweeps=5, omega_s=1.5,
                           nu_growth=2, nu_max=4)
                p = torch.zeros_like(rhs)
                mi = s.mg_solve(rhs, p, 1, 1e-30)
                assert mi.sweeps == 1 and mi.res_rel > 0.0
            u = [torch.from_numpy(wl.noise_rhs(w.nx, w.ny, w.nz, 40 + q)).cuda() for q in range(3)]
            r2 = s.rhs_from_velocity(*u, 1e-3)
            div = s.face_divergence(*u, p, 1e-3)
            s.correct_velocity(p, 1e-3, *u)
            kap = torch.from_numpy(wl.curvature_field(w.nx, w.ny, w.nz, w.centres, w.diameter, w.dx)).cuda()
            t = s.ssf_rhs(F, kap, wl.SIGMA)
            assert all(bool(torch.isfinite(x).all()) for x in (r2, div, t, *u))
            ran += 1
    torch.cuda.synchronize()
    print(f"sanitize target ok: {ran} cases")
    return 0


def run_tool(tool: str, timeout: int):
    exe = os.environ.get("COMPUTE_SANITIZER", "/usr/local/cuda/bin/compute-sanitizer")
    cmd = [exe, "--tool", tool, "--print-limit", "20", "--launch-timeout", "0"]
    if tool == "memcheck":
        cmd += ["--leak-check", "no"]
    if tool == "initcheck":
        cmd += ["--track-unused-memory", "no"]
    cmd += [sys.executable, "-m", "paper_2104_01636_b200.sanitize", "--target"]
    t0 = time.time()
    try:
        res = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout)
        out, rc = res.stdout + res.stderr, res.returncode
    except subprocess.TimeoutExpired as e:
        out = (e.stdout or b"").decode(errors="replace") + (e.stderr or b"").decode(errors="replace")
        rc = -999
    return cmd, rc, time.time() - t0, out


def summarise(tool, cmd, rc, secs, out) -> str:
    summ = re.findall(r"=+ (ERROR SUMMARY: .*|RACECHECK SUMMARY: .*)", out)
    ok = "sanitize target ok" in out
    head = [f"### `{tool}`", "", f"    {' '.join(cmd)}", "",
            f"exit code {rc}, {secs:.0f} s; target finished: {'yes' if ok else 'NO'}; "
            f"summary: {'; '.join(summ) if summ else 'none printed'}", ""]
    reports = [ln for ln in out.splitlines() if ln.startswith("=========")
               and "SUMMARY" not in ln and "COMPUTE-SANITIZER" not in ln]
    if reports:
        head += ["First report lines:", "", "```"] + reports[:40] + ["```", ""]
    elif not summ:
        head += ["Output (tail):", "", "```"] + out.splitlines()[-25:] + ["```", ""]
    return "\n".join(head)


def soak(runs=((3, 20000), (4, 4000), (5, 800))) -> int:
    """Long-run repeatability of the hand-synchronised fused sweep: n sweeps on each config with
    the library's launch options, free running, dependent launches + pacing window 1, and the
    library's options again -- all four fields must be bitwise equal and finite (a rare miss in
    the mbarrier protocol, the pacing or the grid-dependency wait would show up as a difference).
    Prints one JSON line per run; returns the number of runs that differed."""
    import json
    import torch
    from . import binding as B, build, workload as wl
    build.build()
    B.load()
    assert torch.cuda.is_available(), "sanitize --soak needs the GPU"
    bad = 0
    for cfg, n in runs:
        w = wl.make_config(cfg)
        F = torch.from_numpy(w.F).cuda()
        rhs = torch.from_numpy(w.rhs).cuda()
        ref = None
        for dep, window in ((-1, -1), (0, 0), (1, 1), (-1, -1)):
            with B.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
                s.set_kernel(B.KERNEL_FUSED)
                s.set_launch_options(dep, window)
                s.set_fraction(F, w.rho_l, w.rho_g)
                p = torch.zeros_like(rhs)
                s.sweeps(rhs, p, w.omega, n)
                torch.cuda.synchronize()
                if ref is None:
                    ref = p.clone()
                ok = bool(torch.equal(p, ref)) and bool(torch.isfinite(p).all())
                bad += 0 if ok else 1
                print(json.dumps({"config": cfg, "sweeps": n, "dependent_launch, pace_window":
                                  s.get_launch_options(), "bitwise_equal_and_finite": ok}), flush=True)
        del ref
    return bad


def main(argv=None) -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--target", action="store_true")
    ap.add_argument("--soak", action="store_true")
    ap.add_argument("--tools", default="memcheck,initcheck,racecheck,synccheck")
    ap.add_argument("--timeout", type=int, default=1500, help="seconds per tool")
    ap.add_argument("--md", default="")
    args = ap.parse_args(argv)
    if args.target:
        return target()
    if args.soak:
        return 1 if soak() else 0
    parts = []
    for tool in args.tools.split(","):
        parts.append(summarise(tool, *run_tool(tool, args.timeout)))
        print(parts[-1], flush=True)
    if args.md:
        with open(args.md, "w") as f:
            f.write("\n".join(parts))
    return 0


if __name__ == "__main__":
    sys.exit(main())
