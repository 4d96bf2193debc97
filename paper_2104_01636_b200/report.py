"""Five-config report of the CUDA path (BASELINE.json `metric`):

    python -m paper_2104_01636_b200.report [--configs 1,2,3,4,5] [--max-sweeps 1000000] [--md FILE]

For every config: fixed-sweep throughput (Gcell-updates/s, CUDA events around `ps_sweeps`), the
model HBM rate of the kernel that ran (bytes per cell-update of DESIGN.md §7 x throughput), and --
for every config but the largest -- wall time and sweep count of `ps_solve` to a relative
residual of 1e-8 (check cadence K = 50, norm checks and the final read-back included).  Prints a
markdown table.  Needs the B200 and the built library: there is no CPU path.

    python -m paper_2104_01636_b200.report --mg-scan --configs 3,4 --omega-s 1.4,1.5 --omega-c 1.9,1.97 ...
        scan of multigrid parameters (cycles and wall time to 1e-8), see mg_scan
    python -m paper_2104_01636_b200.report --sass [--md FILE]
        architecture list and per-kernel instruction counts of the built library (no GPU)
"""
from __future__ import annotations

import argparse
import json
import sys
import time

BYTES_PER_UPDATE = {"twopass": 80.0, "fused": 48.0, "fused_otf": 32.0, "resident": 80.0,
                    "cluster": 80.0}


def run_config(cfg: int, max_sweeps: int, to_tol: bool, kernel: int, mg_cycles: int = 1000,
               fixed_override: int = 0, launch_options=(-1, -1), mg: bool = True):
    import torch
    from . import binding, workload as wl
    w = wl.make_config(cfg)
    fixed = fixed_override or wl.CONFIGS[cfg][7] or 500
    F_d = torch.from_numpy(w.F).cuda()
    rhs_d = torch.from_numpy(w.rhs).cuda()
    p_d = torch.zeros_like(rhs_d)
    out = {"config": cfg, "workload": w.name, "cells": w.cells, "omega": w.omega}
    with binding.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_kernel(kernel)
        kname = binding.KERNEL_NAMES[s.get_kernel()]
        out["kernel"] = kname
        if kname in ("fused", "fused_otf"):
            s.set_launch_options(*launch_options)
            out["dependent_launch"], out["pace_window"] = s.get_launch_options()
        s.set_fraction(F_d, w.rho_l, w.rho_g)
        s.sweeps(rhs_d, p_d, w.omega, min(fixed, 20))          # warm-up
        torch.cuda.synchronize()
        p_d.zero_()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        s.sweeps(rhs_d, p_d, w.omega, fixed)
        ev1.record()
        torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1)
        res = s.residual(rhs_d, p_d)
        out.update(fixed_sweeps=fixed, fixed_ms=ms,
                   gcell_per_s=w.cells * fixed / (ms / 1e3) / 1e9,
                   model_gb_per_s=w.cells * fixed * BYTES_PER_UPDATE[kname] / (ms / 1e3) / 1e9,
                   res_rel_after_fixed=res[1])
        if to_tol:
            p_d.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            info = s.solve(rhs_d, p_d, w.omega, max_sweeps, 1e-8)
            torch.cuda.synchronize()
            out.update(tol_seconds=time.perf_counter() - t0, tol_sweeps=info.sweeps,
                       tol_converged=bool(info.converged), tol_res_rel=info.res_rel)
        if not mg:
            return out
        # multigrid accelerated solve, binding defaults, every config; an untimed
        # two-cycle warm-up first (level memory, lazy loading of the multigrid kernels), as in
        # bench.py: a time stepper pays those once, not per solve
        s.mg_setup()
        s.mg_solve(rhs_d, p_d, 2, 0.0)
        p_d.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        levels = s.mg_setup()
        mg = s.mg_solve(rhs_d, p_d, mg_cycles, 1e-8)
        torch.cuda.synchronize()
        out.update(mg_seconds=time.perf_counter() - t0, mg_cycles=mg.sweeps, mg_levels=levels,
                   mg_converged=bool(mg.converged), mg_res_rel=mg.res_rel)
    return out


def kernel_rates(cfg: int = 4, reps: int = 20) -> str:
    """Per-kernel device time and algorithmic HBM rate of the single-pass kernels (DESIGN.md §7
    bytes per cell), CUDA events around `reps` back-to-back launches each."""
    import torch
    from . import binding, workload as wl
    w = wl.make_config(cfg)
    F = torch.from_numpy(w.F).cuda()
    u = [torch.randn(F.shape, dtype=torch.float64, device="cuda") for _ in range(3)]
    p = torch.randn(F.shape, dtype=torch.float64, device="cuda")
    kap = torch.rand(F.shape, dtype=torch.float64, device="cuda")
    rhs = torch.empty_like(p)
    rows = []
    with binding.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
        s.set_fraction(F, w.rho_l, w.rho_g)
        cases = [("ps_set_fraction (coefficient build)", lambda: s.set_fraction(F, w.rho_l, w.rho_g), 32),
                 ("ps_residual (norm, incl. final reduction + read-back)", lambda: s.residual(rhs, p), 40),
                 ("ps_mg_residual_restrict", lambda: s.mg_residual_restrict(rhs, p), 41),
                 ("ps_rhs_from_velocity", lambda: s.rhs_from_velocity(*u, 1e-3, rhs), 32),
                 ("ps_correct_velocity", lambda: s.correct_velocity(p, 1e-3, *u), 80),
                 ("ps_face_divergence", lambda: s.face_divergence(*u, p, 1e-3), 64),
                 ("ps_ssf_rhs", lambda: s.ssf_rhs(F, kap, 0.072), 48)]
        for name, fn, nbytes in cases:
            fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            rows.append(f"| `{name}` | {nbytes} | {ms * 1e3:.0f} | {w.cells * nbytes / ms / 1e6:.0f} |")
    return ("| call (config %d, %d cells) | algorithmic B/cell | µs per call | GB/s |\n|---|---|---|---|\n"
            % (cfg, w.cells)) + "\n".join(rows) + "\n"


def write_traffic(raw_csv: str, key: str, source: str, path: str) -> dict:
    """profiles/traffic.json from the raw page of an `ncu --set full` capture of the sweep kernel
    (`ncu -i X.ncu-rep --page raw --csv > raw.csv`): mean over the captured launches of
    dram__bytes_read.sum + dram__bytes_write.sum, stored under `key` ("fused:config4") together
    with the sha256 of the kernel source it was captured with -- bench.py reports the value only
    while that hash still matches."""
    import csv
    import hashlib
    import os
    with open(raw_csv, newline="") as f:
        rows = [r for r in csv.reader(f) if r]
    hdr, units, data = rows[0], rows[1], rows[2:]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}

    def col(name):
        i = hdr.index(name)
        return [float(r[i].replace(",", "")) * scale[units[i]] for r in data]
    tot = [a + b for a, b in zip(col("dram__bytes_read.sum"), col("dram__bytes_write.sum"))]
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "csrc", "ps_kernels_zmarch.cuh"), "rb") as f:
        sha = hashlib.sha256(f.read()).hexdigest()[:16]
    try:
        with open(path) as f:
            rec = json.load(f)
    except (OSError, ValueError):
        rec = {}
    if rec.get("kernel_source_sha16") != sha:      # captures of another kernel version are stale
        rec = {}
    rec[key] = sum(tot) / len(tot)
    rec["kernel_source_sha16"] = sha
    rec["_source"] = source
    with open(path, "w") as f:
        json.dump(rec, f, indent=1)
        f.write("\n")
    return rec


SASS_OPCODES = ("UTMALDG", "UTMAPF", "SYNCS.ARRIVE", "SYNCS.PHASECHK", "SYNCS.EXCH", "UCGABAR",
                "ACQBULK", "PREEXIT", "DFMA", "DMUL", "DADD", "MUFU.RCP64H", "LDG*.128",
                "LDG*.64", "STG*.128", "STG*.64", "LDS", "STS", "ATOMG", "RED", "SHFL", "BAR.SYNC",
                "NANOSLEEP", "HMMA", "UTCHMMA", "UTCQMMA")      # A*.w: opcode A of width w


def sass_summary() -> str:
    """Markdown: the architectures in the built product library (`cuobjdump -lelf`) and, per
    kernel, how often the instructions that tell a Blackwell-native tile-movement kernel from a
    recompiled one occur in its SASS (`cuobjdump -sass`): TMA tensor loads (UTMALDG), mbarrier
    arrive / try-wait (SYNCS.*), the cluster barrier (UCGABAR_*), the dependent-launch pair
    (ACQBULK, PREEXIT), the fp64 arithmetic and the 16-byte global accesses.  No GPU needed."""
    import hashlib
    import re
    import subprocess
    from . import build
    lib = build.build()
    elf = subprocess.run(["cuobjdump", "-lelf", lib], capture_output=True, text=True, check=True).stdout
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    demangle = {}
    names = re.findall(r"Function : (\S+)", sass)
    out = subprocess.run(["cu++filt", *names], capture_output=True, text=True)
    if out.returncode == 0:
        demangle = dict(zip(names, out.stdout.splitlines()))
    kernels, cur = {}, None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = kernels.setdefault(m.group(1), {"n": 0, **{k: 0 for k in SASS_OPCODES}})
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]+)", line)
        if m and cur is not None:
            cur["n"] += 1
            op = m.group(1)
            for k in SASS_OPCODES:
                head, star, width = k.partition("*")
                if op.startswith(head) and (not star or width in op):
                    cur[k] += 1
    used = [k for k in SASS_OPCODES if any(v[k] for v in kernels.values())]
    absent = [k for k in SASS_OPCODES if k not in used]
    srcs = sorted(build._deps())
    h = hashlib.sha256()
    for f in srcs:
        with open(f, "rb") as fh:
            h.update(fh.read())
    md = ["# SASS of libps_poisson.so: architectures and instruction counts per kernel", "",
          "Command: `python -m paper_2104_01636_b200.report --sass` (runs `cuobjdump -lelf` and "
          "`cuobjdump -sass` on the library built from the committed sources; no GPU).",
          f"sha256 over the library's sources (include/ps_poisson.h, csrc/*): `{h.hexdigest()[:16]}`.",
          "", "`cuobjdump -lelf`:", "", "```", elf.strip(), "```", "",
          "Instruction counts (prefix match on the opcode; columns that are zero everywhere are "
          "listed below the table):", "",
          "| kernel | instr | " + " | ".join(used) + " |", "|---|---:|" + "---:|" * len(used)]
    for name, c in sorted(kernels.items(), key=lambda kv: -kv[1]["n"]):
        short = re.sub(r"\((int|bool)\)", "", demangle.get(name, name))
        short = re.sub(r"\(.*", "", short)
        short = re.sub(r"<unnamed>::|ps::|void ", "", short)
        md.append(f"| `{short}` | {c['n']} | " + " | ".join(str(c[k]) for k in used) + " |")
    md += ["", "Absent from every kernel: " + (", ".join(absent) or "-") +
           " (no tensor-core instruction: the path is a stencil, not a contraction).", ""]
    return "\n".join(md)


def _floats(s):
    return [float(x) for x in s.split(",")]


def _ints(s):
    return [int(x) for x in s.split(",")]


def mg_scan(argv=None) -> None:
    """`--mg-scan`: every combination of the listed multigrid parameters through ps_mg_setup +
    ps_mg_solve(tol = 1e-8) from p = 0 on the listed configs (one untimed warm-up solve per config;
    wall time includes the coarsening of all levels); one JSON line per run on stderr and a markdown
    table sorted by the time on the last config.  This is the scan binding.MG_DEFAULTS were chosen
    with (profiles/r02_mg_tuning.md, made when it still was a module of its own,
    `mg_tune`, with the same options)."""
    import itertools
    ap = argparse.ArgumentParser(prog="report --mg-scan")
    ap.add_argument("--configs", default="3,4")
    ap.add_argument("--levels", default="6")
    ap.add_argument("--nu", default="0:2", help="nu1:nu2 pairs, comma separated")
    ap.add_argument("--coarse-sweeps", default="10")
    ap.add_argument("--gamma", default="1")
    ap.add_argument("--omega-s", default="1.5")
    ap.add_argument("--omega-c", default="1.95")
    ap.add_argument("--nu-growth", default="16")
    ap.add_argument("--nu-max", default="32")
    ap.add_argument("--nu-max-deep", default="0", help="cap from level 2 on (0 = nu_max)")
    ap.add_argument("--max-cycles", type=int, default=400)
    ap.add_argument("--seed-offset", type=int, default=0,
                    help="another bubble arrangement and rhs of the same recipe (workload.make_config)")
    ap.add_argument("--md", default="")
    args = ap.parse_args(argv)
    import torch
    from . import binding, build, workload as wl
    if not torch.cuda.is_available():
        raise SystemExit("report --mg-scan: no CUDA device (the CUDA path is the only path)")
    build.build()
    binding.load()
    cfgs = _ints(args.configs)
    nus = [tuple(int(v) for v in q.split(":")) for q in args.nu.split(",")]
    grid = list(itertools.product(_ints(args.levels), nus, _ints(args.coarse_sweeps),
                                  _ints(args.gamma), _floats(args.omega_s), _floats(args.omega_c),
                                  _ints(args.nu_growth), _ints(args.nu_max), _ints(args.nu_max_deep)))
    results = {}
    for cfg in cfgs:
        w = wl.make_config(cfg, seed_offset=args.seed_offset)
        F_d = torch.from_numpy(w.F).cuda()
        rhs_d = torch.from_numpy(w.rhs).cuda()
        p_d = torch.zeros_like(rhs_d)
        with binding.PoissonSolver(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz) as s:
            s.set_fraction(F_d, w.rho_l, w.rho_g)
            s.mg_setup()
            s.mg_solve(rhs_d, p_d, 2, 0.0)
            for lv, (nu1, nu2), cs, gm, os_, oc, g, m, md in grid:
                prm = dict(levels=lv, nu1=nu1, nu2=nu2, coarse_sweeps=cs, gamma=gm, omega_s=os_,
                           omega_c=oc, nu_growth=g, nu_max=m, nu_max_deep=md or m)
                p_d.zero_()
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                s.mg_setup(**prm)
                mg = s.mg_solve(rhs_d, p_d, args.max_cycles, 1e-8)
                torch.cuda.synchronize()
                dt = time.perf_counter() - t0
                rec = dict(cfg=cfg, **prm, cycles=mg.sweeps, converged=bool(mg.converged),
                           res_rel=mg.res_rel, seconds=round(dt, 4))
                print(json.dumps(rec), file=sys.stderr, flush=True)
                results.setdefault(tuple(prm.items()), {})[cfg] = rec
    rows = sorted(results.items(),
                  key=lambda kv: kv[1][cfgs[-1]]["seconds"] if kv[1][cfgs[-1]]["converged"] else 1e9)
    head = ("| levels | V(nu1,nu2) | coarsest | gamma | omega_s | omega_c | growth | nu_max | deep | "
            + " | ".join(f"cfg {c}: cycles | s" for c in cfgs) + " |\n|" + "---|" * (9 + 2 * len(cfgs)) + "\n")
    body = ""
    for key, per in rows:
        q = dict(key)
        cells = " | ".join(
            (f"{per[c]['cycles']} | {per[c]['seconds']:.4f}" if per[c]["converged"]
             else f"not converged ({per[c]['res_rel']:.1e}) | -") for c in cfgs)
        body += (f"| {q['levels']} | V({q['nu1']},{q['nu2']}) | {q['coarse_sweeps']} | {q['gamma']} | "
                 f"{q['omega_s']} | {q['omega_c']} | {q['nu_growth']} | {q['nu_max']} | "
                 f"{q['nu_max_deep']} | {cells} |\n")
    md = head + body
    print(md)
    if args.md:
        with open(args.md, "w") as f:
            f.write(md)


def to_markdown(rows) -> str:
    head = ("| cfg | workload | kernel | sweeps | ms | Gcell-upd/s | model GB/s | res_rel after | "
            "SOR to 1e-8: sweeps | seconds | res_rel | MG to 1e-8: cycles (levels) | seconds | res_rel |\n"
            "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|\n")
    body = ""
    for r in rows:
        tol = (f"{r['tol_sweeps']}{'' if r['tol_converged'] else ' (not converged)'} | "
               f"{r['tol_seconds']:.2f} | {r['tol_res_rel']:.3e}") if "tol_sweeps" in r else "- | - | -"
        body += (f"| {r['config']} | {r['workload']} | {r['kernel']} | {r['fixed_sweeps']} | "
                 f"{r['fixed_ms']:.2f} | {r['gcell_per_s']:.1f} | {r['model_gb_per_s']:.0f} | "
                 f"{r['res_rel_after_fixed']:.3e} | {tol} | "
                 + (f"{r['mg_cycles']}{'' if r['mg_converged'] else ' (not converged)'} "
                    f"({r['mg_levels']}) | {r['mg_seconds']:.3f} | {r['mg_res_rel']:.3e} |\n"
                    if "mg_cycles" in r else "- | - | - |\n"))
    return head + body


def main(argv=None):
    argv = list(sys.argv[1:] if argv is None else argv)
    if "--mg-scan" in argv:                 # its own option set: see mg_scan
        argv.remove("--mg-scan")
        return mg_scan(argv)
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="1,2,3,4,5")
    ap.add_argument("--max-sweeps", type=int, default=1_000_000)
    ap.add_argument("--sor-tol-configs", default="1,2,3",
                    help="configs whose plain-SOR solve to 1e-8 is run (config 4 needs > 1e6 sweeps)")
    ap.add_argument("--no-tol", action="store_true", help="skip the to-tolerance solves")
    ap.add_argument("--mg-cycles", type=int, default=1000, help="cap of multigrid cycles")
    ap.add_argument("--sweeps", type=int, default=0, help="fixed-sweep count (default: the config's)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "twopass", "fused", "fused_otf"])
    ap.add_argument("--no-mg", action="store_true", help="skip the multigrid legs")
    ap.add_argument("--pace-window", type=int, default=-1,
                    help="fused kernel: pacing window (0 = off, -1 = library choice)")
    ap.add_argument("--dependent-launch", type=int, default=-1,
                    help="fused kernel: dependent launches 0/1 (-1 = library choice)")
    ap.add_argument("--md", default="", help="also write the table to this file")
    ap.add_argument("--kernel-rates", action="store_true",
                    help="only time the single-pass kernels on config 4 and print their rates")
    ap.add_argument("--traffic-from", default="",
                    help="raw-page csv of an `ncu --set full` capture of the sweep kernel: write its "
                         "DRAM bytes per launch to profiles/traffic.json (no GPU needed)")
    ap.add_argument("--traffic-key", default="fused:config4")
    ap.add_argument("--traffic-source", default="", help="where the capture is summarised")
    ap.add_argument("--sass", action="store_true",
                    help="only print the architecture list and per-kernel instruction counts of "
                         "the built library (cuobjdump; no GPU needed)")
    args = ap.parse_args(argv)
    if args.sass:
        md = sass_summary()
        print(md)
        if args.md:
            with open(args.md, "w") as f:
                f.write(md)
        return
    if args.traffic_from:
        import os
        root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
        print(json.dumps(write_traffic(args.traffic_from, args.traffic_key, args.traffic_source,
                                       os.path.join(root, "profiles", "traffic.json"))))
        return
    import torch
    from . import binding, build
    if not torch.cuda.is_available():
        raise SystemExit("report: no CUDA device (the CUDA path is the only path)")
    build.build()
    binding.load()
    kernel = {"auto": binding.KERNEL_AUTO, "twopass": binding.KERNEL_TWOPASS,
              "fused": binding.KERNEL_FUSED, "fused_otf": binding.KERNEL_FUSED_OTF}[args.kernel]
    if args.kernel_rates:
        md = kernel_rates()
        print(md)
        if args.md:
            with open(args.md, "w") as f:
                f.write(md)
        return
    rows = []
    for cfg in [int(c) for c in args.configs.split(",")]:
        r = run_config(cfg, args.max_sweeps, to_tol=(not args.no_tol and str(cfg) in args.sor_tol_configs.split(',')), kernel=kernel,
                       mg_cycles=args.mg_cycles, fixed_override=args.sweeps,
                       launch_options=(args.dependent_launch, args.pace_window),
                       mg=not args.no_mg)
        print(json.dumps(r), file=sys.stderr, flush=True)
        rows.append(r)
    md = to_markdown(rows)
    print(md)
    if args.md:
        with open(args.md, "w") as f:
            f.write(md)


if __name__ == "__main__":
    main()
